"""Pins of the CPU oracle against closed forms, invariants and brute force (no GPU).

Every test here checks oracle/lensed_oracle.c against something that is NOT the oracle:
a closed form, a limit, a finite-difference identity, a library routine for a special
case, or brute-force numerical integration.  See SURVEY.md section 8(c.3) / DESIGN.md.
"""
import math
import os

import numpy as np
import pytest
from scipy import integrate, special

from oracle import lensed_oracle as orc
from paper_1505_07674_b200 import synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
RNG = np.random.default_rng(12345)


def _golden(name):
    rows = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                rows.append([float(t) for t in line.split()])
    return rows


def _grad(f, x, y, h=1e-3):
    """five-point central differences (truncation error ~ h^4 f^(5) / 30)"""
    gx = (-f(x + 2 * h, y) + 8 * f(x + h, y) - 8 * f(x - h, y) + f(x - 2 * h, y)) / (12 * h)
    gy = (-f(x, y + 2 * h) + 8 * f(x, y + h) - 8 * f(x, y - h) + f(x, y - 2 * h)) / (12 * h)
    return gx, gy


# --------------------------------------------------------------------------- lenses
def test_sis_deflection_is_radial_with_einstein_radius():
    # alpha = b r_hat: |alpha| = b everywhere, so x = theta_E maps to y = 0 (the ring)
    p = [0.3, -0.2, 0.8]
    for t in np.linspace(0, 2 * math.pi, 17):
        x, y = 0.3 + 0.8 * math.cos(t), -0.2 + 0.8 * math.sin(t)
        ax, ay = orc.deflection(orc.LENS_SIS, p, x, y)
        assert math.hypot(ax, ay) == pytest.approx(0.8, rel=1e-14)
        assert x - ax == pytest.approx(0.3, abs=1e-14) and y - ay == pytest.approx(-0.2, abs=1e-14)
    assert orc.deflection(orc.LENS_SIS, p, 0.3, -0.2) == (0.0, 0.0)


def test_sis_image_positions_of_offaxis_source():
    # source at beta < theta_E on the x axis: images at beta + theta_E and beta - theta_E
    b, beta = 0.8, 0.3
    for xi in (beta + b, beta - b):
        ax, ay = orc.deflection(orc.LENS_SIS, [0, 0, b], xi, 0.0)
        assert xi - ax == pytest.approx(beta, abs=1e-15) and ay == 0.0


@pytest.mark.parametrize("kind,p", [
    (orc.LENS_SIS, [0.1, -0.2, 0.9]),
    (orc.LENS_POINT, [0.1, -0.2, 0.35]),
    (orc.LENS_SHEAR, [0.04, -0.07]),
    (orc.LENS_SIE, [0.1, -0.2, 1.3624, 0.75, 45.0]),
    (orc.LENS_SIE, [-0.05, 0.0, 1.1, 0.3, 130.0]),
])
def test_deflection_is_gradient_of_potential(kind, p):
    pts = RNG.uniform(-2, 2, size=(60, 2))
    n = 0
    for x, y in pts:
        if kind != orc.LENS_SHEAR and math.hypot(x - p[0], y - p[1]) < 0.3:
            continue                               # keep the FD truncation error small
        gx, gy = _grad(lambda a, b: orc.potential(kind, p, a, b), x, y)
        ax, ay = orc.deflection(kind, p, x, y)
        assert ax == pytest.approx(gx, abs=3e-9) and ay == pytest.approx(gy, abs=3e-9)
        n += 1
    assert n > 30


def test_potentials_are_the_textbook_ones():
    # the potentials themselves, retyped: SIS b r, point mass tE^2 ln r, shear (R4)
    x, y = 0.7, -0.4
    assert orc.potential(orc.LENS_SIS, [0.1, 0.2, 0.9], x, y) == pytest.approx(
        0.9 * math.hypot(x - 0.1, y - 0.2), rel=1e-15)
    assert orc.potential(orc.LENS_POINT, [0.1, 0.2, 0.3], x, y) == pytest.approx(
        0.09 * math.log(math.hypot(x - 0.1, y - 0.2)), rel=1e-14)
    assert orc.potential(orc.LENS_SHEAR, [0.05, 0.02], x, y) == pytest.approx(
        0.5 * 0.05 * (x * x - y * y) + 0.02 * x * y, rel=1e-15)


def _div_curl(kind, p, x, y, h=1e-5):
    axp, ayp = orc.deflection(kind, p, x + h, y)
    axm, aym = orc.deflection(kind, p, x - h, y)
    bxp, byp = orc.deflection(kind, p, x, y + h)
    bxm, bym = orc.deflection(kind, p, x, y - h)
    return ((axp - axm) + (byp - bym)) / (2 * h), ((ayp - aym) - (bxp - bxm)) / (2 * h)


def test_sie_divergence_is_twice_kappa_and_curl_free():
    # div(alpha) = 2 kappa = b / R with R of eq. 23: pins the normalisation
    b, q, pa = 1.3624, 0.75, 45.0
    c, s = math.cos(math.radians(pa)), math.sin(math.radians(pa))
    for x, y in RNG.uniform(-2, 2, size=(40, 2)):
        u, v = c * (x - 0.1) + s * (y + 0.2), -s * (x - 0.1) + c * (y + 0.2)
        R = math.sqrt(q * u * u + v * v / q)
        div, curl = _div_curl(orc.LENS_SIE, [0.1, -0.2, b, q, pa], x, y)
        assert div == pytest.approx(b / R, rel=2e-6)
        assert curl == pytest.approx(0.0, abs=2e-8)


def test_point_mass_and_shear_divergence():
    for x, y in RNG.uniform(-2, 2, size=(10, 2)):
        assert _div_curl(orc.LENS_POINT, [0.1, 0.2, 0.3], x, y)[0] == pytest.approx(0, abs=1e-6)
        d, c = _div_curl(orc.LENS_SHEAR, [0.05, 0.02], x, y)
        assert d == pytest.approx(0, abs=1e-9) and c == pytest.approx(0, abs=1e-9)
        d, _ = _div_curl(orc.LENS_SIS, [0.1, 0.2, 0.9], x, y)
        assert d == pytest.approx(0.9 / math.hypot(x - 0.1, y - 0.2), rel=1e-6)


def test_sie_tends_to_sis_as_q_tends_to_one():
    for x, y in RNG.uniform(-2, 2, size=(20, 2)):
        sx, sy = orc.deflection(orc.LENS_SIS, [0.1, -0.2, 1.2], x, y)
        for q, tol in ((1.0, 1e-15), (1 - 1e-10, 1e-9), (1 - 1e-6, 1e-6), (1 - 1e-4, 1e-4)):
            ex, ey = orc.deflection(orc.LENS_SIE, [0.1, -0.2, 1.2, q, 77.0], x, y)
            assert ex == pytest.approx(sx, abs=tol) and ey == pytest.approx(sy, abs=tol)


def test_sie_position_angle_is_ccw_from_x_to_major_axis():
    # PA counter-clockwise between major axis and x axis.  Along the major
    # axis kappa = b/(2R) falls off slowest: R = sqrt(q) r there, sqrt(1/q) r on the minor.
    b, q, pa = 1.0, 0.5, 30.0
    r = 1.5
    t = math.radians(pa)
    d_major, _ = _div_curl(orc.LENS_SIE, [0, 0, b, q, pa], r * math.cos(t), r * math.sin(t))
    d_minor, _ = _div_curl(orc.LENS_SIE, [0, 0, b, q, pa], -r * math.sin(t), r * math.cos(t))
    assert d_major == pytest.approx(b / (math.sqrt(q) * r), rel=1e-6)
    assert d_minor == pytest.approx(b / (r / math.sqrt(q)), rel=1e-6)


def _sie_alpha_by_mass_integral(b, q, u, v):
    """alpha(x) = 1/pi * int kappa(x') (x - x')/|x - x'|^2 d^2x', kappa = b/(2R), brute force in
    elliptical polar coordinates x' = (rho cos(phi)/sqrt q, rho sin(phi) sqrt q), d^2x' = rho drho dphi.
    Homoeoid shells outside the point exert no force, so rho runs to R(u, v) only."""
    R = math.sqrt(q * u * u + v * v / q)
    sq = math.sqrt(q)

    def comp(which):
        def f(rho, phi):
            xp, yp = rho * math.cos(phi) / sq, rho * math.sin(phi) * sq
            dx, dy = u - xp, v - yp
            return 0.5 * b * (dx if which == 0 else dy) / (dx * dx + dy * dy) / math.pi
        phi0 = math.atan2(v / sq, u * sq)          # boundary point where the integrand peaks
        val, _ = integrate.dblquad(f, phi0 - math.pi, phi0 + math.pi, 0.0, R,
                                   epsabs=1e-9, epsrel=1e-9)
        return val
    return comp(0), comp(1)


def test_sie_spot_value_against_golden_and_mass_integral():
    b, q, pa, u, v, au, av = _golden("sie_spot.txt")[0]
    ax, ay = orc.deflection(orc.LENS_SIE, [0, 0, b, q, pa], u, v)
    assert ax == pytest.approx(au, abs=1e-12) and ay == pytest.approx(av, abs=1e-12)
    ix, iy = _sie_alpha_by_mass_integral(b, q, u, v)
    assert ax == pytest.approx(ix, abs=2e-4) and ay == pytest.approx(iy, abs=2e-4)


def test_sie_kormann_asinh_asin_form():
    # Kormann et al. 1994 eq. 27a (major axis along x2 there): with f = q, f' = sqrt(1-f^2),
    # alpha_1 = sqrt(f)/f' asinh(f'/f cos(phi)), alpha_2 = sqrt(f)/f' asin(f' sin(phi)) in units
    # of their xi_0; here the major axis is along u, so the roles of the axes swap.
    b, q = 1.1, 0.6
    qp = math.sqrt(1 - q * q)
    for u, v in RNG.uniform(-2, 2, size=(20, 2)):
        phi = math.atan2(u, v)                     # angle from the v axis (their x1)
        a_v = b * math.sqrt(q) / qp * math.asinh(qp / q * math.cos(phi))
        a_u = b * math.sqrt(q) / qp * math.asin(qp * math.sin(phi))
        ax, ay = orc.deflection(orc.LENS_SIE, [0, 0, b, q, 0.0], u, v)
        assert ax == pytest.approx(a_u, abs=1e-13) and ay == pytest.approx(a_v, abs=1e-13)


def test_shear_maps_circle_to_ellipse():
    # y = x - alpha with shear only: a unit circle maps to an ellipse of axis ratio (1-g)/(1+g)
    g, phi = 0.08, math.radians(25.0)
    p = [g * math.cos(2 * phi), g * math.sin(2 * phi)]
    rr = []
    for t in np.linspace(0, 2 * math.pi, 721):
        x, y = math.cos(t), math.sin(t)
        ax, ay = orc.deflection(orc.LENS_SHEAR, p, x, y)
        rr.append(math.hypot(x - ax, y - ay))
    assert min(rr) / max(rr) == pytest.approx((1 - g) / (1 + g), rel=1e-5)


# ------------------------------------------------------------------ Sersic / Gaussian
def test_bn_golden_values_and_library_inverse():
    for n, bn in _golden("sersic_bn.txt"):
        assert orc.sersic_bn(n) == pytest.approx(bn, rel=2e-12)
    assert orc.sersic_bn(0.5) == pytest.approx(math.log(2.0), rel=1e-14)
    for n in np.linspace(0.3, 10.0, 40):
        assert orc.sersic_bn(n) == pytest.approx(special.gammaincinv(2 * n, 0.5), rel=1e-12)


def test_incomplete_gamma_against_library_and_closed_forms():
    for a in (0.6, 1.0, 2.5, 8.0, 16.0):
        for x in (0.1, 1.0, a, a + 1.5, 3 * a + 5):
            assert orc.gamma_p(a, x) == pytest.approx(special.gammainc(a, x), rel=1e-12)
    assert orc.gamma_p(1.0, 0.7) == pytest.approx(1 - math.exp(-0.7), rel=1e-14)   # P(1,x)
    assert orc.gamma_p(0.5, 0.7) == pytest.approx(math.erf(math.sqrt(0.7)), rel=1e-13)


def _flux_inside(kind, p, Rmax, q):
    """brute-force integral of the brightness over the ellipse R <= Rmax (scale=1: per arcsec^2)"""
    sq = math.sqrt(q)
    x0, y0, pa = p[0], p[1], math.radians(p[-1])
    c, s = math.cos(pa), math.sin(pa)

    def f(rho, phi):
        u, v = rho * math.cos(phi) / sq, rho * math.sin(phi) * sq
        return rho * orc.brightness(kind, p, x0 + c * u - s * v, y0 + s * u + c * v)
    val, _ = integrate.dblquad(f, 0, 2 * math.pi, 0, Rmax, epsabs=1e-10, epsrel=1e-10)
    return val


@pytest.mark.parametrize("n,q,pa", [(0.5, 1.0, 0.0), (1.0, 0.7, 30.0), (2.5, 0.4, 100.0), (4.0, 0.8, 45.0)])
def test_sersic_half_light_and_total_flux(n, q, pa):
    # r_S is the geometric-mean radius of the half-light ellipse and I_0 gives
    # total magnitude mag_S:  F = 10^(-0.4 mag).
    rs, mag = 0.3, -1.2
    F = 10 ** (-0.4 * mag)
    p = [0.1, -0.2, rs, mag, n, q, pa]
    assert _flux_inside(orc.SRC_SERSIC, p, rs, q) == pytest.approx(0.5 * F, rel=1e-8)
    # closed form F = I_0 2 pi n r^2 Gamma(2n) / b^(2n), with scipy's b_n
    bn = special.gammaincinv(2 * n, 0.5)
    I0 = orc.brightness(orc.SRC_SERSIC, p, 0.1, -0.2)
    assert I0 * 2 * math.pi * n * rs * rs * math.gamma(2 * n) / bn ** (2 * n) == pytest.approx(F, rel=1e-11)


def test_sersic_profile_shape_and_ellipse_convention():
    # eq. 22-23: I(R)/I_0 = exp(-b (R/r)^(1/n)), R = sqrt(x^2 q + y^2/q) in the rotated frame;
    # the major axis is along the rotated x (R grows slowest there).
    n, q, rs, pa = 2.0, 0.5, 0.4, 30.0
    p = [0.0, 0.0, rs, 0.0, n, q, pa]
    bn = special.gammaincinv(2 * n, 0.5)
    I0 = orc.brightness(orc.FG_SERSIC, p, 0, 0)
    t = math.radians(pa)
    r = 0.7
    on_major = orc.brightness(orc.FG_SERSIC, p, r * math.cos(t), r * math.sin(t))
    on_minor = orc.brightness(orc.FG_SERSIC, p, -r * math.sin(t), r * math.cos(t))
    assert on_major / I0 == pytest.approx(math.exp(-bn * (r * math.sqrt(q) / rs) ** (1 / n)), rel=1e-12)
    assert on_minor / I0 == pytest.approx(math.exp(-bn * (r / math.sqrt(q) / rs) ** (1 / n)), rel=1e-12)


def test_gaussian_equals_sersic_n_half_and_has_unit_flux():
    sigma, mag, q, pa = 0.12, 0.3, 0.6, 20.0
    g = [0.05, 0.02, sigma, mag, q, pa]
    s = [0.05, 0.02, sigma * math.sqrt(2 * math.log(2)), mag, 0.5, q, pa]
    for x, y in RNG.uniform(-0.5, 0.5, size=(30, 2)):
        assert orc.brightness(orc.SRC_GAUSS, g, x, y) == pytest.approx(
            orc.brightness(orc.SRC_SERSIC, s, x, y), rel=1e-11)
    # I_0 = F / (2 pi sigma^2)
    assert orc.brightness(orc.FG_GAUSS, g, 0.05, 0.02) == pytest.approx(
        10 ** (-0.4 * mag) / (2 * math.pi * sigma ** 2), rel=1e-13)


def test_magnitude_zero_point_and_pixel_scale_units():
    p = [0, 0, 0.2, 24.0, 1.5, 0.7, 10.0]
    a = orc.brightness(orc.SRC_SERSIC, p, 0.1, 0.1, scale=1.0, zp=0.0)
    b = orc.brightness(orc.SRC_SERSIC, p, 0.1, 0.1, scale=0.05, zp=25.0)
    assert b / a == pytest.approx(0.05 ** 2 * 10 ** (0.4 * 25.0), rel=1e-13)


def test_total_flux_of_rendered_image_independent_of_q_and_pa():
    # R6: sum_i L_i -> F (unlensed foreground component on a wide image)
    H = W = 96
    scale = 0.05
    quad = synth.gauss_legendre_rule(5)
    mag = -2.0
    F = 10 ** (-0.4 * mag)
    for q, pa in ((1.0, 0.0), (0.5, 30.0), (0.7, 120.0)):
        L = orc.render_raw(H, W, scale, quad, [orc.FG_GAUSS], [0.01, -0.02, 0.25, mag, q, pa])
        assert L.sum() == pytest.approx(F, rel=1e-7)
    L = orc.render_raw(H, W, scale, quad, [orc.FG_SERSIC], [0.0, 0.0, 0.15, mag, 1.0, 0.8, 40.0])
    # exponential profile: flux outside the 4.8" box is < 1e-6 of the total; the cusp costs ~1e-4
    assert L.sum() == pytest.approx(F, rel=3e-4)


# -------------------------------------------------------------- grid, rays, quadrature
def test_pixel_grid_convention_row_is_y_column_is_x():
    # R1: pixel (i, j) centre = ((j - (W-1)/2) s, (i - (H-1)/2) s); one-point rule at the centre
    H, W, s = 6, 9, 0.05
    p = [0.07, -0.04, 0.08, 0.0, 0.6, 25.0]
    L = orc.render_raw(H, W, s, [[0, 0, 1]], [orc.FG_GAUSS], p)
    for i in range(H):
        for j in range(W):
            x, y = (j - (W - 1) / 2) * s, (i - (H - 1) / 2) * s
            assert L[i, j] == pytest.approx(orc.brightness(orc.FG_GAUSS, p, x, y, scale=s), rel=1e-13)


def test_rule_offsets_are_in_pixel_units_xi_along_x_eta_along_y():
    H, W, s = 4, 5, 0.1
    p = [0.02, 0.03, 0.09, 0.0, 0.5, 60.0]
    L = orc.render_raw(H, W, s, [[0.25, -0.4, 3.0]], [orc.FG_GAUSS], p)   # weight renormalised
    i, j = 1, 3
    x, y = (j - 2.0 + 0.25) * s, (i - 1.5 - 0.4) * s
    assert L[i, j] == pytest.approx(orc.brightness(orc.FG_GAUSS, p, x, y, scale=s), rel=1e-13)


def test_constant_sky_is_returned_exactly_and_weights_are_normalised():
    for quad in (synth.gauss_legendre_rule(3), synth.subsample_rule(4), 7.0 * synth.gauss_kronrod_rule(7)):
        L = orc.render_raw(5, 7, 0.05, quad, [orc.FG_SKY], [0.0123])
        assert np.allclose(L, 0.0123, rtol=1e-14, atol=0)


def _supersample(H, W, s, kinds, params, m=64):
    return orc.render_raw(H, W, s, synth.subsample_rule(m), kinds, params)


def test_quadrature_converges_to_brute_force_supersampling():
    # north_star: "quadrature converging on tiny images checked by brute-force supersampling"
    H = W = 12
    s = 0.05
    kinds = [orc.LENS_SIS, orc.SRC_GAUSS]
    params = [0.0, 0.0, 0.2, 0.03, 0.01, 0.05, 0.0, 0.8, 30.0]
    ref = _supersample(H, W, s, kinds, params)
    errs = []
    for n in (1, 2, 3, 5):
        L = orc.render_raw(H, W, s, synth.gauss_legendre_rule(n), kinds, params)
        errs.append(np.abs(L - ref).max() / ref.max())
    assert errs[0] > errs[1] > errs[2] > errs[3] and errs[3] < 2e-3
    gk = orc.render_raw(H, W, s, synth.gauss_kronrod_rule(7), kinds, params)
    assert np.abs(gk - ref).max() / ref.max() < 2e-3


def test_pixel_integral_of_circular_gaussian_against_erf_closed_form():
    # eq. 3 for a circular Gaussian is a product of erf differences; a wide Gaussian is, within
    # a pixel, a low-degree polynomial, so the 3x3 Gauss-Legendre rule (exact to degree 5 per
    # axis) must hit it to ~1e-10 while 4x4 midpoints are only second order.
    H = W = 8
    s, sig, x0, y0, mag = 0.05, 0.4, 0.013, -0.021, 0.0
    p = [x0, y0, sig, mag, 1.0, 0.0]
    r2 = math.sqrt(2.0) * sig
    ref = np.empty((H, W))
    for i in range(H):
        for j in range(W):
            xa, ya = (j - 3.5 - 0.5) * s - x0, (i - 3.5 - 0.5) * s - y0
            ex = 0.5 * (math.erf((xa + s) / r2) - math.erf(xa / r2))
            ey = 0.5 * (math.erf((ya + s) / r2) - math.erf(ya / r2))
            ref[i, j] = ex * ey                    # flux 1 inside the pixel = mean SB * pixel area
    gl = orc.render_raw(H, W, s, synth.gauss_legendre_rule(3), [orc.FG_GAUSS], p)
    sub = orc.render_raw(H, W, s, synth.subsample_rule(4), [orc.FG_GAUSS], p)
    assert np.abs(gl / ref - 1).max() < 1e-10
    assert 1e-6 < np.abs(sub / ref - 1).max() < 1e-3


# --------------------------------------------------------------- lensing in the image
def test_sis_on_axis_source_renders_the_einstein_ring():
    # I(x) = I_S(|r - theta_E|) for an on-axis circular source behind a SIS
    H = W = 33
    s, b, sig = 0.05, 0.6, 0.07
    L = orc.render_raw(H, W, s, [[0, 0, 1]], [orc.LENS_SIS, orc.SRC_GAUSS],
                       [0, 0, b, 0, 0, sig, 0.0, 1.0, 0.0])
    yy, xx = np.meshgrid((np.arange(H) - 16) * s, (np.arange(W) - 16) * s, indexing="ij")
    r = np.hypot(xx, yy)
    expect = s * s / (2 * math.pi * sig * sig) * np.exp(-(r - b) ** 2 / (2 * sig * sig))
    expect[16, 16] = s * s / (2 * math.pi * sig * sig)     # alpha := 0 at the centre (R3)
    assert np.allclose(L, expect, rtol=1e-12, atol=0)


def test_zero_strength_lenses_leave_the_source_unlensed_and_deflections_add():
    H = W = 16
    s = 0.05
    quad = synth.gauss_legendre_rule(2)
    src = [0.05, -0.03, 0.1, 0.0, 1.5, 0.6, 40.0]
    kinds0 = [orc.LENS_SIS, orc.LENS_SIE, orc.LENS_POINT, orc.LENS_SHEAR, orc.SRC_SERSIC]
    lens0 = [0.1, 0.1, 0.0, -0.1, 0.0, 0.0, 0.7, 20.0, 0.2, 0.2, 0.0, 0.0, 0.0]
    a = orc.render_raw(H, W, s, quad, kinds0, lens0 + src)
    b = orc.render_raw(H, W, s, quad, [orc.FG_SERSIC], src)
    assert np.allclose(a, b, rtol=1e-14, atol=0)
    two = orc.render_raw(H, W, s, quad, [orc.LENS_SIS, orc.LENS_SIS, orc.SRC_SERSIC],
                         [0.01, 0.02, 0.2, 0.01, 0.02, 0.15] + src)
    one = orc.render_raw(H, W, s, quad, [orc.LENS_SIS, orc.SRC_SERSIC], [0.01, 0.02, 0.35] + src)
    assert np.allclose(two, one, rtol=1e-11, atol=0)


def test_image_is_foreground_at_x_plus_source_at_y():
    # eq. 2: foregrounds are not lensed
    H = W = 16
    s = 0.05
    quad = synth.gauss_legendre_rule(2)
    lens, src, fg = [0, 0, 0.3], [0.05, 0, 0.1, 0.0, 1.0, 0.8, 0.0], [0, 0, 0.2, -1.0, 0.7, 50.0]
    both = orc.render_raw(H, W, s, quad, [orc.LENS_SIS, orc.SRC_SERSIC, orc.FG_GAUSS, orc.FG_SKY],
                          lens + src + fg + [0.3])
    a = orc.render_raw(H, W, s, quad, [orc.LENS_SIS, orc.SRC_SERSIC], lens + src)
    b = orc.render_raw(H, W, s, quad, [orc.FG_GAUSS], fg)
    assert np.allclose(both, a + b + 0.3, rtol=1e-13, atol=0)


# ------------------------------------------------------------------------------- PSF
def test_delta_psf_is_the_identity_bitwise():
    L = RNG.uniform(size=(7, 9))
    assert np.array_equal(orc.convolve(L, None), L)
    assert np.array_equal(orc.convolve(L, np.array([[3.0]])), L)
    d = np.zeros((3, 5))
    d[1, 2] = 2.5
    assert np.array_equal(orc.convolve(L, d), L)


def test_one_hot_psf_shifts_with_edge_replication():
    # eq. 15 literally: F one-hot at F_{a,b} gives L*_{ij} = L_{i-a, j-b}, clamped;
    # array element [p+a][q+b] = F_{a,b}, first index = row (R10)
    H, W, p, q = 6, 8, 2, 1
    L = RNG.uniform(size=(H, W))
    for a in range(-p, p + 1):
        for b in range(-q, q + 1):
            F = np.zeros((2 * p + 1, 2 * q + 1))
            F[p + a, q + b] = 1.0
            out = orc.convolve(L, F)
            for i in range(H):
                for j in range(W):
                    assert out[i, j] == L[min(max(i - a, 0), H - 1), min(max(j - b, 0), W - 1)]


def test_convolution_against_library_correlate_with_nearest_padding():
    from scipy import ndimage
    L = RNG.uniform(size=(11, 13))
    F = RNG.uniform(size=(5, 7))
    ref = ndimage.convolve(L, F / F.sum(), mode="nearest")
    assert np.allclose(orc.convolve(L, F), ref, rtol=1e-13, atol=0)


def test_psf_is_normalised_automatically_and_keeps_constants():
    L = RNG.uniform(size=(9, 9))
    F = synth.moffat_psf(5, 2.0, 3.0, e1=0.2)
    assert np.allclose(orc.convolve(L, F), orc.convolve(L, 17.0 * F), rtol=1e-14, atol=0)
    c = np.full((6, 7), 0.37)
    assert np.allclose(orc.convolve(c, F), 0.37, rtol=1e-14, atol=0)        # borders included


# ------------------------------------------------------------------------------ logL
def test_loglike_closed_forms_and_mask():
    H, W = 5, 6
    model = RNG.uniform(size=(H, W))
    w = RNG.uniform(0.5, 2.0, size=(H, W))
    r = RNG.normal(size=(H, W))
    assert orc.chi2_loglike(model, model, w) == 0.0
    assert orc.chi2_loglike(model, model + r, w) == pytest.approx(-0.5 * np.sum(w * r * r), rel=1e-14)
    mask = (RNG.uniform(size=(H, W)) > 0.4).astype(np.uint8)
    d2 = model + r
    base = orc.chi2_loglike(model, d2, w, mask)
    assert base == pytest.approx(-0.5 * np.sum(w * r * r * mask), rel=1e-14)
    d3 = d2.copy()
    d3[mask == 0] += 100.0                       # data under the mask does not matter
    assert orc.chi2_loglike(model, d3, w, mask) == base


def _mini_problem():
    H = W = 20
    s = 0.05
    kinds = [orc.LENS_SIE, orc.LENS_SHEAR, orc.SRC_SERSIC, orc.FG_SERSIC, orc.FG_SKY]
    params = np.array([0.01, -0.02, 0.3, 0.7, 35.0, 0.03, -0.02,
                       0.05, 0.03, 0.06, 1.0, 1.5, 0.6, 70.0,
                       0.01, -0.02, 0.3, -2.0, 2.5, 0.8, 30.0, 0.01])
    return H, W, s, kinds, params, synth.gauss_legendre_rule(3), synth.moffat_psf(5, 2.0, 3.0, e1=0.1)


def test_full_loglike_is_render_convolve_chi2_and_parabola_in_flux():
    H, W, s, kinds, params, quad, psf = _mini_problem()
    truth = orc.render(H, W, s, psf, quad, kinds, params)[0]
    assert np.allclose(truth, orc.convolve(orc.render_raw(H, W, s, quad, kinds, params), psf),
                       rtol=0, atol=0)
    d = truth + 0.01 * RNG.normal(size=truth.shape)
    w = np.full_like(truth, 1e4)
    assert orc.loglike(H, W, s, truth, w, None, psf, quad, kinds, params)[0] == 0.0
    # chi^2 is a parabola in the linear flux of one component: 3 evaluations fix it, a 4th checks
    def ll(f):
        p = params.copy()
        p[10] = params[10] - 2.5 * math.log10(f)
        return orc.loglike(H, W, s, d, w, None, psf, quad, kinds, p)[0]
    f = np.array([0.5, 1.0, 1.5])
    coef = np.polyfit(f, [ll(v) for v in f], 2)
    assert ll(2.25) == pytest.approx(np.polyval(coef, 2.25), rel=1e-10)


def test_invalid_vector_gives_minus_infinity_and_nan_image():
    H, W, s, kinds, params, quad, psf = _mini_problem()
    bad = params.copy()
    bad[3] = 1.2                                  # q > 1
    P = np.stack([params, bad])
    d = np.zeros((H, W))
    logl, model = orc.loglike(H, W, s, d, np.ones((H, W)), None, psf, quad, kinds, P, want_model=True)
    assert np.isfinite(logl[0]) and logl[1] == -np.inf
    assert np.isfinite(model[0]).all() and np.isnan(model[1]).all()


def test_parameter_domain_bound_by_bound_against_hand_written_expectations():
    """params_valid, every kind and every bound: a vector just inside is rendered (finite logL and
    image), one just outside -- or with NaN / inf in any slot -- gives logL = -inf and a NaN image.
    The expectations are written out by hand in tests/cases.py (SURVEY.md section 8(b) "Errors";
    DESIGN.md section 2 "Domain" for 0.02 <= n <= 20 and r = 0 allowed for lenses)."""
    from paper_1505_07674_b200 import synth
    from tests.cases import domain_cases
    H, W, s = 10, 12, 0.05
    quad = synth.get_config(0).quad
    d, w = np.zeros((H, W)), np.ones((H, W))
    cases = domain_cases()
    assert sum(v for _, _, v in cases) >= 25 and sum(not v for _, _, v in cases) >= 130
    for models, p, valid in cases:
        logl, model = orc.loglike(H, W, s, d, w, None, None, quad, synth.kind_ids(models), p[None], want_model=True)
        what = (models, p.tolist())
        if valid:
            assert np.isfinite(logl[0]) and np.isfinite(model[0]).all(), what
        else:
            assert logl[0] == -np.inf and np.isnan(model[0]).all(), what


# -------------------------------------------------------------------- whole pipeline
def test_rotation_by_90_degrees_and_mirror_of_the_whole_pipeline():
    # square image, symmetric rule, PSF rotated/mirrored along: the model image rotates/mirrors
    H, W, s, kinds, params, quad, psf = _mini_problem()
    base = orc.render(H, W, s, psf, quad, kinds, params)[0]
    # rotate every position by +90 deg: (x, y) -> (-y, x), PA -> PA + 90, shear (g1,g2) -> (-g1,-g2)
    r = params.copy()
    for ox in (0, 7, 14):
        r[ox], r[ox + 1] = -params[ox + 1], params[ox]
    r[4] += 90.0
    r[13] += 90.0
    r[20] += 90.0
    r[5], r[6] = -params[5], -params[6]
    # image array of the rotated scene: new[i, j] = old[j, W-1-i]... check via np.rot90 both ways
    rot = orc.render(H, W, s, np.rot90(psf, 1), quad, kinds, r)[0]
    cand = [np.rot90(base, k) for k in range(4)]
    errs = [np.abs(rot - c).max() / base.max() for c in cand]
    assert min(errs) < 1e-12 and sorted(errs)[1] > 1e-3
    # mirror x -> -x: PA -> 180 - PA, g2 -> -g2; image columns flip
    m = params.copy()
    for ox in (0, 7, 14):
        m[ox] = -params[ox]
    m[4], m[13], m[20] = 180.0 - params[4], 180.0 - params[13], 180.0 - params[20]
    m[6] = -params[6]
    mir = orc.render(H, W, s, psf[:, ::-1], quad, kinds, m)[0]
    assert np.abs(mir - base[:, ::-1]).max() / base.max() < 1e-12


def test_whole_pixel_translation_shifts_the_image():
    H, W, s, kinds, params, quad, psf = _mini_problem()
    base = orc.render(H, W, s, None, quad, kinds[:-1] + [orc.FG_SKY], params)[0]
    t = params.copy()
    for ox in (0, 7, 14):
        t[ox] += 2 * s
        t[ox + 1] -= 3 * s
    # shear is about the image centre (R4): translating the scene changes the constant part of
    # the shear deflection, so the test uses zero shear
    t[5] = t[6] = 0.0
    p0 = params.copy()
    p0[5] = p0[6] = 0.0
    base = orc.render(H, W, s, None, quad, kinds, p0)[0]
    moved = orc.render(H, W, s, None, quad, kinds, t)[0]
    assert np.allclose(moved[:-3, 2:], base[3:, :-2], rtol=1e-9, atol=1e-15)


def test_chi2_per_dof_is_about_one_at_the_truth():
    # the paper's diagnostic: with the synthetic noise model chi^2/dof ~ 1
    cfg = synth.shrunk(synth.get_config(1), 40, 40, 4)
    kinds = synth.kind_ids(cfg.models)
    truth = orc.render(cfg.H, cfg.W, cfg.scale, cfg.psf, cfg.quad, kinds, cfg.truth)[0]
    d, w = cfg.observe(truth)
    ll = orc.loglike(cfg.H, cfg.W, cfg.scale, d, w, None, cfg.psf, cfg.quad, kinds, cfg.truth)[0]
    assert 0.85 < -2 * ll / (cfg.H * cfg.W) < 1.15


# ------------------------------------------------- quadrature error estimate
def test_embedded_gauss_weights_are_the_three_point_rule_on_the_kronrod_nodes():
    quad = synth.gauss_kronrod_rule(7)
    emb = synth.gauss_kronrod_embedded_weights(7)
    assert emb.sum() == pytest.approx(1.0, abs=1e-15) and np.count_nonzero(emb) == 9
    # the nonzero points are the 3 x 3 Gauss-Legendre rule on the pixel, weights included
    gl = synth.gauss_legendre_rule(3)
    mine = sorted((round(x, 12), round(y, 12), round(w, 12)) for (x, y, _), w in zip(quad, emb) if w != 0)
    ref = sorted((round(x, 12), round(y, 12), round(w, 12)) for x, y, w in gl)
    assert np.allclose(mine, ref, atol=1e-11)


def test_error_map_vanishes_for_what_both_rules_integrate_exactly():
    # constant sky: both weight sets sum to one -> the estimate is zero up to rounding
    quad, emb = synth.gauss_kronrod_rule(7), synth.gauss_kronrod_embedded_weights(7)
    e = orc.error_map(6, 5, 0.05, quad, emb, [orc.FG_SKY], [0.37])
    assert np.all(e <= 1e-15)


def test_error_map_of_a_separable_gaussian_is_the_product_of_one_dimensional_rules():
    """A circular Gaussian is exp(-x^2/2s^2) exp(-y^2/2s^2): on a pixel the Cartesian-square
    rule gives K1(x) K1(y) and the embedded rule G1(x) G1(y), K1 / G1 = the one-dimensional
    7-point Kronrod / 3-point Gauss sums, evaluated here from the node table of the paper's
    reference (Patterson 1968) without the oracle."""
    kx = np.array([0.0, 0.434243749346802, 0.774596669241483, 0.960491268708020])
    kw = np.array([0.450916538658474, 0.401397414775962, 0.268488089868333, 0.104656226026467])
    x1 = 0.5 * np.concatenate([-kx[:0:-1], kx])
    w1 = 0.5 * np.concatenate([kw[:0:-1], kw])
    g1x, g1w = 0.5 * np.array([-math.sqrt(0.6), 0.0, math.sqrt(0.6)]), 0.5 * np.array([5 / 9, 8 / 9, 5 / 9])
    H, W, s, sig = 7, 6, 0.05, 0.02                  # sigma = 0.4 px: badly resolved on purpose
    cx, cy = 0.013, -0.021
    F = 3.0
    i0 = F / (2 * math.pi * sig * sig) * s * s       # brightness per pixel area (R6, R7)
    quad, emb = synth.gauss_kronrod_rule(7), synth.gauss_kronrod_embedded_weights(7)
    e = orc.error_map(H, W, s, quad, emb, [orc.FG_GAUSS], [cx, cy, sig, synth.mag_of_flux(F), 1.0, 0.0])

    def rule(nodes, weights, c):
        return np.sum(weights * np.exp(-((c + nodes * s) ** 2) / (2 * sig * sig)))

    expect = np.empty((H, W))
    for i in range(H):
        for j in range(W):
            xc, yc = (j - 0.5 * (W - 1)) * s - cx, (i - 0.5 * (H - 1)) * s - cy
            expect[i, j] = i0 * abs(rule(x1, w1, xc) * rule(x1, w1, yc) - rule(g1x, g1w, xc) * rule(g1x, g1w, yc))
    assert e.max() > 1e-4 * i0                       # the estimate is not trivially small here
    assert np.allclose(e, expect, rtol=1e-10, atol=1e-14 * i0)


def test_error_map_tracks_the_true_error_of_the_embedded_rule():
    """The Kronrod sum is far more accurate than the embedded Gauss sum, so |K - G| must be
    the Gauss rule's true error; the exact pixel integral of a circular Gaussian is a product
    of erf differences."""
    H, W, s, sig = 5, 5, 0.05, 0.04
    cx, cy, F = 0.004, 0.009, 1.0
    p = [cx, cy, sig, synth.mag_of_flux(F), 1.0, 0.0]
    quad, emb = synth.gauss_kronrod_rule(7), synth.gauss_kronrod_embedded_weights(7)
    e = orc.error_map(H, W, s, quad, emb, [orc.FG_GAUSS], p)
    gq = quad.copy(); gq[:, 2] = emb
    g = orc.render_raw(H, W, s, gq, [orc.FG_GAUSS], p)

    def cdf(c):                                       # integral over one pixel side, centre offset c
        r = sig * math.sqrt(2.0)
        return 0.5 * (math.erf((c + 0.5 * s) / r) - math.erf((c - 0.5 * s) / r))

    exact = np.array([[F * cdf((j - 0.5 * (W - 1)) * s - cx) * cdf((i - 0.5 * (H - 1)) * s - cy)
                       for j in range(W)] for i in range(H)])
    true_err = np.abs(exact - g)
    assert true_err.max() > 1e-5 * exact.max()
    assert np.allclose(e, true_err, rtol=0.02, atol=1e-3 * true_err.max())


# ------------------------------ render_raw's Sersic against oracle_brightness and the total flux
@pytest.mark.parametrize("n", [0.5, 1.5, 2.5, 4.0, 8.0])
def test_render_raw_sersic_is_the_pinned_brightness_pixel_by_pixel(n):
    """PAPER.md:244-252 eqs. 22-23.  Every GPU parity test compares against oracle_render_raw;
    the half-light / total-flux / profile-shape pins above go through oracle_brightness.  With a
    one-point rule at the pixel centre the two must agree to rounding, as a source behind
    zero-strength lenses (evaluated at y = x) and as a foreground, for q < 1 and PA != 0."""
    H, W, s, zp = 14, 17, 0.05, 1.5
    p = [0.031, -0.047, 0.12, -0.7, n, 0.55, 37.0]
    fg = orc.render_raw(H, W, s, [[0, 0, 1]], [orc.FG_SERSIC], p, zp=zp)
    src = orc.render_raw(H, W, s, [[0, 0, 1]], [orc.LENS_SIS, orc.LENS_SHEAR, orc.SRC_SERSIC],
                         [0.1, 0.1, 0.0, 0.0, 0.0] + p, zp=zp)
    for i in range(H):
        for j in range(W):
            x, y = (j - (W - 1) / 2) * s, (i - (H - 1) / 2) * s
            ref = orc.brightness(orc.SRC_SERSIC, p, x, y, scale=s, zp=zp)
            assert fg[i, j] == pytest.approx(ref, rel=1e-13)
            assert src[i, j] == pytest.approx(ref, rel=1e-13)
    # and the profile itself, retyped with the library's b_n: I/I_0 = exp(-b (R/r)^(1/n)), eq. 22
    bn = special.gammaincinv(2 * n, 0.5)
    I0 = 10 ** (-0.4 * (p[3] - zp)) * bn ** (2 * n) / (2 * math.pi * n * p[2] ** 2 * math.gamma(2 * n)) * s * s
    t = math.radians(p[6])
    i, j = 3, 12
    dx, dy = (j - (W - 1) / 2) * s - p[0], (i - (H - 1) / 2) * s - p[1]
    u, v = math.cos(t) * dx + math.sin(t) * dy, -math.sin(t) * dx + math.cos(t) * dy
    R = math.sqrt(u * u * p[5] + v * v / p[5])
    assert fg[i, j] == pytest.approx(I0 * math.exp(-bn * (R / p[2]) ** (1 / n)), rel=1e-11)


def test_render_raw_sersic_sums_to_the_total_flux():
    """I_0 is chosen so that the source has total magnitude mag_S.  Through
    render_raw: sum_i L_i -> F for n = 1/2 (Gaussian tails, smooth: tight) and n = 4 (de
    Vaucouleurs): there the flux outside radius R is F Q(8, b_4 (R/r)^(1/4)), so the sum over
    the square image lies between the fluxes of its inscribed and circumscribed circles (the
    central cusp is integrated with the 15 x 15 rule; it holds < 1e-3 of the flux error)."""
    H = W = 96
    s, mag = 0.05, -2.0
    F = 10 ** (-0.4 * mag)
    L = orc.render_raw(H, W, s, synth.gauss_legendre_rule(5), [orc.FG_SERSIC], [0.01, -0.02, 0.3, mag, 0.5, 0.6, 25.0])
    assert L.sum() == pytest.approx(F, rel=1e-7)
    rs = 0.1
    L = orc.render_raw(H, W, s, synth.gauss_legendre_rule(15), [orc.FG_SERSIC], [0.0, 0.0, rs, mag, 4.0, 1.0, 0.0])
    b4 = special.gammaincinv(8.0, 0.5)
    half = 0.5 * H * s
    inside = lambda R: F * special.gammainc(8.0, b4 * (R / rs) ** 0.25)
    assert inside(half) * (1 - 1e-3) < L.sum() < inside(half * math.sqrt(2.0))
    assert inside(half * math.sqrt(2.0)) - inside(half) < 4e-3 * F          # the bracket is tight
    # a source behind a zero-strength lens: the same sum
    Ls = orc.render_raw(H, W, s, synth.gauss_legendre_rule(15), [orc.LENS_SIE, orc.SRC_SERSIC],
                        [0.2, 0.1, 0.0, 0.7, 30.0, 0.0, 0.0, rs, mag, 4.0, 1.0, 0.0])
    assert Ls.sum() == pytest.approx(L.sum(), rel=1e-13)


# -------------------------------------- source-plane positions (eq. 1; image-plane priors, L363)
def test_source_position_solves_the_sis_lens_equation_by_inspection():
    # a source at beta < theta_E on the x axis has images at beta + theta_E and beta - theta_E
    b, beta = 0.9, 0.25
    xy = [[beta + b, 0.0], [beta - b, 0.0]]
    out = orc.source_position([orc.LENS_SIS], [0.0, 0.0, b], xy)
    assert np.allclose(out, [[beta, 0.0], [beta, 0.0]], rtol=0, atol=1e-15)
    # off-axis lens centre and a rotated axis: same thing along the direction t
    c, t = np.array([0.3, -0.2]), np.array([math.cos(0.7), math.sin(0.7)])
    out = orc.source_position([orc.LENS_SIS], [c[0], c[1], b], [c + (beta + b) * t, c + (beta - b) * t])
    assert np.allclose(out, [c + beta * t, c + beta * t], rtol=0, atol=1e-15)


def test_source_position_sums_the_lenses_of_the_list_and_skips_the_lights():
    kinds = [orc.LENS_SIE, orc.SRC_SERSIC, orc.LENS_SHEAR, orc.FG_SKY, orc.LENS_POINT, orc.LENS_SIS]
    sie, shear, pm, sis = [0.02, -0.03, 1.2, 0.7, 35.0], [0.03, -0.05], [0.8, 0.6, 0.1], [-0.4, 0.3, 0.3]
    src = [0.1, 0.2, 0.15, 0.0, 2.0, 0.5, 10.0]
    params = sie + src + shear + [0.01] + pm + sis
    pts = RNG.uniform(-2.0, 2.0, size=(20, 2))
    out = orc.source_position(kinds, params, pts)
    lenses = ((orc.LENS_SIE, sie), (orc.LENS_SHEAR, shear), (orc.LENS_POINT, pm), (orc.LENS_SIS, sis))
    for (x, y), (sx, sy) in zip(pts, out):
        # y = x - grad(sum of the potentials), by finite differences of the pinned potentials
        gx, gy = _grad(lambda a, b: sum(orc.potential(k, p, a, b) for k, p in lenses), x, y, h=1e-3)
        assert sx == pytest.approx(x - gx, abs=2e-9) and sy == pytest.approx(y - gy, abs=2e-9)
        ax = sum(orc.deflection(k, p, x, y)[0] for k, p in lenses)
        ay = sum(orc.deflection(k, p, x, y)[1] for k, p in lenses)
        assert sx == pytest.approx(x - ax, abs=1e-15) and sy == pytest.approx(y - ay, abs=1e-15)
    # changing a light changes nothing; a lens outside its domain gives NaN
    params2 = list(params); params2[7] = 99.0
    assert np.array_equal(out, orc.source_position(kinds, params2, pts))
    params3 = list(params); params3[3] = 1.5
    assert np.all(np.isnan(orc.source_position(kinds, params3, pts)))
    # no lens at all: y = x
    assert np.array_equal(orc.source_position([orc.SRC_GAUSS], [0, 0, 0.1, 0, 1, 0], pts), pts)


def test_render_raw_evaluates_sources_at_the_source_position():
    # eq. 2 with the map above: one-point rule, I_S(y(x)) pixel by pixel
    H, W, s = 9, 11, 0.05
    kinds = [orc.LENS_SIE, orc.LENS_SHEAR, orc.SRC_GAUSS]
    params = [0.02, -0.03, 0.2, 0.7, 35.0, 0.05, -0.02, 0.03, 0.01, 0.08, 0.0, 0.6, 20.0]
    L = orc.render_raw(H, W, s, [[0.1, -0.2, 1]], kinds, params)
    pts = [[(j - (W - 1) / 2 + 0.1) * s, (i - (H - 1) / 2 - 0.2) * s] for i in range(H) for j in range(W)]
    src = orc.source_position(kinds, params, pts)
    ref = [orc.brightness(orc.SRC_GAUSS, params[7:], sx, sy, scale=s) for sx, sy in src]
    assert np.allclose(L.ravel(), ref, rtol=1e-13, atol=0)


# --------------------------------------------- variance estimation (eqs. 18-21)
def test_estimate_weights_hand_values_maps_and_the_extra_factor():
    d = np.array([3.0, 0.5, 10.0, -0.25])
    w, var = orc.estimate_weights(d, 2.0, 0.25, want_variance=True)
    # s^2 = (d + b)/g by hand: 3.25/2, 0.75/2, 10.25/2; d + b = 0: no Poisson variance (R15)
    assert np.allclose(var[:3], [1.625, 0.375, 5.125], rtol=1e-15) and np.isnan(var[3])
    assert np.allclose(w, [1 / 1.625, 1 / 0.375, 1 / 5.125, 0.0], rtol=1e-15)
    g, b = np.array([2.0, 4.0, 1.0, 3.0]), np.array([0.25, 0.0, -2.0, 1.0])
    w2 = orc.estimate_weights(d, g, b)
    assert np.allclose(w2, [2 / 3.25, 4 / 0.5, 1 / 8.0, 3 / 0.75], rtol=1e-15)
    x = np.array([1.0, 0.5, 0.0, 2.0])
    assert np.allclose(orc.estimate_weights(d, g, b, x), w2 * x, rtol=1e-15)
    assert np.array_equal(orc.estimate_weights(d, 2.0, 0.25), orc.estimate_weights(d, np.full(4, 2.0), np.full(4, 0.25)))
    for bad in (dict(gain=0.0), dict(gain=-1.0), dict(gain=float("nan")), dict(offset=float("inf")),
                dict(extra=np.array([1.0, -0.1, 1.0, 1.0]))):
        args = dict(image=d, gain=1.0, offset=0.0, extra=None)
        args.update(bad)
        with pytest.raises(ValueError):
            orc.estimate_weights(**args)


def test_estimated_variance_is_the_variance_of_poisson_data():
    """d = k/g - b with k ~ Poisson(mu): Var(d) = mu/g^2 (eq. 21 at k = mu), the sample variance
    of d matches the mean estimated s^2, and w (d - E d)^2 averages to E[(k - mu)^2/k] ~ 1 + 1/mu."""
    rng = np.random.default_rng(150507674)
    mu, g, b = 400.0, 3.0, 20.0
    k = rng.poisson(mu, size=200000)
    d = k / g - b
    w, var = orc.estimate_weights(d, g, b, want_variance=True)
    assert var.mean() == pytest.approx(mu / g ** 2, rel=2e-3)
    assert d.var() == pytest.approx(var.mean(), rel=1e-2)
    assert np.mean(w * (d - (mu / g - b)) ** 2) == pytest.approx(1.0 + 1.0 / mu, abs=0.01)


def test_library_weight_estimate_matches_the_oracle():
    """lensed_estimate_weights is host code of the product library (no device needed): the same
    seeded inputs through it and through the oracle."""
    from paper_1505_07674_b200 import lensed
    rng = np.random.default_rng(7)
    d = rng.uniform(-1.0, 50.0, size=(31, 17)).astype(np.float32)
    g = rng.uniform(0.5, 4.0, size=d.shape).astype(np.float32)
    b = rng.uniform(0.0, 2.0, size=d.shape).astype(np.float32)
    x = rng.uniform(0.0, 2.0, size=d.shape).astype(np.float32)
    for args in ((d, 2.5, 0.75, None), (d, g, b, None), (d, g, 0.5, x)):
        w_lib = lensed.lensed_estimate_weights(*args)
        w_orc = orc.estimate_weights(*args)
        assert np.array_equal(w_lib == 0, w_orc == 0)
        assert np.allclose(w_lib, w_orc, rtol=1e-6, atol=0)
