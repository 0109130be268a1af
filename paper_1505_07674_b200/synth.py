"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the CPU oracle (tests) and the CUDA library (tests, bench).
It holds none of the method's arithmetic: no deflection, no surface brightness, no
quadrature sum, no convolution, no chi-square.  It only produces *inputs*:
model lists, parameter vectors, quadrature-rule tables, PSF arrays, masks, noise.
The noiseless truth image is rendered by whoever calls `observe()` (the oracle in
tests, the CUDA library in bench.py) and passed in.

The configs stand in for the paper's GLAMER/TinyTim mocks and the
SLACS HST F814W cut-outs, which are not available; shapes and parameter
ranges follow PAPER.md:220-232, 252 and SURVEY.md section 8(d).
"""
import math

import numpy as np

SEED0 = 150507674

# model kind names; each side (oracle / CUDA binding) maps them to its own enum
KINDS = ("sis", "sie", "point", "shear", "src_sersic", "src_gauss",
         "fg_sersic", "fg_gauss", "sky")
NPAR = {"sis": 3, "sie": 5, "point": 3, "shear": 2, "src_sersic": 7, "src_gauss": 6,
        "fg_sersic": 7, "fg_gauss": 6, "sky": 1}
KIND_ID = {k: i for i, k in enumerate(KINDS)}   # same numbering in lensed.h and the oracle


def kind_ids(models):
    return np.array([KIND_ID[m] for m in models], dtype=np.int32)


def num_params(models):
    return sum(NPAR[m] for m in models)


# ----------------------------------------------------------------------------- rules
def gauss_legendre_rule(n):
    """n x n Gauss-Legendre rule on the pixel [-1/2, 1/2]^2, weights summing to 1."""
    x, w = np.polynomial.legendre.leggauss(n)
    x, w = 0.5 * x, 0.5 * w
    q = [(x[a], x[b], w[a] * w[b]) for b in range(n) for a in range(n)]
    return np.array(q, dtype=np.float64)


def subsample_rule(n):
    """The paper's `subN` rule: n x n midpoints, equal weights."""
    x = (np.arange(n) + 0.5) / n - 0.5
    q = [(x[a], x[b], 1.0 / (n * n)) for b in range(n) for a in range(n)]
    return np.array(q, dtype=np.float64)


_GK = {  # Gauss-Kronrod (Patterson 1968) nodes / Kronrod weights / embedded Gauss weights on
    # [-1, 1] (0 at the nodes the Gauss rule does not use)
    7: ([0.0, 0.434243749346802, 0.774596669241483, 0.960491268708020],
        [0.450916538658474, 0.401397414775962, 0.268488089868333, 0.104656226026467],
        [8.0 / 9.0, 0.0, 5.0 / 9.0, 0.0]),
}


def kronrod_extension(n_gauss):
    """(nodes, Kronrod weights, embedded Gauss weights) of the (2 n + 1)-point Kronrod extension
    of the n-point Gauss-Legendre rule on [-1, 1], nodes ascending; computed, not tabulated:
    the n + 1 added nodes are the roots of the Stieltjes polynomial E (degree n + 1, orthogonal
    to every polynomial of degree <= n with weight P_n), the weights are the interpolatory ones.
    g3k7 / g5k11 / g7k15 of PAPER.md:341-343 are n_gauss = 3 / 5 / 7."""
    leg = np.polynomial.legendre
    n = n_gauss
    xg, wg = leg.leggauss(n)
    xq, wq = leg.leggauss(2 * n + 4)                              # exact for the integrals below
    Pn = leg.legval(xq, [0] * n + [1])
    basis = np.stack([leg.legval(xq, [0] * j + [1]) for j in range(n + 2)])     # P_0 .. P_{n+1}
    # sum_j c_j int P_n P_j P_k = 0 for k = 0..n, c_{n+1} = 1
    A = np.array([[np.sum(wq * Pn * basis[j] * basis[k]) for j in range(n + 1)] for k in range(n + 1)])
    rhs = -np.array([np.sum(wq * Pn * basis[n + 1] * basis[k]) for k in range(n + 1)])
    c = np.append(np.linalg.solve(A, rhs), 1.0)
    xe = np.real(leg.legroots(c))
    x = np.sort(np.concatenate([xg, xe]))
    x = 0.5 * (x - x[::-1])                                        # symmetrise
    V = np.stack([leg.legval(x, [0] * j + [1]) for j in range(2 * n + 1)])
    w = np.linalg.solve(V, np.array([2.0] + [0.0] * (2 * n)))
    w = 0.5 * (w + w[::-1])
    g = np.zeros_like(w)
    for xi, wi in zip(xg, wg):
        g[np.argmin(np.abs(x - xi))] = wi
    return x, w, g


def gauss_kronrod_rule(n=7):
    """Cartesian square of the n-point Kronrod rule (n = 7 / 11 / 15: the paper's g3k7 default,
    g5k11, g7k15) on the pixel [-1/2, 1/2]^2, weights summing to 1."""
    x, w, _ = kronrod_extension((n - 1) // 2)
    x, w = 0.5 * x, 0.5 * w
    q = [(x[a], x[b], w[a] * w[b]) for b in range(n) for a in range(n)]
    return np.array(q, dtype=np.float64)


def gauss_kronrod_embedded_weights(n=7):
    """Weights of the embedded Gauss rule at the abscissae of gauss_kronrod_rule(n), same order,
    summing to 1: the rule whose difference from the Kronrod sum is the per-pixel error
    estimate of PAPER.md:166."""
    _, _, g = kronrod_extension((n - 1) // 2)
    g = 0.5 * g
    return np.array([g[a] * g[b] for b in range(n) for a in range(n)], dtype=np.float64)


# ------------------------------------------------------------------------------ PSFs
def gaussian_psf(size, fwhm_px):
    sig = fwhm_px / (2.0 * math.sqrt(2.0 * math.log(2.0)))
    r = np.arange(size) - (size - 1) / 2
    yy, xx = np.meshgrid(r, r, indexing="ij")
    return np.exp(-(xx * xx + yy * yy) / (2 * sig * sig))


def moffat_psf(size, fwhm_px, beta, e1=0.0):
    """Moffat profile sampled at pixel centres; e1 != 0 stretches x (asymmetric test PSFs)."""
    alpha = fwhm_px / (2.0 * math.sqrt(2.0 ** (1.0 / beta) - 1.0))
    r = np.arange(size) - (size - 1) / 2
    yy, xx = np.meshgrid(r, r, indexing="ij")
    rr = (xx * (1.0 - e1)) ** 2 + (yy * (1.0 + e1)) ** 2
    return (1.0 + rr / (alpha * alpha)) ** (-beta)


def annulus_mask(H, W, r_in, r_out):
    yy, xx = np.meshgrid(np.arange(H) - (H - 1) / 2, np.arange(W) - (W - 1) / 2, indexing="ij")
    r = np.hypot(xx, yy)
    return ((r >= r_in) & (r < r_out)).astype(np.uint8)


def mag_of_flux(F):
    return -2.5 * math.log10(F)


# --------------------------------------------------------------------- prior sampling
def _u(rng, lo, hi, B):
    return rng.uniform(lo, hi, size=B)


def _disc(rng, rmax, B):
    r = rmax * np.sqrt(rng.uniform(size=B))
    t = rng.uniform(0, 2 * math.pi, size=B)
    return r * np.cos(t), r * np.sin(t)


def _draw_sie(rng, B, pos=0.1, r=(0.8, 1.5)):
    return [_u(rng, -pos, pos, B), _u(rng, -pos, pos, B), _u(rng, r[0], r[1], B),
            _u(rng, 0.5, 1.0, B), _u(rng, 0.0, 180.0, B)]


def _draw_src_sersic(rng, B, r=(0.05, 0.3), flux=20.0):
    m0 = mag_of_flux(flux)
    return [_u(rng, -0.5, 0.5, B), _u(rng, -0.5, 0.5, B), _u(rng, r[0], r[1], B),
            _u(rng, m0 - 1, m0 + 1, B), _u(rng, 0.5, 4.0, B), _u(rng, 0.3, 1.0, B),
            _u(rng, 0.0, 180.0, B)]


def _draw_lens_light(rng, B, flux=2000.0):
    m0 = mag_of_flux(flux)
    return [_u(rng, -0.1, 0.1, B), _u(rng, -0.1, 0.1, B), _u(rng, 0.5, 2.0, B),
            _u(rng, m0 - 1, m0 + 1, B), _u(rng, 1.0, 6.0, B), _u(rng, 0.5, 1.0, B),
            _u(rng, 0.0, 180.0, B)]


def _draw_hst(rng, B, n_src=1):
    cols = _draw_sie(rng, B)
    g1, g2 = _disc(rng, 0.1, B)
    cols += [g1, g2]
    cols += _draw_src_sersic(rng, B)
    for _ in range(n_src - 1):
        cols += _draw_src_sersic(rng, B, r=(0.05, 0.15))
    cols += _draw_lens_light(rng, B)
    cols += [_u(rng, 0.0, 0.02, B)]
    return np.stack(cols, axis=1)


def _draw_multi(rng, B):
    main = _draw_sie(rng, B)
    second = [_u(rng, -2.0, 2.0, B), _u(rng, -2.0, 2.0, B), _u(rng, 0.2, 0.6, B),
              _u(rng, 0.5, 1.0, B), _u(rng, 0.0, 180.0, B)]
    # point-mass perturber: mass ratio 1e-3 => Einstein radius sqrt(1e-3) * main (reading R3),
    # placed within 0.3" of the main ring
    t = rng.uniform(0, 2 * math.pi, size=B)
    rr = main[2] + _u(rng, -0.3, 0.3, B)
    pm = [main[0] + rr * np.cos(t), main[1] + rr * np.sin(t),
          math.sqrt(1e-3) * main[2] * _u(rng, 0.8, 1.2, B)]
    g1, g2 = _disc(rng, 0.1, B)
    m0 = mag_of_flux(5.0)
    gauss = [_u(rng, -0.5, 0.5, B), _u(rng, -0.5, 0.5, B), _u(rng, 0.03, 0.15, B),
             _u(rng, m0 - 1, m0 + 1, B), _u(rng, 0.3, 1.0, B), _u(rng, 0.0, 180.0, B)]
    cols = main + second + pm + [g1, g2] + _draw_src_sersic(rng, B) \
        + _draw_src_sersic(rng, B, r=(0.05, 0.15)) + gauss + _draw_lens_light(rng, B) \
        + [_u(rng, 0.0, 0.02, B)]
    return np.stack(cols, axis=1)


HST_MODELS = ("sie", "shear", "src_sersic", "fg_sersic", "sky")
SLACS_MODELS = ("sie", "shear", "src_sersic", "src_sersic", "fg_sersic", "sky")
MULTI_MODELS = ("sie", "sie", "point", "shear", "src_sersic", "src_sersic", "src_gauss",
                "fg_sersic", "sky")

MOCK_MODELS = ("sie", "fg_sersic", "src_sersic")
_MOCK_TRUTH = [0.0, 0.0, 1.3624, 0.75, 20.0,
               0.0, 0.0, 2.0, mag_of_flux(3000.0), 4.0, 0.75, 20.0,
               0.12, -0.08, 0.2, mag_of_flux(30.0), 2.0, 0.5, 100.0]


def _draw_mock(rng, B):
    """lens fixed type, sources with n in [0.5, 8], q in [0.1, 1],
    r in [0.1, 0.4]", placed in a disc about the caustic; host n = 4 (de Vaucouleurs, R12)."""
    t = np.tile(np.array(_MOCK_TRUTH), (B, 1))
    t[:, [0, 1, 5, 6]] += rng.uniform(-0.05, 0.05, size=(B, 4))
    t[:, 2] = rng.uniform(1.0, 1.5, size=B)
    t[:, 3] = rng.uniform(0.5, 1.0, size=B)
    t[:, 4] = rng.uniform(0.0, 180.0, size=B)
    t[:, 7] *= rng.uniform(0.8, 1.2, size=B)
    sx, sy = _disc(rng, 0.5, B)
    t[:, 12], t[:, 13] = sx, sy
    t[:, 14] = rng.uniform(0.1, 0.4, size=B)
    t[:, 16] = rng.uniform(0.5, 8.0, size=B)
    t[:, 17] = rng.uniform(0.1, 1.0, size=B)
    t[:, 18] = rng.uniform(0.0, 180.0, size=B)
    return t


_HST_TRUTH = [0.02, -0.03, 1.2, 0.75, 35.0, 0.03, -0.02,
              0.15, 0.10, 0.15, mag_of_flux(20.0), 1.5, 0.6, 70.0,
              0.02, -0.03, 1.0, mag_of_flux(2000.0), 4.0, 0.8, 30.0, 0.01]
_SLACS_TRUTH = _HST_TRUTH[:14] + [-0.10, 0.22, 0.08, mag_of_flux(8.0), 1.0, 0.7, 120.0] \
    + _HST_TRUTH[14:]
_MULTI_TRUTH = [0.02, -0.03, 1.2, 0.75, 35.0, 1.4, -0.9, 0.4, 0.85, 110.0,
                -0.9, 0.75, math.sqrt(1e-3) * 1.2, 0.03, -0.02,
                0.15, 0.10, 0.15, mag_of_flux(20.0), 1.5, 0.6, 70.0,
                -0.10, 0.22, 0.08, mag_of_flux(8.0), 1.0, 0.7, 120.0,
                0.30, -0.15, 0.06, mag_of_flux(5.0), 0.8, 20.0,
                0.02, -0.03, 1.0, mag_of_flux(2000.0), 4.0, 0.8, 30.0, 0.01]


J0808_MODELS = ("sie", "sie", "fg_sersic", "fg_sersic", "fg_sersic", "src_sersic", "src_sersic", "sky")
_J0808_TRUTH = [0.0, 0.0, 1.17, 0.80, 9.4,                       # main lens (Table 3: b, q, PA)
                0.9, -0.7, 0.33, 0.99, 111.0,                    # companion
                0.0, 0.0, 0.9, mag_of_flux(2500.0), 4.0, 0.8, 10.0,
                0.0, 0.0, 0.25, mag_of_flux(600.0), 1.2, 0.7, 15.0,
                0.9, -0.7, 0.3, mag_of_flux(400.0), 2.5, 0.9, 100.0,
                0.12, 0.08, 0.12, mag_of_flux(25.0), 1.5, 0.6, 60.0,
                0.05, 0.15, 0.07, mag_of_flux(10.0), 1.0, 0.8, 140.0, 0.005]


def _draw_j0808(rng, B):
    """two SIEs, two + one foreground Sersic components, two source components.
    Priors a few tenths around the stand-in truth; the companion is nearly round (Table 3)."""
    t = np.tile(np.array(_J0808_TRUTH), (B, 1))
    t[:, [0, 1, 5, 6, 10, 11, 17, 18, 24, 25]] += rng.uniform(-0.05, 0.05, size=(B, 10))
    t[:, 2] = rng.uniform(0.9, 1.4, size=B)
    t[:, 3] = rng.uniform(0.5, 1.0, size=B)
    t[:, 4] = rng.uniform(0.0, 180.0, size=B)
    t[:, 7] = rng.uniform(0.2, 0.5, size=B)
    t[:, 8] = rng.uniform(0.8, 1.0, size=B)
    t[:, 9] = rng.uniform(0.0, 180.0, size=B)
    for o, nmax in ((10, 6.0), (17, 3.0), (24, 4.0)):
        t[:, o + 2] *= rng.uniform(0.8, 1.25, size=B)
        t[:, o + 4] = rng.uniform(0.8, nmax, size=B)
        t[:, o + 5] = rng.uniform(0.5, 1.0, size=B)
        t[:, o + 6] = rng.uniform(0.0, 180.0, size=B)
    for o in (31, 38):
        sx, sy = _disc(rng, 0.4, B)
        t[:, o], t[:, o + 1] = sx, sy
        t[:, o + 2] = rng.uniform(0.05, 0.25, size=B)
        t[:, o + 4] = rng.uniform(0.5, 4.0, size=B)
        t[:, o + 5] = rng.uniform(0.3, 1.0, size=B)
        t[:, o + 6] = rng.uniform(0.0, 180.0, size=B)
    t[:, 45] = rng.uniform(0.0, 0.01, size=B)
    return t


class Config:
    """One synthetic workload: geometry, model list, rule, PSF, mask, truth, batch draw."""

    def __init__(self, index, name, H, W, scale, models, quad, psf, mask, truth, B, draw,
                 sigma_sky, gain, zp=0.0):
        self.index, self.name = index, name
        self.H, self.W, self.scale = H, W, scale
        self.models, self.quad, self.psf, self.mask = tuple(models), quad, psf, mask
        self.truth = np.asarray(truth, dtype=np.float64)
        self.B, self._draw = B, draw
        self.sigma_sky, self.gain, self.zp = sigma_sky, gain, zp
        assert self.truth.size == num_params(models)

    @property
    def P(self):
        return num_params(self.models)

    def rng(self, stream):
        return np.random.default_rng([SEED0 + self.index, stream])

    def batch(self, B=None, stream=2):
        """params[B][P] float32, drawn from the config's priors (seeded)."""
        B = self.B if B is None else B
        return np.ascontiguousarray(self._draw(self.rng(stream), B), dtype=np.float32)

    def observe(self, truth_model):
        """(image f32, weight f32) from the noiseless truth image L* rendered by the caller:
        s^2 = sigma_sky^2 + max(L*, 0)/gain, d = L* + N(0, s^2), w = 1/s^2."""
        t = np.asarray(truth_model, dtype=np.float64).reshape(self.H, self.W)
        var = self.sigma_sky ** 2 + (np.maximum(t, 0.0) / self.gain if self.gain else 0.0)
        noise = self.rng(1).standard_normal(t.shape) * np.sqrt(var)
        w = np.broadcast_to(1.0 / var, t.shape)
        return (t + noise).astype(np.float32), np.ascontiguousarray(w, dtype=np.float32)

    def n_traced(self, extra_rows=0):
        """m_d: pixels in the PSF-dilated unmasked set (what loglike must ray-trace);
        extra_rows widens every window by that many rows each way."""
        if self.mask is None:
            return self.H * self.W
        return int(dilate_mask(self.mask, self.psf, extra_rows).sum())


def dilate_mask(mask, psf, extra_rows=0):
    """Pixels any unmasked pixel's PSF window (with border clamping) touches."""
    m = np.asarray(mask, dtype=bool)
    if psf is None and not extra_rows:
        return m
    p, q = ((psf.shape[0] - 1) // 2, (psf.shape[1] - 1) // 2) if psf is not None else (0, 0)
    p += extra_rows
    H, W = m.shape
    rows = np.zeros_like(m)
    for k in range(-p, p + 1):                      # unmasked row i reads row clamp(i + k)
        np.logical_or.at(rows, (np.clip(np.arange(H) + k, 0, H - 1), slice(None)), m)
    out = np.zeros_like(m)
    rt = np.ascontiguousarray(rows.T)
    ot = np.zeros_like(rt)
    for l in range(-q, q + 1):
        np.logical_or.at(ot, (np.clip(np.arange(W) + l, 0, W - 1), slice(None)), rt)
    out = np.ascontiguousarray(ot.T)
    return out


def _tiny():
    sigma, s = 0.1, 0.05
    F = 2 * math.pi * sigma * sigma / (s * s)      # so that I_0 = 1 per pixel
    truth = [0.0, 0.0, 0.8, 0.1, 0.0, sigma, mag_of_flux(F), 1.0, 0.0]

    def draw(rng, B):
        t = np.array(truth)
        p = np.tile(t, (B, 1))
        for c, v in enumerate(truth):
            if c in (7, 8):                         # q, pa fixed
                continue
            if c in (0, 1, 3, 4):                   # positions: +-0.02" about the truth
                p[:, c] = v + rng.uniform(-0.02, 0.02, size=B)
            else:                                   # +-20 % of the truth
                p[:, c] = v * rng.uniform(0.8, 1.2, size=B)
        return p

    return Config(0, "tiny", 32, 32, s, ("sis", "src_gauss"), gauss_legendre_rule(2), None, None,
                  truth, 16, draw, 0.01, 0.0)


def get_config(index):
    if index == 0:
        return _tiny()
    if index == 1:
        return Config(1, "hst", 100, 100, 0.05, HST_MODELS, gauss_legendre_rule(3),
                      gaussian_psf(9, 2.0), None, _HST_TRUTH, 1024, _draw_hst, 0.005, 2000.0)
    if index == 2:
        return Config(2, "slacs", 200, 200, 0.05, SLACS_MODELS, subsample_rule(4),
                      moffat_psf(21, 2.4, 3.0), annulus_mask(200, 200, 10.0, 72.06), _SLACS_TRUTH,
                      4096, lambda rng, B: _draw_hst(rng, B, n_src=2), 0.005, 2000.0)
    if index == 3:
        return Config(3, "multi", 256, 256, 0.05, MULTI_MODELS, gauss_legendre_rule(5),
                      moffat_psf(15, 2.0, 3.0), None, _MULTI_TRUTH, 4096, _draw_multi, 0.005, 2000.0)
    if index == 4:
        return Config(4, "euclid", 512, 512, 0.1, HST_MODELS, subsample_rule(4),
                      moffat_psf(31, 1.8, 2.5), None, _HST_TRUTH, 16384, _draw_hst, 0.005, 2000.0)
    if index == 5:
        # The paper's own mock scenario: 120x120 at
        # 0.05"/px, SIE + de Vaucouleurs host + Sersic source (18 parameters), default g3k7 rule
        # (PAPER.md:166).  Context for "thousands of individual parameter settings per second"
        # (PAPER.md:445), not one of BASELINE.json's configs.  The TinyTim PSF is not in the
        # container: a 15x15 Moffat (beta = 3, FWHM 0.1") stands in for it.
        return Config(5, "mock", 120, 120, 0.05, MOCK_MODELS, gauss_kronrod_rule(7),
                      moffat_psf(15, 2.0, 3.0), None, _MOCK_TRUTH, 4096, _draw_mock, 0.005, 2000.0)
    if index == 6:
        # The paper's largest fitted model, SDSS J0808+4706: two SIEs, three
        # foreground and two source Sersic components, sky -- 46 parameters here (the paper ties
        # centres and counts 35).  5" cut-out at 0.05"/px (Fig. 5), sub4 rule, a
        # 15x15 Moffat standing in for the HST PSF.  Context row, not one of BASELINE.json's.
        return Config(6, "j0808", 100, 100, 0.05, J0808_MODELS, subsample_rule(4),
                      moffat_psf(15, 2.0, 3.0), None, _J0808_TRUTH, 2048, _draw_j0808, 0.005, 2000.0)
    raise ValueError("config index 0..6")


def shrunk(cfg, H, W, B):
    """A smaller copy of a config (same models, rule, PSF, priors) for parity tests the
    oracle finishes in seconds; the mask, if any, is rebuilt as an annulus of the same shape."""
    mask = None
    if cfg.mask is not None:
        mask = annulus_mask(H, W, 0.05 * min(H, W), 0.36 * min(H, W))
    return Config(cfg.index, cfg.name + "_small", H, W, cfg.scale, cfg.models, cfg.quad, cfg.psf,
                  mask, cfg.truth, B, cfg._draw, cfg.sigma_sky, cfg.gain, cfg.zp)
