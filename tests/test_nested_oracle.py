"""Pins of the CPU nested-sampling oracle (oracle/nested_oracle.py) against what does not depend
on it: the generator's published known-answer vectors, moments of its uniforms / normals, the
geometry of the ellipsoidal bound, and the closed-form evidence and posterior of Gaussian
likelihoods under a uniform prior.  No GPU."""
import math
import os

import numpy as np
import pytest
from scipy import special

from oracle import nested_oracle as ns

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def test_philox_known_answer_vectors():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "philox_kat.txt")) if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        out = ns.philox4x32(np.uint32(v[0]), np.uint32(v[1]), np.uint32(v[2]), np.uint32(v[3]), v[4], v[5])
        assert [int(x) for x in out] == v[6:]
    # vectorised over counters = one call per counter
    a = np.arange(5, dtype=np.uint32)
    many = ns.philox4x32(a, 7, 9, 1, 123, 456)
    for i in range(5):
        one = ns.philox4x32(np.uint32(i), np.uint32(7), np.uint32(9), np.uint32(1), 123, 456)
        assert [int(w[i]) for w in many] == [int(w) for w in one]


def test_uniforms_and_normals_have_the_right_moments():
    i = np.arange(200000, dtype=np.uint32)
    u = np.concatenate(ns.uniforms4(77, 0, i, 3, 5))
    assert u.min() > 0.0 and u.max() < 1.0
    assert abs(u.mean() - 0.5) < 3e-3 and abs(u.var() - 1 / 12) < 1e-3
    z = np.stack(ns.normals4(77, 1, i, 3, 5))
    assert abs(z.mean()) < 5e-3 and abs(z.var() - 1.0) < 1e-2
    assert abs(np.mean(z ** 4) - 3.0) < 0.05                      # kurtosis of a normal
    assert np.abs(np.corrcoef(z)[np.triu_indices(4, 1)]).max() < 0.01
    # different streams / counters are different numbers
    assert not np.array_equal(ns.uniforms4(77, 0, i, 3, 5)[0], ns.uniforms4(77, 1, i, 3, 5)[0])
    assert not np.array_equal(ns.uniforms4(77, 0, i, 3, 5)[0], ns.uniforms4(78, 0, i, 3, 5)[0])


def test_bound_holds_every_live_point_and_proposals_are_uniform_inside_it():
    rng = np.random.default_rng(3)
    d = 5
    A = rng.normal(size=(d, d)) * 0.03
    u = 0.5 + rng.normal(size=(300, d)) @ A.T
    m, G, s = ns.bound(u, 1.0)
    y = np.linalg.solve(G, (u - m).T)
    r = np.sqrt((y * y).sum(axis=0)) / s
    assert r.max() == pytest.approx(1.0, abs=1e-12)               # tight at enlarge = 1
    assert np.allclose(G @ G.T, np.cov(u.T, bias=True), rtol=1e-10, atol=1e-14)
    m2, G2, s2 = ns.bound(u, 1.3)
    assert s2 == pytest.approx(1.3 * s, rel=1e-14)
    x = ns.propose(11, 0, 20000, m, G, s)
    assert not np.isnan(x).any()                                  # the ellipsoid is well inside the cube
    rr = np.sqrt((np.linalg.solve(G, (x - m).T) ** 2).sum(axis=0)) / s
    assert rr.max() <= 1.0 + 1e-12
    for f in (0.5, 0.8):                                          # volume fraction inside radius f is f^d
        assert np.mean(rr < f) == pytest.approx(f ** d, abs=4 * math.sqrt(f ** d / len(rr)))
    # directions are isotropic in the whitened frame
    yy = np.linalg.solve(G, (x - m).T)
    assert np.abs(np.corrcoef(yy)[np.triu_indices(d, 1)]).max() < 0.03


def test_proposals_outside_the_unit_cube_are_redrawn_or_void():
    d = 3
    m, G = np.array([0.02, 0.5, 0.5]), np.eye(d) * 0.05
    x = ns.propose(5, 2, 4000, m, G, 1.0)
    ok = ~np.isnan(x[:, 0])
    assert ok.mean() > 0.99 and np.all((x[ok] > 0) & (x[ok] < 1))
    far = ns.propose(5, 2, 100, np.array([-3.0, 0.5, 0.5]), G, 1.0)
    assert np.isnan(far).all()                                    # never inside: void


def _gauss(mu, cov):
    P = np.linalg.inv(cov)

    def loglike(t):
        x = t - mu
        return -0.5 * np.einsum("bi,ij,bj->b", x, P, x)
    return loglike


def test_evidence_and_posterior_of_a_gaussian_likelihood_under_a_uniform_prior():
    """Z = int L dpi = (2 pi)^(d/2) sqrt(det C) / V for a Gaussian well inside the box; the
    estimate must sit within its own error bar (sqrt(H/N), Skilling 2006) of it, H itself near
    its closed form, and the weighted samples must give back mean and standard deviation."""
    d = 4
    lo, hi = np.array([-1.0, 0.0, 2.0, -3.0]), np.array([1.0, 4.0, 3.0, 5.0])
    mu = np.array([0.1, 2.5, 2.4, 0.5])
    sig = np.array([0.05, 0.2, 0.03, 0.3])
    cov = np.diag(sig ** 2)
    res = ns.run(_gauss(mu, cov), lo, hi, n_live=500, batch=128, tol=1e-4, seed=42)
    ln_z_true = 0.5 * d * math.log(2 * math.pi) + np.log(sig).sum() - np.log(hi - lo).sum()
    assert res["converged"]
    assert abs(res["ln_z"] - ln_z_true) < 3.0 * res["ln_z_err"] + 0.02
    # information H = int P ln(P/pi) = -ln Z_true - d/2 for a Gaussian posterior in a wide box
    assert res["information"] == pytest.approx(-ln_z_true - 0.5 * d, abs=0.5)
    assert res["ln_z_err"] == pytest.approx(math.sqrt(res["information"] / 500), rel=1e-12)
    mean, std = ns.posterior_moments(res)
    assert np.all(np.abs(mean - mu) < 0.15 * sig) and np.all(np.abs(std / sig - 1.0) < 0.1)
    assert np.exp(res["logw"]).sum() == pytest.approx(1.0, rel=1e-9)
    assert res["n_dead"] + 500 == len(res["logl"]) and np.all(np.diff(res["logl"][:res["n_dead"]]) >= 0)


def test_correlated_gaussian_truncated_by_the_box_and_fixed_parameters():
    """A strongly correlated likelihood (the ellipsoid must follow it) whose mode sits ON an edge
    of the box in one coordinate: Z picks up the factor 1/2 of the half Gaussian.  Two more
    parameters are fixed (lo == hi) and must not enter the sampling."""
    mu = np.array([0.0, 1.0])
    cov = np.array([[0.04, 0.018], [0.018, 0.01]])
    lo, hi = np.array([0.0, 7.0, 0.0, -2.0]), np.array([2.0, 7.0, 2.0, -2.0])   # x0 >= mu0: half of the mass

    def loglike(t):
        assert np.all(t[:, 1] == 7.0) and np.all(t[:, 3] == -2.0)
        return _gauss(mu, cov)(t[:, [0, 2]])
    res = ns.run(loglike, lo, hi, n_live=400, batch=64, tol=1e-4, seed=7)
    ln_z_true = math.log(2 * math.pi) + 0.5 * math.log(np.linalg.det(cov)) - math.log(4.0) + math.log(0.5)
    assert abs(res["ln_z"] - ln_z_true) < 3.0 * res["ln_z_err"] + 0.02
    mean, std = ns.posterior_moments(res)
    # half-normal in x0: mean sigma sqrt(2/pi); x1 follows through the correlation
    s0 = math.sqrt(cov[0, 0])
    assert mean[0] == pytest.approx(s0 * math.sqrt(2 / math.pi), abs=0.02)
    assert mean[2] == pytest.approx(1.0 + cov[0, 1] / cov[0, 0] * s0 * math.sqrt(2 / math.pi), abs=0.01)
    assert std[1] < 1e-12 and std[3] < 1e-12


def test_transform_hook_and_seed_reproducibility():
    lo, hi = np.zeros(2), np.ones(2)
    f = _gauss(np.array([0.3, 0.6]), np.diag([0.01, 0.01]))
    a = ns.run(f, lo, hi, n_live=100, batch=32, seed=3, tol=1e-2)
    b = ns.run(f, lo, hi, n_live=100, batch=32, seed=3, tol=1e-2)
    c = ns.run(f, lo, hi, n_live=100, batch=32, seed=4, tol=1e-2)
    assert a["ln_z"] == b["ln_z"] and a["ln_z"] != c["ln_z"]
    # a transform that swaps the coordinates: the likelihood sees the swapped vector
    sw = ns.run(f, lo, hi, n_live=100, batch=32, seed=3, tol=1e-2, transform=lambda t: t[:, ::-1].copy())
    mean, _ = ns.posterior_moments(sw)
    assert mean == pytest.approx([0.3, 0.6], abs=0.03)            # samples are stored after the transform
