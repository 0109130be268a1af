"""The device-resident nested-sampling driver (lensed_ns_run, csrc/nested.cu) against the CPU
oracle driver (oracle/nested_oracle.py) running the oracle likelihood: the same counter-based
random numbers on both sides, so short runs agree point by point and full runs agree in ln Z and
in the posterior within the sampler's own statistical error."""
import math

import numpy as np
import pytest

from oracle import lensed_oracle as orc
from oracle import nested_oracle as ns
from paper_1505_07674_b200 import synth
from tests.cases import Problem

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def L():
    import torch
    assert torch.cuda.is_available()
    from paper_1505_07674_b200 import lensed
    lensed.lib()
    return lensed


def _tiny_priors(cfg):
    """BASELINE.json `tiny`: +-20 % of the truth, zero-valued positions +-0.02", q and PA fixed"""
    t = cfg.truth
    lo, hi = t.copy(), t.copy()
    for c, v in enumerate(t):
        if c in (7, 8):
            continue
        if c in (0, 1, 3, 4):
            lo[c], hi[c] = v - 0.02, v + 0.02
        else:
            lo[c], hi[c] = sorted((0.8 * v, 1.2 * v))
    return lo.astype(np.float32), hi.astype(np.float32)


def _gpu_run(L, prob, lo, hi, cap, **kw):
    import torch
    P = len(lo)
    samples = torch.zeros((cap, P), dtype=torch.float32, device="cuda")
    logl = torch.zeros(cap, dtype=torch.float32, device="cuda")
    logw = torch.zeros(cap, dtype=torch.float32, device="cuda")
    h = prob.create()
    try:
        res = L.lensed_ns_run(h, lo, hi, samples_dev=samples, logl_dev=logl, logw_dev=logw, **kw)
    finally:
        L.lensed_destroy(h)
    n = res["n_samples"]
    res.update(samples=samples[:n].cpu().numpy(), logl=logl[:n].cpu().numpy().astype(np.float64),
               logw=logw[:n].cpu().numpy().astype(np.float64))
    return res


def _moments(res):
    w = np.exp(res["logw"] - res["logw"].max())
    w /= w.sum()
    mean = (w[:, None] * res["samples"]).sum(axis=0)
    return mean, np.sqrt((w[:, None] * (res["samples"] - mean) ** 2).sum(axis=0))


def test_generator_known_answers_on_the_library_side(L):
    for line in open(__file__.replace("test_nested_gpu.py", "golden/philox_kat.txt")):
        if line.strip() and not line.startswith("#"):
            v = [int(x, 16) for x in line.split()]
            assert L.lensed_ns_philox(v[:4], v[4:6]) == v[6:]


def test_three_rounds_agree_point_by_point_with_the_oracle_driver(L):
    """Same seed, same options, three rounds: initial draw, bound, proposals, prior transform,
    acceptance against the rising threshold, weights and the final live-point step must give the
    same set of points with the same weights (float32 parameter vectors: exactly)."""
    cfg = synth.get_config(0)
    prob = Problem(cfg)
    lo, hi = _tiny_priors(cfg)
    kw = dict(n_live=64, batch=48, tol=1e-9, enlarge=1.25, seed=2024, max_rounds=3)
    # max_rounds = 3 is not a multiple of the driver's convergence-check interval (4): it must stop at 3
    ref = ns.run(lambda t: prob.oracle_loglike(t.astype(np.float32), want_model=False), lo, hi, **kw)
    got = _gpu_run(L, prob, lo, hi, 4096, **kw)
    assert got["n_rounds"] == 3 and ref["n_rounds"] == 3 and not got["converged"]
    assert got["n_likelihood"] == ref["n_likelihood"] == 64 + 3 * 48
    assert got["n_dead"] == ref["n_dead"] and got["n_samples"] == len(ref["logl"])
    nd = ref["n_dead"]
    assert np.array_equal(got["samples"][:nd], ref["samples"][:nd].astype(np.float32))       # deaths, in order
    key = lambda a: a[np.lexsort(a.T[::-1])]
    assert np.array_equal(key(got["samples"][nd:]), key(ref["samples"][nd:].astype(np.float32)))   # live set
    assert np.allclose(got["logl"][:nd], ref["logl"][:nd], rtol=1e-5)
    assert got["ln_z"] == pytest.approx(ref["ln_z"], rel=1e-5)
    assert got["information"] == pytest.approx(ref["information"], rel=1e-3, abs=1e-3)
    assert np.exp(got["logw"]).sum() == pytest.approx(1.0, rel=1e-4)


def test_large_batch_and_ragged_live_set_agree_point_by_point(L):
    """More candidates per round than the update kernel stages at once (1024) and a live set that
    is not a multiple of the warp size: the same deaths, in the same order, with the same weights
    as the oracle driver's candidate-by-candidate loop."""
    cfg = synth.get_config(0)
    prob = Problem(cfg)
    lo, hi = _tiny_priors(cfg)
    kw = dict(n_live=70, batch=1300, tol=1e-12, enlarge=1.3, seed=99, max_rounds=4)
    ref = ns.run(lambda t: prob.oracle_loglike(t.astype(np.float32), want_model=False), lo, hi, **kw)
    got = _gpu_run(L, prob, lo, hi, 8192, **kw)
    assert got["n_rounds"] == 4 and got["n_dead"] == ref["n_dead"] and got["n_samples"] == len(ref["logl"])
    nd = ref["n_dead"]
    assert np.array_equal(got["samples"][:nd], ref["samples"][:nd].astype(np.float32))
    # ln w itself is a function of the death count only; logw carries logL (FP32 vs the oracle's double)
    assert np.allclose(got["logw"], ref["logw"], rtol=2e-5, atol=2e-2)
    assert got["ln_z"] == pytest.approx(ref["ln_z"], rel=1e-5)
    assert got["information"] == pytest.approx(ref["information"], rel=1e-3, abs=1e-3)


def test_tiny_config_evidence_and_posterior_match_the_oracle_driver_and_recover_the_truth(L):
    cfg = synth.get_config(0)
    prob = Problem(cfg)
    lo, hi = _tiny_priors(cfg)
    kw = dict(n_live=300, batch=256, tol=1e-3, enlarge=1.2, seed=7)
    got = _gpu_run(L, prob, lo, hi, 60000, **kw)
    # a different seed for the oracle driver: "within 3 sigma" then compares two independent runs
    ref = ns.run(lambda t: prob.oracle_loglike(t.astype(np.float32), want_model=False), lo, hi, **dict(kw, seed=1007))
    assert got["converged"] and ref["converged"]
    err = math.hypot(got["ln_z_err"], ref["ln_z_err"])
    assert abs(got["ln_z"] - ref["ln_z"]) < 3.0 * err, (got["ln_z"], ref["ln_z"], err)
    assert got["information"] == pytest.approx(ref["information"], rel=0.1)
    assert got["ln_z_err"] == pytest.approx(math.sqrt(got["information"] / 300), rel=1e-9)
    mg, sg = _moments(got)
    mr, sr = ns.posterior_moments(ref)
    free = np.flatnonzero(hi > lo)
    assert np.all(np.abs(mg[free] - mr[free]) < 0.5 * sr[free])            # same posterior ...
    assert np.all(np.abs(sg[free] / sr[free] - 1.0) < 0.35)
    assert np.all(np.abs(mg[free] - cfg.truth[free]) < 4.0 * sr[free])      # ... that holds the truth
    assert np.all(sg[[7, 8]] < 1e-12)                                        # fixed parameters stay fixed
    assert got["n_likelihood"] >= 300 + got["n_rounds"] * 256
    assert np.all(np.diff(got["logl"][:got["n_dead"]]) >= 0)               # deaths in order of likelihood


def test_shrunk_hst_case_with_an_image_plane_prior(L):
    """SIE + shear + Sersic source + lens light + sky on a 40 x 36 image; six free parameters with
    priors a few posterior widths around the truth, the source position drawn in the IMAGE plane
    around one of its images and mapped through each vector's own lens."""
    cfg = synth.shrunk(synth.get_config(1), 40, 36, 4)
    prob = Problem(cfg)
    t = cfg.truth.astype(np.float64)
    # image-plane position of the source's brightest image under the true lens
    _, model = prob.oracle_loglike(t.astype(np.float32)[None], want_model=True)
    fg = orc.render(cfg.H, cfg.W, cfg.scale, cfg.psf, cfg.quad, synth.kind_ids(("fg_sersic", "sky")), t[14:].astype(np.float32))[0]
    i, j = np.unravel_index(np.argmax(model[0] - fg), fg.shape)
    img = np.array([(j - (cfg.W - 1) / 2) * cfg.scale, (i - (cfg.H - 1) / 2) * cfg.scale])
    lo, hi = t.copy(), t.copy()
    lo[2], hi[2] = t[2] - 0.03, t[2] + 0.03                 # Einstein radius
    lo[3], hi[3] = t[3] - 0.05, t[3] + 0.05                 # axis ratio
    lo[7:9], hi[7:9] = img - 0.06, img + 0.06               # source (x, y): an IMAGE-plane box
    lo[9], hi[9] = 0.8 * t[9], 1.25 * t[9]                  # source radius
    lo[10], hi[10] = t[10] - 0.3, t[10] + 0.3               # source magnitude
    lo, hi = lo.astype(np.float32), hi.astype(np.float32)
    src = [2]                                               # index of src_sersic in the model list
    kw = dict(n_live=200, batch=256, tol=1e-2, enlarge=1.3, seed=11)

    def transform(theta):
        out = theta.copy()
        for b in range(len(out)):
            out[b, 7:9] = orc.source_position(prob.kinds, theta[b], theta[b, 7:9][None])[0]
        return out.astype(np.float32).astype(np.float64)

    got = _gpu_run(L, prob, lo, hi, 40000, image_plane_sources=src, **kw)
    ref = ns.run(lambda th: prob.oracle_loglike(th.astype(np.float32), want_model=False), lo, hi, transform=transform,
                 **dict(kw, seed=1011))                     # independent of the GPU run's seed
    assert got["converged"] and ref["converged"]
    err = math.hypot(got["ln_z_err"], ref["ln_z_err"])
    assert abs(got["ln_z"] - ref["ln_z"]) < 3.0 * err, (got["ln_z"], ref["ln_z"], err)
    mg, sg = _moments(got)
    mr, sr = ns.posterior_moments(ref)
    for c in (2, 3, 7, 8, 9, 10):
        assert abs(mg[c] - mr[c]) < 0.6 * sr[c], (c, mg[c], mr[c], sr[c])
    # the samples hold SOURCE-plane positions (after the map): near the true source position
    assert abs(mg[7] - t[7]) < 5 * sr[7] + 0.01 and abs(mg[8] - t[8]) < 5 * sr[8] + 0.01


def test_tied_parameters_follow_the_parameter_they_are_tied_to(L):
    """the mass centre forced onto the centre of the light.  tied_to makes a parameter
    take the drawn value of another; the oracle driver does the same through its transform hook.
    tiny config: the source position (x, y) tied to the lens position, which is free."""
    cfg = synth.get_config(0)
    prob = Problem(cfg)
    lo, hi = _tiny_priors(cfg)
    lo[3:5] = hi[3:5] = 0.0                      # source (x, y): not drawn
    tied = -np.ones(len(lo), dtype=np.int32)
    tied[3], tied[4] = 0, 1

    def transform(theta):
        out = theta.copy()
        out[:, 3], out[:, 4] = out[:, 0], out[:, 1]
        return out

    kw = dict(n_live=48, batch=64, tol=1e-12, enlarge=1.3, seed=3, max_rounds=4)
    ref = ns.run(lambda t: prob.oracle_loglike(t.astype(np.float32), want_model=False), lo, hi, transform=transform, **kw)
    got = _gpu_run(L, prob, lo, hi, 4096, tied_to=tied, **kw)
    nd = ref["n_dead"]
    assert got["n_dead"] == nd and nd > 0
    assert np.array_equal(got["samples"][:nd], ref["samples"][:nd].astype(np.float32))
    assert np.array_equal(got["samples"][:, 3], got["samples"][:, 0]) and np.array_equal(got["samples"][:, 4], got["samples"][:, 1])
    h = prob.create()
    try:
        bad = tied.copy(); bad[0] = 3            # a chain: 3 -> 0 -> 3
        with pytest.raises(L.LensedError) as e:
            L.lensed_ns_run(h, lo, hi, tied_to=bad, **kw)
        assert e.value.status == L.EINVAL
        lo2, hi2 = lo.copy(), hi.copy(); hi2[3] = 0.1     # a tied parameter with a free prior
        with pytest.raises(L.LensedError):
            L.lensed_ns_run(h, lo2, hi2, tied_to=tied, **kw)
    finally:
        L.lensed_destroy(h)


def test_bad_arguments_are_rejected(L):
    cfg = synth.get_config(0)
    lo, hi = _tiny_priors(cfg)
    h = Problem(cfg).create()
    try:
        for kw, status in ((dict(n_live=4), L.EINVAL), (dict(n_live=5000), L.EINVAL), (dict(batch=0), L.EINVAL),
                           (dict(tol=0.0), L.EINVAL), (dict(enlarge=0.5), L.EINVAL),
                           (dict(image_plane_sources=[0]), L.EINVAL)):          # model 0 is the lens
            with pytest.raises(L.LensedError) as e:
                L.lensed_ns_run(h, lo, hi, **dict(dict(n_live=32, batch=8, max_rounds=2), **kw))
            assert e.value.status == status, kw
        with pytest.raises(L.LensedError):
            L.lensed_ns_run(h, hi, lo)                                          # hi < lo
        with pytest.raises(L.LensedError):
            L.lensed_ns_run(h, lo, lo)                                          # nothing free
    finally:
        L.lensed_destroy(h)


@pytest.mark.parametrize("seed", [1, 2])
def test_evidence_of_a_sky_only_model_equals_its_closed_form(L, seed):
    """A pin of the GPU sampler that does not go through oracle/nested_oracle.py (which follows the
    kernel's structure).  With the model list ("sky",) eq. 17 is a parabola in the
    one parameter: logL(level) = -1/2 [A (level - mu)^2 + C] with A = sum w, mu = sum w d / A,
    C = sum w (d - mu)^2, so under a uniform prior on [lo, hi]
        Z = exp(-C/2) sqrt(2 pi / A) [Phi((hi - mu) sqrt A) - Phi((lo - mu) sqrt A)] / (hi - lo)
    and, the prior being many posterior widths wide, H = <ln L> - ln Z = -C/2 - 1/2 - ln Z.
    (tol = 0.02, not smaller: lensed_loglike returns FP32, so in one dimension the live points reach
    the plateau where every logL rounds to the same float -- |level - mu| < ~0.003 posterior widths
    here -- before a remaining-evidence fraction of 1e-4 is reached, and a draw that only ties the
    threshold is never accepted.  The live points' share is added at the end either way.)"""
    import torch
    rng = np.random.default_rng(40 + seed)
    H, W, sigma, level = 12, 10, 0.05, 1.3
    d = (level + sigma * rng.standard_normal((H, W))).astype(np.float32)
    w = np.full((H, W), 1.0 / sigma ** 2, dtype=np.float32)
    A = float(w.astype(np.float64).sum())
    mu = float((w.astype(np.float64) * d).sum() / A)
    C = float((w.astype(np.float64) * (d - mu) ** 2).sum())
    s = 1.0 / math.sqrt(A)
    lo = np.array([mu - 25.0 * s], dtype=np.float32)
    hi = np.array([mu + 15.0 * s], dtype=np.float32)
    phi = lambda x: 0.5 * (1.0 + math.erf(x / math.sqrt(2.0)))
    ln_z = -0.5 * C + math.log(math.sqrt(2.0 * math.pi / A) * (phi((hi[0] - mu) / s) - phi((lo[0] - mu) / s)) / float(hi[0] - lo[0]))
    info = -0.5 * C - 0.5 - ln_z
    cap = 40000
    samples = torch.zeros((cap, 1), dtype=torch.float32, device="cuda")
    logl = torch.zeros(cap, dtype=torch.float32, device="cuda")
    logw = torch.zeros(cap, dtype=torch.float32, device="cuda")
    h = L.lensed_create(d, w, None, None, synth.get_config(0).quad, synth.kind_ids(("sky",)), 0.05, 0.0)
    try:
        res = L.lensed_ns_run(h, lo, hi, n_live=400, batch=128, tol=0.02, enlarge=1.2, seed=seed, max_rounds=2000,
                              samples_dev=samples, logl_dev=logl, logw_dev=logw)
    finally:
        L.lensed_destroy(h)
    assert res["converged"], res
    assert abs(res["ln_z"] - ln_z) < 3.0 * res["ln_z_err"], (res["ln_z"], ln_z, res["ln_z_err"])
    assert res["information"] == pytest.approx(info, rel=0.15)
    n = res["n_samples"]
    wgt = np.exp(logw[:n].cpu().numpy().astype(np.float64))
    x = samples[:n, 0].cpu().numpy().astype(np.float64)
    mean = (wgt * x).sum() / wgt.sum()
    sd = math.sqrt((wgt * (x - mean) ** 2).sum() / wgt.sum())
    assert abs(mean - mu) < 0.25 * s and sd == pytest.approx(s, rel=0.15)
