"""One pass over the asynchronous machinery of the CUDA path at smoke size, meant to be run under
compute-sanitizer (SURVEY.md section 5 "Race detection / sanitizers"):

    compute-sanitizer --tool memcheck|racecheck|initcheck|synccheck python tests/sanitizer_driver.py

Not collected by pytest (the name does not start with test_).  It exercises: lensed_loglike and
lensed_render through the four convolution shapes x both tap paths (TMA stages, mbarrier parity,
independent one-warp workers, pad-cell writers), the three tracer kinds (built-in specialised,
specialised at run time, interpreting), the FP64 refinement both with a few flagged pixels and
with more flagged pixels than its queue holds (the in-place overflow path), two rounds of the
device-resident sampler, three clones on three streams, and lensed_chisq_static twice in a row.
Results are checked for finiteness and for agreement between the variants only (no oracle: the
sanitizer slows everything by 10-100x); parity is the business of tests/test_parity_gpu.py.
Prints one line per section and "SANITIZER_DRIVER_OK" at the end.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import torch  # noqa: E402

from paper_1505_07674_b200 import lensed as L, synth  # noqa: E402


def _inputs(cfg, seed):
    """image = a smooth positive ramp + seeded noise (no oracle render needed here), weight = 1 / sigma^2"""
    rng = np.random.default_rng(seed)
    yy, xx = np.mgrid[0:cfg.H, 0:cfg.W]
    image = (0.02 + 1e-4 * (xx + 2 * yy) + 0.005 * rng.standard_normal((cfg.H, cfg.W))).astype(np.float32)
    weight = np.full((cfg.H, cfg.W), 1.0 / 0.005 ** 2, dtype=np.float32)
    return image, weight


def _create(cfg, image, weight):
    return L.lensed_create(image, weight, cfg.mask, cfg.psf, cfg.quad, synth.kind_ids(cfg.models), cfg.scale, cfg.zp)


def _eval(h, params, H, W, render=True):
    p = torch.from_numpy(np.ascontiguousarray(params, dtype=np.float32)).cuda()
    logl = torch.empty(len(params), dtype=torch.float32, device="cuda")
    L.lensed_loglike(h, p, logl)
    model = None
    if render:
        model = torch.empty((len(params), H, W), dtype=torch.float32, device="cuda")
        L.lensed_render(h, p, model)
    torch.cuda.synchronize()
    return logl.cpu().numpy(), None if model is None else model.cpu().numpy()


def shapes_and_taps():
    # masked SLACS-like list (21 x 21 PSF: every shape fits) on a small frame with ragged tiles
    cfg = synth.shrunk(synth.get_config(2), 75, 93, 5)
    image, weight = _inputs(cfg, 1)
    params = cfg.batch(5)
    ref = None
    for global_taps in (0, 1):
        L.lensed_debug_force_global_taps(global_taps)
        h = _create(cfg, image, weight)
        L.lensed_debug_force_global_taps(0)
        try:
            assert L.lensed_uses_global_taps(h) == global_taps
            for shape in (3, 2, 1, 0):
                L.lensed_set_conv_shape(h, shape)
                logl, model = _eval(h, params, cfg.H, cfg.W)
                assert np.all(np.isfinite(logl)) and np.all(np.isfinite(model))
                if ref is None:
                    ref = (logl, model)
                assert np.array_equal(model, ref[1]), "rendered pixels differ between shapes / tap paths"
                assert np.allclose(logl, ref[0], rtol=1e-6)
        finally:
            L.lensed_destroy(h)
    print("shapes x taps: 4 x 2 ok")


def tracers():
    cfg = synth.shrunk(synth.get_config(1), 45, 52, 4)
    image, weight = _inputs(cfg, 2)
    params = cfg.batch(4)
    h = _create(cfg, image, weight)
    try:
        assert L.lensed_get_static_tracer(h) == 1
        a = _eval(h, params, cfg.H, cfg.W)
        L.lensed_set_static_tracer(h, 0)
        b = _eval(h, params, cfg.H, cfg.W)
        assert np.allclose(a[0], b[0], rtol=1e-4) and np.all(np.isfinite(b[1]))
    finally:
        L.lensed_destroy(h)
    # a list without a built-in signature: specialised at run time (or interpreted where NVRTC is missing)
    models = ("sie", "shear", "src_gauss", "src_gauss", "fg_gauss", "sky")
    truth = [0.02, -0.03, 0.5, 0.7, 35.0, 0.03, -0.02, 0.05, 0.08, 0.06, synth.mag_of_flux(30.0), 0.8, 20.0,
             -0.1, 0.02, 0.04, synth.mag_of_flux(10.0), 0.6, 100.0, 0.0, 0.01, 0.3, synth.mag_of_flux(400.0), 0.7, 60.0, 0.01]
    jcfg = synth.Config(9, "jit", 45, 52, 0.05, models, synth.gauss_legendre_rule(3), synth.gaussian_psf(7, 2.0), None, truth, 3,
                        lambda rng, B: np.tile(np.array(truth), (B, 1)), 0.01, 0.0)
    h = _create(jcfg, *_inputs(jcfg, 3))
    try:
        kind = L.lensed_get_static_tracer(h)
        logl, model = _eval(h, jcfg.batch(3), jcfg.H, jcfg.W)
        assert np.all(np.isfinite(logl)) and np.all(np.isfinite(model))
    finally:
        L.lensed_destroy(h)
    print("tracers: built-in, interpreting, run-time specialised (kind %d) ok" % kind)


def refinement():
    cfg = synth.shrunk(synth.get_config(5), 72, 66, 2)          # the paper's mock prior: n up to 8, cusps
    image, weight = _inputs(cfg, 4)
    h = _create(cfg, image, weight)
    try:
        params = cfg.batch(2)
        L.lensed_reset_profile(h)
        a, _ = _eval(h, params, cfg.H, cfg.W, render=False)
        few = L.lensed_get_refined(h)
        # one vector, every traced pixel flagged: more entries than the queue of a 1-vector chunk holds
        # (64 + 4096), so the scan kernel refines the overflow in place (refine.cu)
        L.lensed_set_refine(h, 1e-6)
        L.lensed_reset_profile(h)
        b, _ = _eval(h, params[:1], cfg.H, cfg.W, render=False)
        many = L.lensed_get_refined(h)
        assert np.all(np.isfinite(a)) and np.all(np.isfinite(b))
        assert many > 64 + 4096 and many >= few, (few, many)
        assert abs(b[0] - a[0]) <= 1e-4 * abs(a[0])
    finally:
        L.lensed_destroy(h)
    print("refinement: %d flagged pixels, then %d (queue overflow path) ok" % (few, many))


def sampler():
    cfg = synth.get_config(0)
    image, weight = _inputs(cfg, 5)
    t = cfg.truth
    lo, hi = t.copy(), t.copy()
    for c in (0, 1, 2, 5):
        lo[c], hi[c] = t[c] - 0.02, t[c] + 0.02
    h = _create(cfg, image, weight)
    try:
        res = L.lensed_ns_run(h, lo.astype(np.float32), hi.astype(np.float32), n_live=32, batch=24, tol=1e-9, seed=3, max_rounds=2)
        assert res["n_rounds"] == 2 and np.isfinite(res["ln_z"])
    finally:
        L.lensed_destroy(h)
    print("sampler: 2 rounds ok")


def clones():
    cfg = synth.shrunk(synth.get_config(1), 40, 36, 4)
    image, weight = _inputs(cfg, 6)
    h0 = _create(cfg, image, weight)
    handles = [h0, L.lensed_clone(h0), L.lensed_clone(h0)]
    try:
        streams = [torch.cuda.Stream() for _ in handles]
        ps = [torch.from_numpy(cfg.batch(24, stream=10 + i)).cuda() for i in range(3)]
        outs = [torch.empty(24, dtype=torch.float32, device="cuda") for _ in handles]
        torch.cuda.synchronize()
        for _ in range(2):
            for h, st, p, o in zip(handles, streams, ps, outs):
                L.lensed_loglike(h, p, o, stream=st.cuda_stream)
        torch.cuda.synchronize()
        single = torch.empty(24, dtype=torch.float32, device="cuda")
        for i in range(3):
            L.lensed_loglike(h0, ps[i], single)
            torch.cuda.synchronize()
            assert torch.equal(single, outs[i]), "clone %d on its own stream differs from a serial call" % i
    finally:
        for h in handles:
            L.lensed_destroy(h)
    print("clones: 3 handles on 3 streams ok")


def chisq_static():
    g = torch.Generator().manual_seed(1)
    n = 9001
    image, weight = torch.randn(n, generator=g).cuda(), (torch.rand(n, generator=g) + 0.5).cuda()
    for B in (7, 3):
        model = torch.randn(B, n, generator=g).cuda()
        logl = torch.empty(B, dtype=torch.float32, device="cuda")
        L.lensed_chisq_static(image, weight, model, logl)
        torch.cuda.synchronize()
        ref = -0.5 * (weight.double() * (image.double() - model.double()) ** 2).sum(dim=1)
        assert torch.allclose(logl.double(), ref, rtol=1e-6)
    print("chisq_static: two calls in a row ok")


if __name__ == "__main__":
    assert torch.cuda.is_available(), "needs a CUDA device"
    only = sys.argv[1:]
    for fn in (shapes_and_taps, tracers, refinement, sampler, clones, chisq_static):
        if not only or fn.__name__ in only:
            fn()
    print("SANITIZER_DRIVER_OK")
