"""Parity of the CUDA library (through the C ABI) against the CPU oracle, on a B200.

Element by element on seeded inputs at sizes the oracle finishes in seconds (several tiles
and a ragged tail), then at BASELINE.json's full sizes in the launch configuration
bench.py times, on sampled vectors the oracle computes one by one.  Tolerances are
north_star's: 1e-4 relative per rendered pixel above 1e-3 of the image peak, 1e-5 relative
on logL (tests/cases.py).
"""
import numpy as np
import pytest

from paper_1505_07674_b200 import synth
from tests.cases import LOGL_RTOL, PIXEL_RTOL, Problem, logl_errors, pixel_errors

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def L():
    import torch
    assert torch.cuda.is_available()
    from paper_1505_07674_b200 import lensed
    lensed.lib()
    return lensed


def _gpu_eval(L, h, params, H, W, render=True):
    import torch
    p = torch.from_numpy(np.ascontiguousarray(params, dtype=np.float32)).cuda()
    logl = torch.empty(p.shape[0], dtype=torch.float32, device="cuda")
    L.lensed_loglike(h, p, logl)
    model = None
    if render:
        model = torch.empty((p.shape[0], H, W), dtype=torch.float32, device="cuda")
        L.lensed_render(h, p, model)
        model = model.cpu().numpy()
    torch.cuda.synchronize()
    return logl.cpu().numpy(), model


def _check(L, prob, params, render=True, static=None):
    """static: None = whatever lensed_create picked; True = require the compile-time
    specialised tracer; False = force the interpreting one (include/lensed.h)."""
    c = prob.cfg
    h = prob.create()
    try:
        if static is True:
            assert L.lensed_get_static_tracer(h) == 1
        elif static is False:
            L.lensed_set_static_tracer(h, 0)
            assert L.lensed_get_static_tracer(h) == 0
        logl_g, model_g = _gpu_eval(L, h, params, c.H, c.W, render)
    finally:
        L.lensed_destroy(h)
    logl_o, model_o = prob.oracle_loglike(params, want_model=True)
    el = logl_errors(logl_g, logl_o)
    assert np.all(np.isfinite(logl_g))
    assert el.max() <= LOGL_RTOL, "logL rel err %.3g at vector %d" % (el.max(), el.argmax())
    if render:
        ep = pixel_errors(model_g, model_o)
        assert ep.max() <= PIXEL_RTOL, "pixel rel err %.3g at vector %d" % (ep.max(), ep.argmax())
    return el.max()


# ------------------------------------------------------------------ small, whole batches
def test_tiny_config_whole_batch(L):
    cfg = synth.get_config(0)
    prob = Problem(cfg)
    _check(L, prob, np.vstack([cfg.batch(), cfg.truth.astype(np.float32)[None]]))


@pytest.mark.parametrize("index,H,W,B", [(1, 90, 70, 24), (2, 75, 93, 12), (3, 70, 80, 8), (4, 101, 67, 6)])
def test_shrunk_configs_span_tiles_and_ragged_tails(L, index, H, W, B):
    cfg = synth.shrunk(synth.get_config(index), H, W, B)
    prob = Problem(cfg)
    _check(L, prob, np.vstack([cfg.batch(), cfg.truth.astype(np.float32)[None]]))


@pytest.mark.parametrize("index,H,W,B", [(0, 32, 32, 16), (1, 90, 70, 24), (2, 75, 93, 12), (3, 70, 80, 8), (4, 101, 67, 6),
                                         (5, 60, 64, 6), (6, 64, 70, 8)])
@pytest.mark.parametrize("static", [True, False])
def test_both_tracers_on_every_config_list(L, index, H, W, B, static):
    """The model lists of BASELINE.json's configs have a compile-time specialised tracer; the
    interpreting kernel must give the same answer (both against the oracle)."""
    cfg = synth.get_config(index)
    if index > 0:
        cfg = synth.shrunk(cfg, H, W, B)
    _check(L, Problem(cfg), cfg.batch(), static=static)


@pytest.mark.parametrize("static", [True, False])
def test_sie_axis_ratio_sweep_covers_every_polynomial_mode(L, static):
    """The SIE's atan / atanh approximations are chosen per vector from q (trace_math.cuh):
    thresholds q^2 = 0.84, 0.64, 0.5, 1/3, 0.25; one vector on each side of each, plus the
    extremes, in the HST-like list (SIE + shear + Sersic source + Sersic lens light + sky)."""
    cfg = synth.shrunk(synth.get_config(1), 64, 60, 4)
    assert cfg.models[0] == "sie"
    iq = 3                                             # SIE parameters: x, y, theta_E, q, PA
    qs = [1.0, 0.999, 0.93, 0.9, 0.82, 0.78, 0.72, 0.69, 0.6, 0.56, 0.52, 0.48, 0.3, 0.1, 0.03]
    params = np.tile(cfg.truth.astype(np.float32), (len(qs), 1))
    params[:, iq] = qs
    _check(L, Problem(cfg), params, static=static)


def test_paper_mock_scenario_gauss_kronrod_rule(L):
    """120x120 @ 0.05", SIE + de Vaucouleurs host + Sersic source (18
    parameters), default g3k7 rule -- 49 points, R = 7 register blocking."""
    base = synth.get_config(1)
    models = ("sie", "fg_sersic", "src_sersic")
    truth = [0.0, 0.0, 1.3624, 0.75, 20.0,
             0.0, 0.0, 2.0, synth.mag_of_flux(3000.0), 4.0, 0.75, 20.0,
             0.12, -0.08, 0.2, synth.mag_of_flux(30.0), 2.0, 0.5, 100.0]

    def draw(rng, B):
        t = np.tile(np.array(truth), (B, 1))
        t[:, [0, 1, 5, 6, 12, 13]] += rng.uniform(-0.05, 0.05, size=(B, 6))
        t[:, [2, 7, 14]] *= rng.uniform(0.8, 1.2, size=(B, 3))
        t[:, 16] = rng.uniform(0.5, 8.0, size=B)
        t[:, 17] = rng.uniform(0.1, 1.0, size=B)
        return t

    cfg = synth.Config(1, "mock", 60, 64, 0.05, models, synth.gauss_kronrod_rule(7), base.psf, None,
                       truth, 6, draw, 0.005, 2000.0)
    _check(L, Problem(cfg), cfg.batch())


# ------------------------------------------------- full sizes, bench launch configuration
@pytest.mark.parametrize("index,B,n_sample", [(1, 1024, 128), (2, 4096, 96), (3, 4096, 64), (4, 16384, 64), (5, 4096, 128),
                                              (6, 2048, 64)])
def test_full_size_configs_on_sampled_vectors(L, index, B, n_sample):
    """BASELINE.json's full sizes in the launch configuration bench.py times; 64-128 vectors per
    config spread over the batch, each against the oracle on every pixel, so that the test sees
    the tail of the prior (about one draw in a hundred has a source cusp on a pixel)."""
    import torch
    cfg = synth.get_config(index)
    prob = Problem(cfg)
    params = cfg.batch(B)
    h = prob.create()
    try:
        # the library traces the required set m_d plus one guard row each way (conv.cu pairing)
        assert cfg.n_traced() <= L.lensed_num_traced(h) <= cfg.n_traced(extra_rows=1)
        p = torch.from_numpy(params).cuda()
        logl = torch.empty(B, dtype=torch.float32, device="cuda")
        L.lensed_loglike(h, p, logl)
        logl2 = torch.empty(B, dtype=torch.float32, device="cuda")
        L.lensed_loglike(h, p, logl2)
        assert torch.equal(logl, logl2), "loglike is not bitwise reproducible"
        idx = np.linspace(0, B - 1, n_sample).astype(int)
        model = torch.empty((n_sample, cfg.H, cfg.W), dtype=torch.float32, device="cuda")
        L.lensed_render(h, p[torch.from_numpy(idx).cuda()].contiguous(), model)
        torch.cuda.synchronize()
        logl_g, model_g = logl.cpu().numpy(), model.cpu().numpy()
    finally:
        L.lensed_destroy(h)
    assert np.all(np.isfinite(logl_g))
    logl_o, model_o = prob.oracle_loglike(params[idx], want_model=True)
    assert logl_errors(logl_g[idx], logl_o).max() <= LOGL_RTOL
    assert pixel_errors(model_g, model_o).max() <= PIXEL_RTOL


# ------------------------------------------------------------------------------ edge cases
def _mini(models, truth, H=24, W=20, psf=None, mask=None, quad=None, scale=0.05):
    quad = synth.gauss_legendre_rule(2) if quad is None else quad
    return synth.Config(9, "mini", H, W, scale, models, quad, psf, mask, truth, 1,
                        lambda rng, B: np.tile(np.array(truth), (B, 1)), 0.01, 0.0)


def test_ray_through_the_lens_centre_and_degenerate_lenses(L):
    """psi = 0 / r = 0 exactly on a rule point (the rule has a point at the pixel centre and
    the lens sits on a pixel centre); q = 1 SIE; zero-strength lenses."""
    quad = np.array([[0.0, 0.0, 0.5], [0.25, -0.25, 0.5]])
    g = [0.1, -0.05, 0.12, synth.mag_of_flux(50.0), 0.8, 30.0]
    s = 0.05
    cx, cy = (10 - 9.5) * s, (12 - 11.5) * s          # centre of pixel (row 12, col 10) of 24 x 20
    for models, lens in ((("sie",), [cx, cy, 0.3, 0.7, 25.0]), (("sis",), [cx, cy, 0.3]),
                         (("point",), [cx, cy, 0.2]), (("sie",), [cx, cy, 0.3, 1.0, 40.0]),
                         (("sie",), [0.01, 0.02, 0.3, 0.999999, 40.0]),
                         (("sie", "sis", "point"), [cx, cy, 0.0, 0.5, 10.0, cx, cy, 0.0, cx, cy, 0.0])):
        cfg = _mini(models + ("src_gauss",), lens + g, quad=quad)
        _check(L, Problem(cfg), cfg.truth.astype(np.float32)[None])


def test_source_centre_on_a_rule_point(L):
    """R = 0 exactly: lg2(0) = -inf must give I = I0 (unlensed foreground Sersic on a pixel centre)."""
    quad = np.array([[0.0, 0.0, 1.0]])
    s = 0.05
    cfg = _mini(("fg_sersic", "sky"), [(10 - 9.5) * s, (12 - 11.5) * s, 0.2, synth.mag_of_flux(100.0), 2.5,
                                        0.6, 15.0, 0.01], quad=quad)
    _check(L, Problem(cfg), cfg.truth.astype(np.float32)[None])


def test_asymmetric_non_square_psf_pins_the_flip_and_axis_order(L):
    rng = np.random.default_rng(5)
    psf = rng.uniform(0.0, 1.0, size=(5, 9))
    psf[0, 8] = 7.0                                   # strongly off-centre tap: F_{-2,+4}
    cfg = _mini(("sis", "src_gauss", "sky"), [0.0, 0.0, 0.25, 0.05, 0.02, 0.08, synth.mag_of_flux(30.0),
                                                0.7, 50.0, 0.02], H=70, W=75, psf=psf)
    _check(L, Problem(cfg), cfg.truth.astype(np.float32)[None])


def test_largest_psf_and_one_column_image(L):
    psf = synth.moffat_psf(63, 3.0, 2.5, e1=0.1)
    cfg = _mini(("sie", "src_sersic", "sky"), [0.0, 0.0, 0.5, 0.8, 10.0, 0.1, 0.05, 0.1,
                                                 synth.mag_of_flux(30.0), 1.0, 0.7, 50.0, 0.02],
                H=66, W=40, psf=psf)
    _check(L, Problem(cfg), cfg.truth.astype(np.float32)[None])
    cfg = _mini(("fg_gauss",), [0.0, 0.0, 0.1, synth.mag_of_flux(30.0), 0.7, 50.0], H=37, W=1,
                psf=synth.gaussian_psf(5, 2.0))
    _check(L, Problem(cfg), cfg.truth.astype(np.float32)[None])


def test_invalid_vectors_give_minus_infinity_and_nan_image(L):
    import torch
    cfg = synth.shrunk(synth.get_config(1), 40, 36, 4)
    prob = Problem(cfg)
    params = cfg.batch(6)
    params[1, 3] = 1.5          # SIE q > 1
    params[2, 9] = -0.1         # Sersic r <= 0
    params[4, 11] = np.nan      # non-finite
    params[5, 11] = 25.0        # Sersic n > 20
    h = prob.create()
    try:
        logl_g, model_g = _gpu_eval(L, h, params, cfg.H, cfg.W)
    finally:
        L.lensed_destroy(h)
    logl_o, model_o = prob.oracle_loglike(params)
    bad = np.array([False, True, True, False, True, True])
    assert np.array_equal(np.isneginf(logl_g), bad) and np.array_equal(np.isneginf(logl_o), bad)
    assert np.all(np.isnan(model_g[bad])) and np.all(np.isfinite(model_g[~bad]))
    assert logl_errors(logl_g[~bad], logl_o[~bad]).max() <= LOGL_RTOL


def test_parameter_domain_bound_by_bound_against_hand_written_expectations(L):
    """The table of tests/cases.py (every kind, every bound of the domain, NaN / inf in every slot;
    expectations written by hand, pinned on the oracle in test_oracle_pins.py) through the library:
    inside -> finite logL and image, outside -> -inf and NaN."""
    import torch
    from tests.cases import domain_cases
    H, W, s = 10, 12, 0.05
    quad = synth.get_config(0).quad
    d, w = np.zeros((H, W), dtype=np.float32), np.ones((H, W), dtype=np.float32)
    by_list = {}
    for models, p, valid in domain_cases():
        by_list.setdefault(models, []).append((p, valid))
    for models, rows in by_list.items():
        params = np.stack([p for p, _ in rows])
        valid = np.array([v for _, v in rows])
        h = L.lensed_create(d, w, None, None, quad, synth.kind_ids(models), s, 0.0)
        try:
            logl, model = _gpu_eval(L, h, params, H, W)
        finally:
            L.lensed_destroy(h)
        assert np.array_equal(np.isneginf(logl), ~valid), (models, np.flatnonzero(np.isneginf(logl) == valid))
        assert np.all(np.isfinite(logl[valid])) and np.all(np.isfinite(model[valid]))
        assert np.all(np.isnan(model[~valid]))


def test_a_vector_that_overflows_fp32_gives_minus_infinity_not_nan(L):
    """A valid vector whose source flux overflows FP32 (magnitude -300): its pixels are +inf, and
    the convolution must not turn them into NaN through a structurally zero tap (the tracers clamp
    what they store, trace_block.cuh store_pixel): logL = -inf like any hopeless vector, the
    other vectors of the batch are untouched."""
    cfg = synth.shrunk(synth.get_config(1), 40, 36, 4)
    prob = Problem(cfg)
    params = cfg.batch(4)
    params[2, 10] = -300.0       # source magnitude
    h = prob.create()
    try:
        logl_g, model_g = _gpu_eval(L, h, params, cfg.H, cfg.W)
    finally:
        L.lensed_destroy(h)
    assert np.isneginf(logl_g[2]) and not np.any(np.isnan(model_g[2]))
    ok = np.array([True, True, False, True])
    logl_o = prob.oracle_loglike(params[ok], want_model=False)
    assert logl_errors(logl_g[ok], logl_o).max() <= LOGL_RTOL


def test_a_step_captured_into_a_cuda_graph_replays_bit_for_bit(L):
    """After one call at a batch size (scratch at its high-water mark, no allocation left in the
    path) lensed_loglike is a fixed sequence of kernel launches and memsets on the caller's stream:
    it can be captured into a CUDA graph -- what a sampler does with its inner loop -- and the
    replay writes the same bits; new parameter values in the same buffer are picked up."""
    import torch
    cfg = synth.shrunk(synth.get_config(2), 64, 56, 4)
    prob = Problem(cfg)
    params = cfg.batch(40)
    h = prob.create()
    try:
        p = torch.from_numpy(params[:20]).cuda()
        direct = torch.empty(20, dtype=torch.float32, device="cuda")
        out = torch.empty_like(direct)
        L.lensed_loglike(h, p, direct)
        torch.cuda.synchronize()
        s = torch.cuda.Stream()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.stream(s):
            L.lensed_loglike(h, p, out, stream=s)
            s.synchronize()
            with torch.cuda.graph(g, stream=s):
                L.lensed_loglike(h, p, out, stream=torch.cuda.current_stream())
        out.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(out, direct)
        p.copy_(torch.from_numpy(params[20:]))               # the sampler's next batch, same buffers
        g.replay()
        torch.cuda.synchronize()
        L.lensed_loglike(h, p, direct)
        torch.cuda.synchronize()
        assert torch.equal(out, direct)
        assert logl_errors(out.cpu().numpy(), prob.oracle_loglike(params[20:], want_model=False)).max() <= LOGL_RTOL
    finally:
        L.lensed_destroy(h)


def test_fully_masked_image_and_zero_weights(L):
    cfg = synth.shrunk(synth.get_config(1), 30, 30, 3)
    prob = Problem(cfg)
    cfg.mask = np.zeros((30, 30), dtype=np.uint8)
    h = prob.create()
    try:
        assert L.lensed_num_traced(h) == 0
        logl_g, _ = _gpu_eval(L, h, cfg.batch(3), 30, 30, render=False)
    finally:
        L.lensed_destroy(h)
    assert np.array_equal(logl_g, np.zeros(3, dtype=np.float32))


def test_host_buffer_calls_match_device_calls_and_chunking_does_not_change_results(L):
    import torch
    cfg = synth.shrunk(synth.get_config(2), 80, 72, 40)
    prob = Problem(cfg)
    params = cfg.batch(40)
    h = prob.create()
    try:
        logl_dev, model_dev = _gpu_eval(L, h, params, cfg.H, cfg.W)
        logl_host = np.empty(40, dtype=np.float32)
        L.lensed_loglike_host(h, params, logl_host)
        pinned = torch.from_numpy(params).pin_memory()
        out_pinned = torch.empty(40, dtype=torch.float32).pin_memory()
        L.lensed_loglike_host(h, pinned, out_pinned)
        model_host = np.empty((40, cfg.H, cfg.W), dtype=np.float32)
        L.lensed_render_host(h, params, model_host)
        L.lensed_set_chunk_bytes(h, 3 * L.lensed_frame_bytes(h))  # 3 vectors per chunk, ragged last chunk
        logl_chunked, model_chunked = _gpu_eval(L, h, params, cfg.H, cfg.W)
        L.lensed_set_profiling(h, True)
        L.lensed_reset_profile(h)
        _gpu_eval(L, h, params, cfg.H, cfg.W, render=False)
        ms, n = L.lensed_get_profile(h)
    finally:
        L.lensed_destroy(h)
    assert np.array_equal(logl_dev, logl_host) and np.array_equal(logl_dev, out_pinned.numpy())
    assert np.array_equal(model_dev, model_host)
    assert np.array_equal(logl_dev, logl_chunked) and np.array_equal(model_dev, model_chunked)
    assert n == {"prep": 2, "trace": 14, "refine": 28, "conv": 14, "final": 1}       # prep = prep_kernel + order_kernel
    assert all(v > 0 for v in ms.values())


def test_clones_share_the_problem_and_run_concurrently_on_their_own_streams(L):
    """the problem data is immutable after create and usable from several streams:
    lensed_clone gives each stream its own scratch on the shared arrays.  Three handles, three
    streams, overlapping calls with different batches; then the original is destroyed first and
    the clones still work."""
    import torch
    cfg = synth.shrunk(synth.get_config(2), 80, 72, 8)
    prob = Problem(cfg)
    batches = [cfg.batch(200, stream=10 + i) for i in range(3)]
    h0 = prob.create()
    handles = [h0, L.lensed_clone(h0), L.lensed_clone(h0)]
    streams = [torch.cuda.Stream() for _ in handles]
    ps = [torch.from_numpy(b).cuda() for b in batches]
    outs = [torch.empty(200, dtype=torch.float32, device="cuda") for _ in handles]
    torch.cuda.synchronize()
    try:
        for rep in range(3):                                   # overlapping launches, repeated
            for h, st, p, o in zip(handles, streams, ps, outs):
                L.lensed_loglike(h, p, o, stream=st.cuda_stream)
        torch.cuda.synchronize()
        got = [o.cpu().numpy() for o in outs]
        L.lensed_destroy(handles[0])                           # the original goes first
        again = torch.empty(200, dtype=torch.float32, device="cuda")
        L.lensed_loglike(handles[2], ps[2], again)
        torch.cuda.synchronize()
        assert np.array_equal(again.cpu().numpy(), got[2])
    finally:
        for h in handles:
            L.lensed_destroy(h)
    for b, g in zip(batches, got):
        ref = prob.oracle_loglike(b[::8], want_model=False)
        assert logl_errors(g[::8], ref).max() <= LOGL_RTOL


def test_create_rejects_bad_arguments_on_the_gpu_box_too(L):
    cfg = synth.get_config(0)
    img = np.zeros((8, 8), np.float32)
    w = np.ones((8, 8), np.float32)
    kinds = synth.kind_ids(cfg.models)
    with pytest.raises(L.LensedError) as e:
        L.lensed_create(img, w, None, np.ones((4, 3), np.float32), cfg.quad, kinds, 0.05)
    assert e.value.status == L.EINVAL
    with pytest.raises(L.LensedError) as e:
        L.lensed_create(img, -w, None, None, cfg.quad, kinds, 0.05)
    assert e.value.status == L.EINVAL


# --------------------------------------------------- quadrature error estimate
@pytest.mark.parametrize("n_kronrod", [7, 11, 15])
def test_quadrature_error_map_of_the_gauss_kronrod_rule(L, n_kronrod):
    """lensed_render_error against the oracle's |K - G| with the paper's g3k7 (default), g5k11
    and g7k15 rules; the estimate is a small difference of two FP32 sums, so the bound is
    absolute: 3e-5 of the pixel's own luminosity (floored at 1e-3 of the image peak), the FP32
    noise of a pixel that holds the centre of a cuspy source.  With g3k7
    the map stands well above that floor; with the higher rules most of it lies below."""
    import torch
    from oracle import lensed_oracle as orc
    models = ("sie", "shear", "src_sersic", "fg_sersic", "sky")
    base = synth.shrunk(synth.get_config(1), 40, 44, 5)
    quad, emb = synth.gauss_kronrod_rule(n_kronrod), synth.gauss_kronrod_embedded_weights(n_kronrod)
    cfg = synth.Config(1, "gk", base.H, base.W, base.scale, models, quad, base.psf, None, base.truth, 5,
                       base._draw, 0.005, 2000.0)
    params = cfg.batch()
    params[4, 3] = 1.5                                   # q > 1: outside the domain -> NaN map
    h = Problem(cfg).create()
    try:
        p = torch.from_numpy(params).cuda()
        err = torch.empty((len(params), cfg.H, cfg.W), dtype=torch.float32, device="cuda")
        with pytest.raises(L.LensedError):
            L.lensed_render_error(h, p, err)             # no embedded rule yet
        L.lensed_set_error_rule(h, emb)
        L.lensed_render_error(h, p, err)
        logl = torch.empty(len(params), dtype=torch.float32, device="cuda")
        L.lensed_loglike(h, p, logl)                     # the likelihood path is untouched by the rule
        torch.cuda.synchronize()
        err = err.cpu().numpy()
    finally:
        L.lensed_destroy(h)
    kinds = synth.kind_ids(models)
    assert np.all(np.isnan(err[4])) and np.isneginf(logl[4].item())
    for b in range(4):
        ref = orc.error_map(cfg.H, cfg.W, cfg.scale, quad, emb, kinds, params[b], zp=cfg.zp)
        raw = orc.render_raw(cfg.H, cfg.W, cfg.scale, quad, kinds, params[b], zp=cfg.zp)
        bound = 3e-5 * np.maximum(raw, 1e-3 * raw.max())
        if n_kronrod == 7:
            assert ref.max() > 10 * bound.max()          # the map is well above the bound somewhere
        assert np.all(np.abs(err[b] - ref) <= bound), "error map off by %.3g of the bound" % (
            np.abs(err[b] - ref) / bound).max()


@pytest.mark.parametrize("index,H,W", [(2, 75, 93), (1, 72, 66), (3, 70, 80)])
def test_frame_cells_the_tracer_never_writes_reach_no_result(L, index, H, W):
    """Stand-in for an uninitialised-read checker (compute-sanitizer is closed on this pool).  The
    padded frames of the unconvolved images hold cells no kernel writes: pad cells no border pixel
    clamps to and, on a masked image, pixels outside the traced set.  The convolution reads some of
    them under structurally zero taps or for outputs it discards (conv.cu "Input").  Overwriting
    EVERY cell of the frames between two calls (lensed_debug_fill_frames, include/lensed_tune.h)
    must not change one bit of logL or of the rendered images, in any convolution shape."""
    cfg = synth.shrunk(synth.get_config(index), H, W, 5)
    prob = Problem(cfg)
    params = cfg.batch(5)
    h = prob.create()
    try:
        for shape in (3, 2, 1, 0):
            try:
                L.lensed_set_conv_shape(h, shape)
            except L.LensedError as e:
                assert e.status == L.EUNSUPPORTED
                continue
            ref = _gpu_eval(L, h, params, H, W)
            for value in (1e30, -7.5):
                L.lensed_debug_fill_frames(h, value)
                logl = _gpu_eval(L, h, params, H, W, render=False)[0]
                assert np.array_equal(logl, ref[0]), (shape, value)
                L.lensed_debug_fill_frames(h, value)
                model = _gpu_eval(L, h, params, H, W)[1]
                assert np.array_equal(model, ref[1]), (shape, value)
    finally:
        L.lensed_destroy(h)


def test_full_constant_tap_pool_falls_back_to_global_memory_taps(L):
    """The PSF taps of the live handles share 60 KB of constant memory (include/lensed.h).  Two
    63x63 PSFs (32.5 KB each) do not fit together: the second handle keeps its taps in global
    memory and must compute the same thing; so must the 9th .. 16th of sixteen live 31x31 handles
    (8 KB each) -- a sampler fitting several images or bands at once."""
    rng = np.random.default_rng(7)
    psf = rng.uniform(0.1, 1.0, size=(63, 63))
    small = synth.shrunk(synth.get_config(1), 20, 24, 2)
    cfg = synth.Config(1, "pool", small.H, small.W, small.scale, small.models, small.quad, psf, None,
                       small.truth, 2, small._draw, 0.005, 2000.0)
    prob = Problem(cfg)
    logl_o = prob.oracle_loglike(cfg.batch())[0]
    h1 = prob.create()
    h2 = prob.create()
    try:
        assert L.lensed_uses_global_taps(h1) == 0 and L.lensed_uses_global_taps(h2) == 1
        for h in (h1, h2):
            logl, _ = _gpu_eval(L, h, cfg.batch(), cfg.H, cfg.W, render=False)
            assert logl_errors(logl, logl_o).max() <= LOGL_RTOL
    finally:
        L.lensed_destroy(h1); L.lensed_destroy(h2)
    h3 = prob.create()                                    # room in the pool again
    try:
        assert L.lensed_uses_global_taps(h3) == 0
    finally:
        L.lensed_destroy(h3)

    cfg = synth.shrunk(synth.get_config(4), 70, 90, 3)    # 31 x 31 PSF
    prob = Problem(cfg)
    params = cfg.batch()
    logl_o, model_o = prob.oracle_loglike(params, want_model=True)
    handles = [prob.create() for _ in range(16)]
    try:
        flags = [L.lensed_uses_global_taps(h) for h in handles]
        assert flags[0] == 0 and flags[-1] == 1 and 7 <= flags.count(0) <= 8
        for h in (handles[0], handles[8], handles[15]):
            logl, model = _gpu_eval(L, h, params, cfg.H, cfg.W)
            assert logl_errors(logl, logl_o).max() <= LOGL_RTOL
            assert pixel_errors(model, model_o).max() <= PIXEL_RTOL
    finally:
        for h in handles:
            L.lensed_destroy(h)


@pytest.mark.parametrize("index,H,W,B", [(1, 90, 70, 12), (2, 75, 93, 8), (3, 70, 150, 6), (4, 101, 67, 4), (5, 60, 64, 6)])
@pytest.mark.parametrize("global_taps", [False, True])
def test_all_convolution_shapes_and_both_tap_paths(L, index, H, W, B, global_taps):
    """strip (8 independent warps per SM on 16 x 64 strips), wide (256 threads, 64 x 128 tiles) and
    narrow (128 threads, 64 x 64 tiles, two blocks per SM), taps from the constant pool or from
    global memory: same results against the oracle, and the rendered images of the three shapes
    agree bit for bit (same per-pixel arithmetic; only the chi-square partials are grouped
    differently)."""
    cfg = synth.shrunk(synth.get_config(index), H, W, B)
    prob = Problem(cfg)
    params = cfg.batch()
    logl_o, model_o = prob.oracle_loglike(params, want_model=True)
    L.lensed_debug_force_global_taps(global_taps)
    try:
        h = prob.create()
    finally:
        L.lensed_debug_force_global_taps(False)
    try:
        assert L.lensed_uses_global_taps(h) == int(global_taps)
        models = []
        for shape in (3, 2, 1, 0):
            L.lensed_set_conv_shape(h, shape)
            assert L.lensed_get_conv_shape(h) == shape
            logl, model = _gpu_eval(L, h, params, cfg.H, cfg.W)
            assert logl_errors(logl, logl_o).max() <= LOGL_RTOL
            assert pixel_errors(model, model_o).max() <= PIXEL_RTOL
            models.append(model)
        assert all(np.array_equal(models[0], m) for m in models[1:])
        with pytest.raises(L.LensedError) as e:
            L.lensed_set_conv_shape(h, 4)
        assert e.value.status == L.EINVAL
    finally:
        L.lensed_destroy(h)


def test_shape_picked_at_create_and_shared_memory_limits(L):
    """lensed_create: wide for a full image with a large PSF, half-width strips for the SLACS annulus
    (39 of them compute 20.0 k pixels, 23 full strips 23.6 k, 8 narrow tiles 32.8 k); a 63 x 63 PSF
    does not fit the strip shapes' eight stages."""
    for index, want in ((4, 1), (2, 3)):
        h = Problem(synth.get_config(index), image=np.zeros((synth.get_config(index).H, synth.get_config(index).W), np.float32),
                    weight=np.ones((synth.get_config(index).H, synth.get_config(index).W), np.float32)).create()
        try:
            assert L.lensed_get_conv_shape(h) == want
        finally:
            L.lensed_destroy(h)
    cfg = synth.shrunk(synth.get_config(1), 40, 36, 2)
    cfg.psf = synth.moffat_psf(63, 3.0, 2.5)
    h = Problem(cfg, image=np.zeros((40, 36), np.float32), weight=np.ones((40, 36), np.float32)).create()
    try:
        assert L.lensed_get_conv_shape(h) in (0, 1)
        for shape in (2, 3):
            with pytest.raises(L.LensedError) as e:
                L.lensed_set_conv_shape(h, shape)
            assert e.value.status == L.EUNSUPPORTED
    finally:
        L.lensed_destroy(h)


def _require_jit(L, h):
    """the handle's tracer must be the run-time specialised one.  A box without NVRTC FAILS here (the
    specialised tracer is the default path of every list without a built-in signature: it must not
    lose its coverage silently); the tests are skipped only where the run-time specialisation was
    switched off on purpose with LENSED_JIT=0 in the environment of the test run."""
    import os
    kind, why = L.lensed_get_static_tracer(h), L.lensed_last_error(h) or ""
    if kind != 2 and os.environ.get("LENSED_JIT", "")[:1] == "0":
        pytest.skip("run-time specialisation switched off: LENSED_JIT=0")
    assert kind == 2, "run-time specialisation unavailable on this box: " + why


def test_a_list_without_a_built_in_signature_gets_its_tracer_compiled_at_create(L):
    """SIE + shear + two Gaussian sources + Gaussian lens light + sky has none of the built-in
    signatures: lensed_create specialises the tracer for it with NVRTC (csrc/jit.cu; the paper
    compiles its kernel at run time too).  Same results as the oracle and as the
    interpreting tracer within the tolerances; LENSED_JIT=0 keeps the interpreter."""
    import os
    models = ("sie", "shear", "src_gauss", "src_gauss", "fg_gauss", "sky")
    truth = [0.02, -0.03, 0.5, 0.7, 35.0, 0.03, -0.02,
             0.05, 0.08, 0.06, synth.mag_of_flux(30.0), 0.8, 20.0,
             -0.1, 0.02, 0.04, synth.mag_of_flux(10.0), 0.6, 100.0,
             0.0, 0.01, 0.3, synth.mag_of_flux(400.0), 0.7, 60.0,
             0.01]
    cfg = _mini(models, truth, H=45, W=52, psf=synth.gaussian_psf(7, 2.0), quad=synth.gauss_legendre_rule(3))
    prob = Problem(cfg)
    rng = np.random.default_rng(5)
    params = np.vstack([cfg.truth] * 6).astype(np.float32)
    params[1:] *= (1.0 + 0.05 * rng.standard_normal(params[1:].shape)).astype(np.float32)
    params[:, 3] = np.clip(params[:, 3], 0.3, 1.0)
    params[:, [11, 17, 23]] = np.clip(params[:, [11, 17, 23]], 0.2, 1.0)
    logl_o, model_o = prob.oracle_loglike(params, want_model=True)
    h = prob.create()
    try:
        _require_jit(L, h)
        logl_j, model_j = _gpu_eval(L, h, params, cfg.H, cfg.W)
        L.lensed_set_static_tracer(h, 0)
        assert L.lensed_get_static_tracer(h) == 0
        logl_i, model_i = _gpu_eval(L, h, params, cfg.H, cfg.W)
        L.lensed_set_static_tracer(h, 1)
        assert L.lensed_get_static_tracer(h) == 2
    finally:
        L.lensed_destroy(h)
    for logl, model in ((logl_j, model_j), (logl_i, model_i)):
        assert logl_errors(logl, logl_o).max() <= LOGL_RTOL
        assert pixel_errors(model, model_o).max() <= PIXEL_RTOL
    os.environ["LENSED_JIT"] = "0"
    try:
        h = prob.create()
        try:
            assert L.lensed_get_static_tracer(h) == 0
            with pytest.raises(L.LensedError):
                L.lensed_set_static_tracer(h, 1)
        finally:
            L.lensed_destroy(h)
    finally:
        del os.environ["LENSED_JIT"]


_PARS = {"sis": lambda r: [r.uniform(-.1, .1), r.uniform(-.1, .1), r.uniform(.2, .5)],
         "sie": lambda r: [r.uniform(-.1, .1), r.uniform(-.1, .1), r.uniform(.3, .6), r.uniform(.25, 1.), r.uniform(0, 180)],
         "point": lambda r: [r.uniform(-.3, .3), r.uniform(-.3, .3), r.uniform(.02, .08)],
         "shear": lambda r: [r.uniform(-.05, .05), r.uniform(-.05, .05)],
         "src_sersic": lambda r: [r.uniform(-.1, .1), r.uniform(-.1, .1), r.uniform(.05, .2), synth.mag_of_flux(r.uniform(10, 40)),
                                  r.uniform(.5, 4.), r.uniform(.4, 1.), r.uniform(0, 180)],
         "fg_sersic": lambda r: [r.uniform(-.1, .1), r.uniform(-.1, .1), r.uniform(.2, .5), synth.mag_of_flux(r.uniform(200, 800)),
                                 r.uniform(1., 4.), r.uniform(.5, 1.), r.uniform(0, 180)],
         "src_gauss": lambda r: [r.uniform(-.1, .1), r.uniform(-.1, .1), r.uniform(.04, .1), synth.mag_of_flux(r.uniform(10, 40)),
                                 r.uniform(.4, 1.), r.uniform(0, 180)],
         "fg_gauss": lambda r: [r.uniform(-.1, .1), r.uniform(-.1, .1), r.uniform(.2, .4), synth.mag_of_flux(r.uniform(100, 300)),
                                r.uniform(.5, 1.), r.uniform(0, 180)],
         "sky": lambda r: [r.uniform(0, .02)]}


@pytest.mark.parametrize("seed,models,n_rule", [
    (1, ("fg_sersic", "fg_gauss", "sky"), 2),                                  # no lens, no source: foreground only
    (2, ("sis", "point", "src_sersic", "src_gauss"), 3),                       # circular lenses only, two kinds of source
    (3, ("sie", "sis", "shear", "src_sersic", "fg_gauss", "sky"), 2),          # one SIE but not "direct" (a SIS beside it)
    (4, ("sie", "sie", "sie", "src_gauss", "sky"), 3),                         # three SIEs, their modes mixed
    (5, ("point", "shear", "src_gauss", "src_gauss", "src_gauss", "fg_sersic", "fg_sersic"), 5),
    (6, ("sie", "src_sersic", "src_sersic", "src_sersic", "fg_sersic", "fg_gauss", "fg_gauss", "sky", "sky"), 4),
    (7, ("shear", "src_gauss"), 7),                                            # 49-point rule: 5 points per pass, one dummy
])
def test_run_time_specialised_tracers_of_assorted_lists_against_the_oracle(L, seed, models, n_rule):
    """The specialised tracer is one template over the per-kind counts; the built-in signatures
    exercise nine points of that space.  Here NVRTC instantiates it for lists that take its other
    paths (no lens / no source / several SIEs / SIE + SIS without direct frames / foreground
    Gaussians first / 4-, 9-, 16-, 25- and 49-point rules) and each is compared with the oracle and
    with the interpreting tracer on drawn vectors, masked image, odd number of traced pixels."""
    rng = np.random.default_rng(100 + seed)
    draw = lambda: np.concatenate([_PARS[m](rng) for m in models])
    truth = draw()
    H, W = 33, 29
    mask = synth.annulus_mask(H, W, 2.0, 13.5)
    cfg = _mini(models, list(truth), H=H, W=W, psf=synth.gaussian_psf(5, 1.8), mask=mask, quad=synth.gauss_legendre_rule(n_rule))
    prob = Problem(cfg)
    params = np.vstack([truth] + [draw() for _ in range(5)]).astype(np.float32)
    logl_o, model_o = prob.oracle_loglike(params, want_model=True)
    h = prob.create()
    try:
        _require_jit(L, h)
        got = [_gpu_eval(L, h, params, H, W)]
        L.lensed_set_static_tracer(h, 0)
        got.append(_gpu_eval(L, h, params, H, W))
    finally:
        L.lensed_destroy(h)
    for logl, model in got:
        assert logl_errors(logl, logl_o).max() <= LOGL_RTOL
        assert pixel_errors(model, model_o).max() <= PIXEL_RTOL


@pytest.mark.parametrize("n_kronrod", [11, 15])
@pytest.mark.parametrize("which", ["hst", "mock", "jit"])
def test_the_papers_large_rules_through_the_specialised_tracers(L, which, n_kronrod):
    """g5k11 (121 points) and g7k15 (225 points), through the pixel-pair tracers:
    the HST list (built-in signature b), the paper's mock list (signature e) and a list specialised
    at run time, lensed_loglike AND lensed_render against the oracle, on a masked image with an odd
    number of traced pixels (a ragged last pixel pair)."""
    quad = synth.gauss_kronrod_rule(n_kronrod)
    assert len(quad) == n_kronrod ** 2
    H, W = 37, 41
    if which == "jit":
        models = ("sie", "shear", "src_gauss", "src_gauss", "fg_gauss", "sky")
        truth = np.array([0.02, -0.03, 0.5, 0.7, 35.0, 0.03, -0.02,
                          0.05, 0.08, 0.06, synth.mag_of_flux(30.0), 0.8, 20.0,
                          -0.1, 0.02, 0.04, synth.mag_of_flux(10.0), 0.6, 100.0,
                          0.0, 0.01, 0.3, synth.mag_of_flux(400.0), 0.7, 60.0,
                          0.01])
        rng = np.random.default_rng(50 + n_kronrod)

        def draw(_, B):
            out = np.tile(truth, (B, 1)) * (1.0 + 0.05 * rng.standard_normal((B, truth.size)))
            out[:, 3] = np.clip(out[:, 3], 0.3, 1.0)
            out[:, [11, 17, 23]] = np.clip(out[:, [11, 17, 23]], 0.2, 1.0)
            return out
        base = synth.Config(9, "jit", H, W, 0.05, models, quad, synth.gaussian_psf(7, 2.0), None, truth, 4, draw, 0.01, 0.0)
    else:
        base = synth.shrunk(synth.get_config(1 if which == "hst" else 5), H, W, 4)
    mask = synth.annulus_mask(H, W, 2.5, 15.3)
    cfg = synth.Config(base.index, base.name, H, W, base.scale, base.models, quad, base.psf, mask, base.truth, 4,
                       base._draw, base.sigma_sky, base.gain, base.zp)
    prob = Problem(cfg)
    params = np.vstack([cfg.batch(), cfg.truth.astype(np.float32)[None]])
    h = prob.create()
    try:
        if which == "jit":
            _require_jit(L, h)
        else:
            assert L.lensed_get_static_tracer(h) == 1
        if L.lensed_num_traced(h) % 2 == 0:                    # make the traced count odd: unmask one far pixel
            L.lensed_destroy(h)
            mask[0, 0] = 1
            h = prob.create()
        assert L.lensed_num_traced(h) % 2 == 1
        logl_g, model_g = _gpu_eval(L, h, params, H, W)
    finally:
        L.lensed_destroy(h)
    logl_o, model_o = prob.oracle_loglike(params, want_model=True)
    assert np.all(np.isfinite(logl_g))
    el, ep = logl_errors(logl_g, logl_o), pixel_errors(model_g, model_o)
    assert el.max() <= LOGL_RTOL, "logL rel err %.3g at vector %d" % (el.max(), el.argmax())
    assert ep.max() <= PIXEL_RTOL, "pixel rel err %.3g at vector %d" % (ep.max(), ep.argmax())


def test_issue_probe_measures_the_fp32_pipe_at_its_full_rate(L):
    """lensed_issue_probe (csrc/peak.cu), the micro-benchmark behind profiles/r2b.md: 64 packed FFMA2
    per body take 128 cycles (2 each), extra ALU-pipe instructions cost less than a cycle each,
    integer multiply-adds about two; bad arguments are EINVAL."""
    import os
    base = L.lensed_issue_probe(0, 0, 0, 2)
    assert np.isfinite(base) and base > 0.0
    if os.environ.get("LENSED_TIMING_TESTS") == "1":      # cycle counts: a quiet, full-clock box only (not the default run)
        assert 126.0 <= base <= 136.0
        assert base <= L.lensed_issue_probe(0, 1, 16, 2) <= base + 16.0
        assert L.lensed_issue_probe(0, 4, 32, 2) >= base + 40.0
    with pytest.raises(L.LensedError) as e:
        L.lensed_issue_probe(0, 1, 5, 2)
    assert e.value.status == L.EINVAL


def test_largest_rule_and_longest_model_list(L):
    """LENSED_MAX_QUAD-class rule (15 x 15 = 225 points, the size of the paper's g7k15) and a list
    of LENSED_MAX_MODELS = 32 objects (interpreting tracer, every kind present)."""
    rng = np.random.default_rng(11)
    models, truth = [], []
    for i in range(6):
        models.append("sis"); truth += [rng.uniform(-0.3, 0.3), rng.uniform(-0.3, 0.3), rng.uniform(0.02, 0.08)]
    for i in range(3):
        models.append("sie"); truth += [rng.uniform(-0.2, 0.2), rng.uniform(-0.2, 0.2), rng.uniform(0.05, 0.15),
                                        rng.uniform(0.3, 1.0), rng.uniform(0, 180)]
    for i in range(3):
        models.append("point"); truth += [rng.uniform(-0.3, 0.3), rng.uniform(-0.3, 0.3), rng.uniform(0.01, 0.04)]
    models += ["shear", "shear"]; truth += [0.03, -0.02, -0.01, 0.04]
    for i in range(6):
        models.append("src_gauss"); truth += [rng.uniform(-0.2, 0.2), rng.uniform(-0.2, 0.2), rng.uniform(0.03, 0.1),
                                              synth.mag_of_flux(rng.uniform(5, 20)), rng.uniform(0.4, 1.0), rng.uniform(0, 180)]
    for i in range(5):
        models.append("src_sersic"); truth += [rng.uniform(-0.2, 0.2), rng.uniform(-0.2, 0.2), rng.uniform(0.05, 0.15),
                                               synth.mag_of_flux(rng.uniform(5, 20)), rng.uniform(0.5, 4.0),
                                               rng.uniform(0.4, 1.0), rng.uniform(0, 180)]
    for i in range(3):
        models.append("fg_sersic"); truth += [rng.uniform(-0.2, 0.2), rng.uniform(-0.2, 0.2), rng.uniform(0.2, 0.6),
                                              synth.mag_of_flux(rng.uniform(50, 200)), rng.uniform(1.0, 4.0),
                                              rng.uniform(0.5, 1.0), rng.uniform(0, 180)]
    models += ["fg_gauss", "fg_gauss"]
    for i in range(2):
        truth += [rng.uniform(-0.2, 0.2), rng.uniform(-0.2, 0.2), rng.uniform(0.1, 0.3),
                  synth.mag_of_flux(rng.uniform(20, 50)), rng.uniform(0.5, 1.0), rng.uniform(0, 180)]
    models += ["sky", "sky"]; truth += [0.01, 0.005]
    assert len(models) == 32
    cfg = _mini(tuple(models), truth, H=20, W=22, psf=synth.gaussian_psf(5, 1.6), quad=synth.gauss_legendre_rule(15))
    assert len(cfg.quad) == 225
    prob = Problem(cfg)
    h = prob.create()
    try:
        assert L.lensed_get_static_tracer(h) == 0
    finally:
        L.lensed_destroy(h)
    _check(L, prob, np.vstack([cfg.truth.astype(np.float32)[None]] * 2))


@pytest.mark.parametrize("static", [True, False])
@pytest.mark.parametrize("index,H,W", [(1, 48, 40), (2, 64, 56), (3, 56, 48), (4, 60, 52), (5, 60, 64), (6, 56, 60)])
def test_every_one_of_192_draws_of_the_prior_meets_the_tolerances(L, index, H, W, static):
    """192 draws per prior -- BASELINE.json's four and the paper's own mock prior (n <= 8,
    q_S >= 0.1) -- on shrunk images, both tracers: EVERY vector inside north_star's
    bounds.  In plain FP32 about one draw in a hundred misses 1e-5 on logL (a source cusp on a
    pixel: DESIGN.md section 6); the FP64 refinement of the flagged pixels (refine.cu) closes
    that tail, and switching it off brings it back (test_refinement_switch below)."""
    import os
    cfg = synth.shrunk(synth.get_config(index), H, W, 4)
    params = cfg.batch(int(os.environ.get("LENSED_ENVELOPE_DRAWS", "192")))     # more draws: DESIGN.md section 6
    prob = Problem(cfg)
    h = prob.create()
    try:
        if not static:
            L.lensed_set_static_tracer(h, 0)
        logl_g, model_g = _gpu_eval(L, h, params, cfg.H, cfg.W)
    finally:
        L.lensed_destroy(h)
    logl_o, model_o = prob.oracle_loglike(params, want_model=True)
    el, ep = logl_errors(logl_g, logl_o), pixel_errors(model_g, model_o)
    assert np.median(el) <= 0.1 * LOGL_RTOL and el.max() <= LOGL_RTOL, "logL rel err %.3g at %d" % (el.max(), el.argmax())
    assert ep.max() <= PIXEL_RTOL, "pixel rel err %.3g at %d" % (ep.max(), ep.argmax())


def test_refinement_switch(L):
    """lensed_set_refine: with the default gain a few pixels per vector are re-traced in FP64 and
    the paper's mock prior meets the tolerances; with gain 0 nothing is refined and the known FP32
    tail is back (if this second half ever passes the tolerances, the refinement is dead weight);
    a larger gain refines fewer pixels; results are bitwise reproducible either way."""
    import torch
    cfg = synth.shrunk(synth.get_config(5), 60, 64, 4)
    params = cfg.batch(192)
    prob = Problem(cfg)
    logl_o = prob.oracle_loglike(params, want_model=False)
    p = torch.from_numpy(params).cuda()
    out = {}
    h = prob.create()
    try:
        for gain in (1.0, 4.0, 0.0):
            L.lensed_set_refine(h, gain)
            L.lensed_reset_profile(h)
            a = torch.empty(len(params), dtype=torch.float32, device="cuda")
            b = torch.empty_like(a)
            L.lensed_loglike(h, p, a)
            n = L.lensed_get_refined(h)
            L.lensed_loglike(h, p, b)
            assert torch.equal(a, b)
            assert L.lensed_get_refined(h) == 2 * n
            out[gain] = (logl_errors(a.cpu().numpy(), logl_o), n)
    finally:
        L.lensed_destroy(h)
    assert out[1.0][0].max() <= LOGL_RTOL and 192 <= out[1.0][1] <= 192 * 40
    assert 0 < out[4.0][1] < out[1.0][1]
    assert out[0.0][1] == 0 and out[0.0][0].max() > 3 * LOGL_RTOL


def test_a_compact_source_just_above_n_1_does_not_have_every_pixel_refined(L):
    """prep.cu's refinement threshold T2 = (G n sqrt(q) r_S / b_n)^(-2n/(n-1)) runs away as n -> 1+:
    for a source with r_S of a fraction of a pixel it used to hit its clamp and flag EVERY traced
    pixel of the vector for the FP64 re-trace.  It is now capped at the radius where the profile is
    exp(-24) of its centre: the refined pixels stay a small part of the image, and the results
    still meet the tolerances."""
    import torch
    cfg = synth.shrunk(synth.get_config(1), 72, 66, 4)
    assert cfg.models[2] == "src_sersic"
    params = np.repeat(cfg.truth.astype(np.float32)[None], 6, axis=0)
    o = 7                                                      # sie (5) + shear (2): x y r mag n q pa
    params[:, o + 2] = cfg.scale * np.array([0.25, 0.2, 0.15, 0.1, 0.25, 0.12], dtype=np.float32)   # r_S in pixels
    params[:, o + 4] = np.array([1.02, 1.05, 1.08, 1.1, 1.001, 1.05], dtype=np.float32)
    prob = Problem(cfg)
    logl_o, model_o = prob.oracle_loglike(params, want_model=True)
    h = prob.create()
    try:
        L.lensed_reset_profile(h)
        logl_g, model_g = _gpu_eval(L, h, params, cfg.H, cfg.W, render=False)
        refined = L.lensed_get_refined(h)
        traced = L.lensed_num_traced(h)
        p = torch.from_numpy(params).cuda()
        model = torch.empty((len(params), cfg.H, cfg.W), dtype=torch.float32, device="cuda")
        L.lensed_render(h, p, model)
        torch.cuda.synchronize()
    finally:
        L.lensed_destroy(h)
    assert 0 < refined <= 0.25 * traced * len(params), (refined, traced)
    assert logl_errors(logl_g, logl_o).max() <= LOGL_RTOL
    assert pixel_errors(model.cpu().numpy(), model_o).max() <= PIXEL_RTOL


@pytest.mark.parametrize("rule", ["sub4", "gl3", "g3k7", "lopsided"])
def test_foreground_expansion_reproduces_the_rule_sum(L, rule):
    """The specialised tracers take a foreground Sersic's pixel integral from its fourth-order
    moment expansion where tau <= 0.15 (trace_static.cuh "foreground expansion").  Unlensed
    foreground components over their whole parameter range -- n from 0.3 (steeper than a Gaussian
    outside, range bounded ABOVE) to 8, axis ratios to 0.2, radii from 1.5 pixels up -- against the
    oracle with the expansion on (default), off, and at the loosest setting the API takes; the
    lopsided rule has odd moments, so the library must not use the expansion at all."""
    import torch
    quad = {"sub4": synth.subsample_rule(4), "gl3": synth.gauss_legendre_rule(3), "g3k7": synth.gauss_kronrod_rule(7),
            "lopsided": np.array([[0.3, 0.1, 0.5], [-0.2, 0.25, 0.2], [-0.1, -0.3, 0.3]])}[rule]
    models = ("sie", "src_sersic", "fg_sersic", "sky")
    rng = np.random.default_rng(21)
    rows = []
    for n in (0.3, 0.5, 0.8, 1.0, 1.5, 2.5, 4.0, 6.0, 8.0):
        for _ in range(3):
            rows.append([0.0, 0.0, 0.3, 0.8, 20.0, 0.2, 0.1, 0.1, synth.mag_of_flux(20.0), 1.5, 0.7, 30.0,
                         rng.uniform(-0.3, 0.3), rng.uniform(-0.3, 0.3), np.exp(rng.uniform(np.log(0.075), np.log(1.5))),
                         synth.mag_of_flux(2000.0), n, rng.uniform(0.2, 1.0), rng.uniform(0, 180), 0.01])
    params = np.array(rows, dtype=np.float32)
    cfg = _mini(models, rows[0], H=60, W=56, psf=synth.gaussian_psf(5, 1.7), quad=quad)
    prob = Problem(cfg)
    logl_o, model_o = prob.oracle_loglike(params, want_model=True)
    h = prob.create()
    try:
        assert L.lensed_get_static_tracer(h) == 1
        out = {}
        for tau in (0.15, 0.0, 0.5):
            L.lensed_set_fg_expansion(h, tau)
            logl, model = _gpu_eval(L, h, params, cfg.H, cfg.W)
            out[tau] = (logl, model)
            if tau < 0.5:
                assert logl_errors(logl, logl_o).max() <= LOGL_RTOL
                assert pixel_errors(model, model_o).max() <= PIXEL_RTOL
        with pytest.raises(L.LensedError):
            L.lensed_set_fg_expansion(h, 0.7)
    finally:
        L.lensed_destroy(h)
    d = np.abs(out[0.15][1] - out[0.0][1]).max() / np.abs(model_o).max()
    if rule == "lopsided":
        assert np.array_equal(out[0.15][1], out[0.0][1]) and np.array_equal(out[0.5][1], out[0.0][1])
    else:
        assert 0 < d < 3e-6                                  # used, and as accurate as derived
        assert pixel_errors(out[0.5][1], model_o).max() < 20 * PIXEL_RTOL   # tau = 0.5: 0.016 tau^6 = 2.5e-4


@pytest.mark.parametrize("static", [True, False])
def test_two_sies_in_different_modes_one_flat_one_round(L, static):
    """The SIE mode is per vector (the most general one any of its SIEs needs).  A flat SIE
    (q = 0.3: log-form atanh) beside a round one (q = 1, 0.9999, 0.97: A = b sqrt(q)/q' is huge)
    must not push the round one through the log form (its absolute error times A); realistic
    Einstein radii, the multi-lens list of config 3 in both tracers."""
    cfg = synth.shrunk(synth.get_config(3), 64, 72, 4)
    assert cfg.models[:2] == ("sie", "sie")
    rows = []
    for q1, q2 in ((0.3, 1.0), (0.3, 0.9999), (0.45, 0.97), (1.0, 0.3), (0.99999, 0.2), (0.3, 0.35)):
        p = cfg.truth.astype(np.float32).copy()
        p[3], p[8] = q1, q2
        p[7] = 0.9                                     # second Einstein radius 0.9": 18 pixels
        rows.append(p)
    _check(L, Problem(cfg), np.array(rows), static=static)


@pytest.mark.parametrize("static", [True, False])
@pytest.mark.parametrize("models", [("sie", "src_sersic"), ("sie", "shear", "src_sersic", "sky"),
                                    ("sis", "src_sersic", "sky", "sky")])
def test_static_signatures_outside_the_configs(L, models, static):
    """trace_sig_[f-h].cu: common lists that are not BASELINE.json configs; sky components do not
    enter the signature.  Both tracers against the oracle, SIE axis ratios across the modes."""
    rng = np.random.default_rng(5)
    rows = []
    for q in (0.97, 0.85, 0.72, 0.6, 0.52, 0.3):
        p = []
        for m in models:
            if m == "sie":
                p += [0.02, -0.03, 0.45, q, rng.uniform(0, 180)]
            elif m == "sis":
                p += [0.02, -0.03, 0.45]
            elif m == "shear":
                p += [0.04, -0.03]
            elif m == "src_sersic":
                p += [rng.uniform(-0.1, 0.1), rng.uniform(-0.1, 0.1), 0.1, synth.mag_of_flux(20.0), rng.uniform(0.7, 3.0),
                      0.7, rng.uniform(0, 180)]
            else:
                p += [0.01]
        rows.append(p)
    params = np.array(rows, dtype=np.float32)
    cfg = _mini(models, rows[2], H=40, W=36, psf=synth.gaussian_psf(5, 1.7), quad=synth.subsample_rule(4))
    _check(L, Problem(cfg), params, static=static)
