"""Image-plane priors and create-time variance estimation (PAPER.md:190-212
eqs. 18-21) through the C ABI on a B200, against the CPU oracle."""
import numpy as np
import pytest

from oracle import lensed_oracle as orc
from paper_1505_07674_b200 import synth
from tests.cases import LOGL_RTOL, Problem, logl_errors

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def L():
    import torch
    assert torch.cuda.is_available()
    from paper_1505_07674_b200 import lensed
    lensed.lib()
    return lensed


def _all_lens_problem():
    """every lens kind in one list, lights in between (they must be skipped)"""
    models = ("sie", "src_sersic", "shear", "sis", "sky", "point", "sie", "src_gauss")
    truth = [0.02, -0.03, 1.2, 0.75, 35.0,
             0.1, 0.2, 0.15, synth.mag_of_flux(20.0), 2.0, 0.5, 10.0,
             0.03, -0.05,
             -0.4, 0.3, 0.3,
             0.01,
             0.8, 0.6, 0.1,
             1.1, -0.7, 0.4, 0.9, 110.0,
             -0.2, 0.1, 0.08, synth.mag_of_flux(5.0), 0.7, 50.0]
    cfg = synth.Config(9, "lenses", 40, 44, 0.05, models, synth.gauss_legendre_rule(2), None, None, truth, 1,
                       lambda rng, B: np.tile(np.array(truth), (B, 1)), 0.01, 0.0)
    return cfg


def test_deflect_matches_the_oracle_over_all_lens_kinds_and_axis_ratios(L):
    import torch
    cfg = _all_lens_problem()
    prob = Problem(cfg)
    rng = np.random.default_rng(3)
    qs = [1.0, 0.99999, 0.999, 0.93, 0.82, 0.72, 0.6, 0.52, 0.45, 0.3, 0.1, 0.03]
    params = np.tile(cfg.truth.astype(np.float32), (len(qs), 1))
    params[:, 3] = qs
    params[:, 24] = qs[::-1]
    params[:, 2] *= rng.uniform(0.8, 1.2, size=len(qs)).astype(np.float32)
    K = 37
    xy = rng.uniform(-2.0, 2.0, size=(len(qs), K, 2)).astype(np.float32)
    xy[0, 0] = params[0, 0:2]                       # exactly on the first SIE's centre
    xy[1, 1] = params[1, 14:16]                     # on the SIS centre
    xy[2, 2] = params[2, 18:20]                     # on the point mass
    h = prob.create()
    try:
        out = torch.empty((len(qs), K, 2), dtype=torch.float32, device="cuda")
        L.lensed_deflect(h, torch.from_numpy(params).cuda(), torch.from_numpy(xy).cuda(), out)
        torch.cuda.synchronize()
        out = out.cpu().numpy()
    finally:
        L.lensed_destroy(h)
    for b in range(len(qs)):
        ref = orc.source_position(prob.kinds, params[b].astype(np.float64), xy[b].astype(np.float64))
        err_px = np.abs(out[b] - ref).max() / cfg.scale
        assert err_px <= 1e-5, "vector %d (q = %g, %g): %.3g px" % (b, params[b, 3], params[b, 24], err_px)


def test_deflect_gives_nan_for_vectors_with_a_lens_outside_its_domain(L):
    import torch
    cfg = _all_lens_problem()
    params = np.tile(cfg.truth.astype(np.float32), (4, 1))
    params[1, 3] = 1.5            # SIE q > 1
    params[2, 16] = -0.1          # SIS b < 0
    params[3, 9] = 99.0           # a LIGHT outside its domain does not matter here
    xy = np.random.default_rng(1).uniform(-1, 1, size=(4, 5, 2)).astype(np.float32)
    h = Problem(cfg).create()
    try:
        out = torch.empty((4, 5, 2), dtype=torch.float32, device="cuda")
        L.lensed_deflect(h, torch.from_numpy(params).cuda(), torch.from_numpy(xy).cuda(), out)
        out = out.cpu().numpy()
        with pytest.raises(L.LensedError):
            L.lensed_deflect(h, torch.from_numpy(params).cuda(), torch.from_numpy(xy[:3]).cuda(), torch.empty((3, 5, 2), device="cuda"))
    finally:
        L.lensed_destroy(h)
    assert np.all(np.isfinite(out[0])) and np.all(np.isnan(out[1])) and np.all(np.isnan(out[2])) and np.all(np.isfinite(out[3]))


def test_image_plane_prior_assigns_the_mapped_positions_in_place_and_the_likelihood_follows(L):
    """Draw image-plane positions for the two sources of the SLACS-like list, let the library map
    and assign them, and compare (a) the rewritten parameter columns with the oracle's map and
    (b) logL of the rewritten vectors with the oracle's logL of the oracle-mapped vectors."""
    import torch
    cfg = synth.shrunk(synth.get_config(2), 64, 60, 8)
    prob = Problem(cfg)
    params = cfg.batch(24)
    src = [i for i, m in enumerate(cfg.models) if m.startswith("src_")]
    offs = [sum(synth.NPAR[m] for m in cfg.models[:i]) for i in src]
    rng = np.random.default_rng(9)
    for o in offs:                                   # image-plane draws in a box around the ring
        params[:, o:o + 2] = rng.uniform(-1.4, 1.4, size=(len(params), 2))
    expect = params.astype(np.float64).copy()
    for b in range(len(params)):
        pts = np.array([expect[b, o:o + 2] for o in offs])
        mapped = orc.source_position(prob.kinds, params[b].astype(np.float64), pts)
        for o, xy in zip(offs, mapped):
            expect[b, o:o + 2] = xy
    h = prob.create()
    try:
        p = torch.from_numpy(params).cuda()
        L.lensed_image_plane_prior(h, p, src)
        logl = torch.empty(len(params), dtype=torch.float32, device="cuda")
        L.lensed_loglike(h, p, logl)
        torch.cuda.synchronize()
        got = p.cpu().numpy()
        for bad in ([0], [src[0], src[0]], [99]):    # a lens, a repeat, out of range
            with pytest.raises(L.LensedError) as e:
                L.lensed_image_plane_prior(h, p, bad)
            assert e.value.status == L.EINVAL
    finally:
        L.lensed_destroy(h)
    keep = np.ones(params.shape[1], dtype=bool)
    for o in offs:
        keep[o:o + 2] = False
    assert np.array_equal(got[:, keep], params[:, keep])                   # nothing else touched
    assert np.abs(got[:, ~keep] - expect[:, ~keep]).max() / cfg.scale <= 1e-5
    logl_o = prob.oracle_loglike(expect.astype(np.float32), want_model=False)
    assert logl_errors(logl.cpu().numpy(), logl_o).max() <= LOGL_RTOL


def test_estimated_weights_feed_create_and_loglike_like_the_oracle(L):
    """SURVEY 8(f).2 as a checked row: raw counts -> lensed_estimate_weights -> lensed_create ->
    lensed_loglike against the oracle doing the same from the same counts (eqs. 18-21, then 17),
    with gain / offset maps, the extra weight factor and pixels R15 masks."""
    import torch
    cfg = synth.shrunk(synth.get_config(1), 56, 50, 8)
    kinds = synth.kind_ids(cfg.models)
    rng = np.random.default_rng(150507674)
    truth = orc.render(cfg.H, cfg.W, cfg.scale, cfg.psf, cfg.quad, kinds, cfg.truth.astype(np.float32), zp=cfg.zp)[0]
    gain = rng.uniform(1500.0, 2500.0, size=truth.shape)
    sky = 0.02                                                   # subtracted background (offset b_i)
    counts = rng.poisson(gain * (truth + sky))
    data = (counts / gain - sky).astype(np.float32)
    data[3, 4] = -sky - 0.01                                     # non-positive counts: R15
    extra = rng.uniform(0.5, 1.0, size=truth.shape).astype(np.float32)
    gain32 = gain.astype(np.float32)
    w_lib = L.lensed_estimate_weights(data, gain32, sky, extra)
    w_orc = orc.estimate_weights(data, gain32, sky, extra)
    assert w_lib[3, 4] == 0.0 and w_orc[3, 4] == 0.0
    assert np.allclose(w_lib, w_orc, rtol=1e-6, atol=0)
    params = cfg.batch(16)
    h = L.lensed_create(data, w_lib, None, cfg.psf, cfg.quad, kinds, cfg.scale, cfg.zp, 0)
    try:
        logl = torch.empty(len(params), dtype=torch.float32, device="cuda")
        L.lensed_loglike(h, torch.from_numpy(params).cuda(), logl)
        torch.cuda.synchronize()
    finally:
        L.lensed_destroy(h)
    logl_o = orc.loglike(cfg.H, cfg.W, cfg.scale, data, w_orc, None, cfg.psf, cfg.quad, kinds, params, zp=cfg.zp)
    assert logl_errors(logl.cpu().numpy(), logl_o).max() <= LOGL_RTOL
    # chi-square per pixel of the truth is ~1 with these weights scaled back by the extra factor
    lt = orc.loglike(cfg.H, cfg.W, cfg.scale, data, w_orc / np.maximum(extra, 1e-30), None, cfg.psf, cfg.quad, kinds,
                     cfg.truth.astype(np.float32), zp=cfg.zp)[0]
    assert 0.9 < -2.0 * lt / truth.size < 1.1
