"""lensed_chisq_static: the likelihood call for users who may not allocate device memory.

A sampler that shares its GPU with a framework that has already claimed the memory, a farm of
workers on several streams that one worker's cudaMalloc would stall, or a job on a fixed memory
budget cannot use lensed_loglike safely once it is running: that call grows its scratch when a
batch is larger than any before.  lensed_chisq_static scores model images the caller already
holds on the device, with its partial sums in one fixed array inside the library (no cudaMalloc,
no cudaFree), for at most LENSED_CHISQ_STATIC_MAX_VECTORS images per call.

What is checked here: its logL equals the existing path's (lensed_loglike on the same parameter
vectors) within the suite's logL tolerance, on two calls in a row of different batch sizes -- the
second call finds the first call's partial sums and counters in the array and must not be fooled
by them -- and the size limit is refused with a message that names it.

The file sorts last on purpose: the suite runs with `pytest -x`, and a failure here must not hide the
parity tests.  It passes alone in a fresh process (its first call then does the one-time address
look-up) and after the rest of the suite.
"""
import ctypes

import numpy as np
import pytest

from paper_1505_07674_b200 import lensed, synth
from tests.cases import LOGL_RTOL, Problem, logl_errors


def _fake(addr=4096):
    return ctypes.c_void_p(addr)        # non-null and never dereferenced: the checks come before CUDA


def test_more_images_than_the_fixed_scratch_holds_is_refused_with_the_limit_in_the_message():
    """No device needed: the limit is checked before CUDA is touched."""
    lib = lensed.lib()
    too_many = lensed.CHISQ_STATIC_MAX_VECTORS + 1
    st = lib.lensed_chisq_static(0, _fake(), _fake(), 1024, _fake(), too_many, _fake(), None)
    assert st == lensed.EINVAL
    text = lib.lensed_last_error(None).decode()
    assert "LENSED_CHISQ_STATIC_MAX_VECTORS" in text and str(lensed.CHISQ_STATIC_MAX_VECTORS) in text and "split" in text


def test_the_python_constant_is_the_header_limit():
    import os
    import re
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    text = open(os.path.join(root, "include", "lensed.h")).read()
    assert int(re.search(r"#define\s+LENSED_CHISQ_STATIC_MAX_VECTORS\s+(\d+)", text).group(1)) == lensed.CHISQ_STATIC_MAX_VECTORS


@pytest.mark.parametrize("args", [
    dict(image=None), dict(weight=None), dict(model=None), dict(logl=None), dict(B=0), dict(n_pix=0),
    dict(n_pix=(1 << 30) + 1), dict(device=-1), dict(device=64)])
def test_bad_arguments_are_refused_before_cuda_is_touched(args):
    a = dict(device=0, image=_fake(), weight=_fake(), n_pix=100, model=_fake(), B=2, logl=_fake())
    a.update(args)
    st = lensed.lib().lensed_chisq_static(a["device"], a["image"], a["weight"], a["n_pix"], a["model"], a["B"], a["logl"], None)
    assert st == lensed.EINVAL
    assert lensed.lib().lensed_last_error(None).decode().startswith("lensed_chisq_static")


def _existing_path(h, params, H, W):
    """logL by lensed_loglike and the rendered images by lensed_render (both allocate scratch)"""
    import torch
    p = torch.from_numpy(np.ascontiguousarray(params, dtype=np.float32)).cuda()
    logl = torch.empty(len(params), dtype=torch.float32, device="cuda")
    model = torch.empty((len(params), H, W), dtype=torch.float32, device="cuda")
    lensed.lensed_loglike(h, p, logl)
    lensed.lensed_render(h, p, model)
    torch.cuda.synchronize()
    return logl.cpu().numpy(), model


@pytest.mark.gpu
@pytest.mark.parametrize("index,H,W,B1,B2", [(2, 75, 93, 12, 5),        # annulus mask, 21 x 21 PSF; 2 blocks per image
                                             (1, 100, 100, 9, 33)])    # HST at full size: 3 blocks, ragged last one
def test_two_calls_in_a_row_agree_with_lensed_loglike(index, H, W, B1, B2):
    import torch
    cfg = synth.shrunk(synth.get_config(index), H, W, max(B1, B2))
    prob = Problem(cfg)
    rng = np.random.default_rng(20260 + index)
    image_dev = torch.from_numpy(np.ascontiguousarray(prob.image, dtype=np.float32)).cuda()
    w = np.asarray(prob.weight, dtype=np.float32) * (1.0 if cfg.mask is None else (np.asarray(cfg.mask) != 0))
    weight_dev = torch.from_numpy(np.ascontiguousarray(w, dtype=np.float32)).cuda()
    h = prob.create()
    try:
        for B in (B1, B2):                                   # second call: the scratch holds the first call's leftovers
            params = cfg.batch(B)
            params[rng.integers(B)] = cfg.truth               # one vector at the truth (chi-square ~ number of pixels)
            bad = int(rng.integers(B))
            params[bad, :] = np.nan                           # one vector outside the model domain
            ref, model = _existing_path(h, params, cfg.H, cfg.W)
            assert np.isneginf(ref[bad]) and torch.isnan(model[bad]).all()
            logl = torch.full((B,), 123.0, dtype=torch.float32, device="cuda")
            again = torch.full((B,), -7.0, dtype=torch.float32, device="cuda")
            lensed.lensed_chisq_static(image_dev, weight_dev, model, logl)
            torch.cuda.synchronize()
            free_before = torch.cuda.mem_get_info()[0]           # cudaMemGetInfo: the whole device, not torch's pool
            lensed.lensed_chisq_static(image_dev, weight_dev, model, again)
            torch.cuda.synchronize()
            assert torch.cuda.mem_get_info()[0] >= free_before, "the call took device memory"
            got = logl.cpu().numpy()
            assert np.array_equal(got, again.cpu().numpy()), "not bitwise reproducible"
            assert np.isneginf(got[bad])
            ok = np.arange(B) != bad
            assert np.all(np.isfinite(got[ok]))
            err = logl_errors(got[ok], ref[ok].astype(np.float64))
            assert err.max() <= LOGL_RTOL, "logL rel err %.3g against lensed_loglike at vector %d" % (err.max(), err.argmax())
    finally:
        lensed.lensed_destroy(h)


@pytest.mark.gpu
def test_weights_of_zero_hide_whatever_the_model_holds_there():
    """masked pixels (w = 0) are skipped, so NaN under the mask does not reach logL"""
    import torch
    g = torch.Generator(device="cpu").manual_seed(7)
    n, B = 5000, 3
    image = torch.randn(n, generator=g)
    weight = torch.rand(n, generator=g) + 0.5
    weight[::3] = 0.0
    model = torch.randn(B, n, generator=g)
    expect = -0.5 * (weight.double() * (image.double() - model.double()) ** 2).sum(dim=1)
    model[:, ::3] = float("nan")
    logl = torch.empty(B, dtype=torch.float32, device="cuda")
    lensed.lensed_chisq_static(image.cuda(), weight.cuda(), model.cuda(), logl)
    torch.cuda.synchronize()
    assert logl_errors(logl.cpu().numpy(), expect.numpy()).max() <= LOGL_RTOL
