"""Thin binding of the C-ABI library (include/lensed.h): argument marshalling only.

Same names as the C entry points.  Every step of the path runs in the CUDA kernels of
`liblensed_b200.so`; torch is used for device memory and streams.  There is no CPU
fallback: if the library is missing it is built with nvcc, and if that fails, or there
is no CUDA device, the calls raise.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblensed_b200.so")

OK, EINVAL, ENOMEM, ECUDA, EUNSUPPORTED = 0, 1, 2, 3, 4
STATUS_NAMES = {0: "LENSED_OK", 1: "LENSED_EINVAL", 2: "LENSED_ENOMEM", 3: "LENSED_ECUDA",
                4: "LENSED_EUNSUPPORTED"}
# lensed_kind (include/lensed.h)
LENS_SIS, LENS_SIE, LENS_POINT, LENS_SHEAR = 0, 1, 2, 3
SRC_SERSIC, SRC_GAUSS, FG_SERSIC, FG_GAUSS, FG_SKY = 4, 5, 6, 7, 8
PHASES = ("prep", "trace", "refine", "conv", "final")

# every symbol include/lensed.h and include/lensed_tune.h declare: (restype, argtypes)
_c, _i, _d, _p, _ll = ctypes.c_char_p, ctypes.c_int, ctypes.c_double, ctypes.c_void_p, ctypes.c_longlong
SYMBOLS = {
    "lensed_create": (_i, [_i, _i, _d, _p, _p, _p, _p, _i, _i, _p, _i, _p, _i, _d, _i, _p]),
    "lensed_clone": (_i, [_p, _p]),
    "lensed_num_params": (_i, [_p]),
    "lensed_num_traced": (_i, [_p]),
    "lensed_num_pixels": (_i, [_p]),
    "lensed_render": (_i, [_p, _p, _i, _p, _p]),
    "lensed_loglike": (_i, [_p, _p, _i, _p, _p]),
    "lensed_render_host": (_i, [_p, _p, _i, _p, _p]),
    "lensed_deflect": (_i, [_p, _p, _i, _p, _i, _p, _p]),
    "lensed_image_plane_prior": (_i, [_p, _p, _i, _p, _i, _p]),
    "lensed_estimate_weights": (_i, [_ll, _p, _p, _d, _p, _d, _p, _p]),
    "lensed_set_error_rule": (_i, [_p, _p]),
    "lensed_render_error": (_i, [_p, _p, _i, _p, _p]),
    "lensed_loglike_host": (_i, [_p, _p, _i, _p, _p]),
    "lensed_set_profiling": (_i, [_p, _i]),
    "lensed_get_profile": (_i, [_p, _p, _p]),
    "lensed_reset_profile": (_i, [_p]),
    "lensed_set_refine": (_i, [_p, _d]),
    "lensed_set_fg_expansion": (_i, [_p, _d]),
    "lensed_get_refined": (_i, [_p, _p]),
    "lensed_debug_fill_frames": (_i, [_p, ctypes.c_float]),
    "lensed_set_chunk_bytes": (_i, [_p, _ll]),
    "lensed_frame_bytes": (_ll, [_p]),
    "lensed_set_conv_shape": (_i, [_p, _i]),
    "lensed_get_conv_shape": (_i, [_p]),
    "lensed_uses_global_taps": (_i, [_p]),
    "lensed_debug_force_global_taps": (None, [_i]),
    "lensed_set_static_tracer": (_i, [_p, _i]),
    "lensed_get_static_tracer": (_i, [_p]),
    "lensed_debug_jit_compile": (_i, [_p, _i, _i, ctypes.c_char_p, _i]),
    "lensed_ns_run": (_i, [_p, _p, _p, _p, _i, _p, _p, _p, _p, _p, _ll, _p]),
    "lensed_ns_philox": (None, [_p, _p, _p]),
    "lensed_fma_peak": (_i, [_i, _i, _p]),
    "lensed_issue_probe": (_i, [_i, _i, _i, _i, _p]),
    "lensed_chisq_static": (_i, [_i, _p, _p, _ll, _p, _i, _p, _p]),
    "lensed_last_error": (_c, [_p]),
    "lensed_destroy": (None, [_p]),
}


class LensedError(RuntimeError):
    def __init__(self, status, text):
        super().__init__("%s: %s" % (STATUS_NAMES.get(status, status), text))
        self.status = status


_lib = None


def lib():
    """The loaded shared library; built in-tree with nvcc if it is not there."""
    global _lib
    if _lib is None:
        path = os.environ.get("LENSED_B200_LIB") or LIB_PATH     # override: a differently tuned build
        if path == LIB_PATH and not os.path.exists(LIB_PATH):
            from . import build as _build
            _build.build()
        L = ctypes.CDLL(path)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def _np(a, dtype):
    return None if a is None else np.ascontiguousarray(a, dtype=dtype)


def _hp(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _check(status, handle=None):
    if status != OK:
        text = lib().lensed_last_error(handle)
        raise LensedError(status, text.decode() if text else "")


def _stream(stream):
    """None = torch's current stream; else a torch.cuda.Stream or a raw cudaStream_t value"""
    if stream is not None:
        return ctypes.c_void_p(int(getattr(stream, "cuda_stream", stream)))
    import torch
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def lensed_create(image, weight, mask, psf, quad, models, pixel_scale, mag_zero_point=0.0, device=0):
    """-> opaque handle (ctypes.c_void_p).  Arrays are host numpy arrays; see lensed.h."""
    image = _np(image, np.float32)
    H, W = image.shape
    weight = _np(weight, np.float32)
    mask = _np(mask, np.uint8)
    psf = _np(psf, np.float32)
    ph, pw = (0, 0) if psf is None else psf.shape
    quad = _np(quad, np.float32).reshape(-1, 3)
    models = _np(models, np.int32)
    if weight.shape != image.shape or (mask is not None and mask.shape != image.shape):
        raise LensedError(EINVAL, "weight / mask shape differs from the image")
    h = ctypes.c_void_p()
    st = lib().lensed_create(H, W, float(pixel_scale), _hp(image), _hp(weight), _hp(mask), _hp(psf),
                             ph, pw, _hp(quad), len(quad), _hp(models), len(models),
                             float(mag_zero_point), int(device), ctypes.byref(h))
    _check(st)
    return h


def lensed_clone(h):
    """-> a second handle on the same problem (shared immutable arrays, own scratch)."""
    out = ctypes.c_void_p()
    _check(lib().lensed_clone(h, ctypes.byref(out)))
    return out


def lensed_num_params(h):
    return lib().lensed_num_params(h)


def lensed_num_traced(h):
    return lib().lensed_num_traced(h)


def lensed_num_pixels(h):
    """H * W of the handle's image."""
    return lib().lensed_num_pixels(h)


def lensed_render(h, params_dev, model_dev, stream=None):
    """params_dev [B][P], model_dev [B][H][W]: contiguous float32 CUDA tensors."""
    B = _check_dev(h, params_dev)
    _check_out(model_dev, B, B * lensed_num_pixels(h))
    _check(lib().lensed_render(h, params_dev.data_ptr(), B, model_dev.data_ptr(), _stream(stream)), h)
    return model_dev


def lensed_estimate_weights(image, gain, offset=0.0, extra=None):
    """w = extra * gain / (image + offset) (eqs. 18-21); gain / offset: scalars or maps."""
    img = _np(image, np.float32)
    g = None if np.isscalar(gain) else _np(gain, np.float32)
    b = None if np.isscalar(offset) else _np(offset, np.float32)
    x = _np(extra, np.float32)
    out = np.empty(img.shape, dtype=np.float32)
    _check(lib().lensed_estimate_weights(img.size, _hp(img), _hp(g), float(gain) if g is None else 0.0,
                                         _hp(b), float(offset) if b is None else 0.0, _hp(x), _hp(out)))
    return out


def lensed_set_error_rule(h, w_embedded):
    """w_embedded [n_quad]: weights of the embedded lower-order rule (host array)."""
    w = _np(w_embedded, np.float32)
    _check(lib().lensed_set_error_rule(h, _hp(w)), h)


def lensed_render_error(h, params_dev, err_dev, stream=None):
    """params_dev [B][P], err_dev [B][H][W]: contiguous float32 CUDA tensors."""
    B = _check_dev(h, params_dev)
    _check_out(err_dev, B, B * lensed_num_pixels(h))
    _check(lib().lensed_render_error(h, params_dev.data_ptr(), B, err_dev.data_ptr(), _stream(stream)), h)
    return err_dev


def lensed_loglike(h, params_dev, logl_dev, stream=None):
    """params_dev [B][P], logl_dev [B]: contiguous float32 CUDA tensors."""
    B = _check_dev(h, params_dev)
    _check_out(logl_dev, B, B)
    _check(lib().lensed_loglike(h, params_dev.data_ptr(), B, logl_dev.data_ptr(), _stream(stream)), h)
    return logl_dev


def lensed_deflect(h, params_dev, xy_dev, out_dev, stream=None):
    """params_dev [B][P], xy_dev / out_dev [B][K][2]: contiguous float32 CUDA tensors (arcsec)."""
    B = _check_dev(h, params_dev)
    if xy_dev.dim() != 3 or xy_dev.shape[0] != B or xy_dev.shape[2] != 2 or xy_dev.shape[1] < 1:
        raise LensedError(EINVAL, "xy must be [B][K][2]")
    for t in (xy_dev, out_dev):
        _check_out(t, B, xy_dev.numel())
    _check(lib().lensed_deflect(h, params_dev.data_ptr(), B, xy_dev.data_ptr(), int(xy_dev.shape[1]),
                                out_dev.data_ptr(), _stream(stream)), h)
    return out_dev


def lensed_image_plane_prior(h, params_dev, source_models, stream=None):
    """In place: the (x, y) of the listed source components, image plane -> source plane."""
    B = _check_dev(h, params_dev)
    idx = _np(source_models, np.int32).reshape(-1)
    _check(lib().lensed_image_plane_prior(h, params_dev.data_ptr(), B, _hp(idx), len(idx), _stream(stream)), h)
    return params_dev


def lensed_render_host(h, params_host, model_host, stream=None):
    """Host float32 arrays (numpy, or pinned torch CPU tensors); returns after the copy back."""
    pin, B = _host_ptr(params_host, lensed_num_params(h))
    pout, _ = _host_ptr(model_host, None)
    _check(lib().lensed_render_host(h, pin, B, pout, _stream(stream)), h)
    return model_host


def lensed_loglike_host(h, params_host, logl_host, stream=None):
    pin, B = _host_ptr(params_host, lensed_num_params(h))
    pout, _ = _host_ptr(logl_host, None)
    _check(lib().lensed_loglike_host(h, pin, B, pout, _stream(stream)), h)
    return logl_host


CHISQ_STATIC_MAX_VECTORS = 4096     # LENSED_CHISQ_STATIC_MAX_VECTORS (include/lensed.h)


def lensed_chisq_static(image_dev, weight_dev, model_dev, logl_dev, stream=None):
    """logL of model images already on the device, from a call that allocates no device memory
    (for callers that may not: see lensed.h).  image_dev / weight_dev [n_pix] (weight 0 where
    masked), model_dev [B][n_pix] or [B][H][W], logl_dev [B]: contiguous float32 CUDA tensors on
    one device.  At most CHISQ_STATIC_MAX_VECTORS images per call; calls that overlap on the GPU
    race on the library's one scratch array.  Marshalling only: no tensor is created here."""
    for t in (image_dev, weight_dev, model_dev, logl_dev):
        if not (t.is_cuda and t.is_contiguous() and str(t.dtype) == "torch.float32"):
            raise LensedError(EINVAL, "lensed_chisq_static takes contiguous float32 CUDA tensors")
        if t.device != image_dev.device:
            raise LensedError(EINVAL, "lensed_chisq_static: tensors on different devices")
    n_pix, B = int(image_dev.numel()), int(logl_dev.numel())
    if weight_dev.numel() != n_pix or B < 1 or model_dev.numel() != B * n_pix or model_dev.shape[0] != B:
        raise LensedError(EINVAL, "lensed_chisq_static: image / weight [n_pix], model [B][n_pix], logl [B]")
    _check(lib().lensed_chisq_static(int(image_dev.device.index or 0), image_dev.data_ptr(), weight_dev.data_ptr(), n_pix,
                                     model_dev.data_ptr(), B, logl_dev.data_ptr(), _stream(stream)))
    return logl_dev


def lensed_set_profiling(h, on):
    _check(lib().lensed_set_profiling(h, int(bool(on))), h)


def lensed_get_profile(h):
    """-> ({phase: ms}, {phase: launches}) since the last reset."""
    ms = (ctypes.c_double * len(PHASES))()
    n = (ctypes.c_longlong * len(PHASES))()
    _check(lib().lensed_get_profile(h, ms, n), h)
    return dict(zip(PHASES, ms)), dict(zip(PHASES, n))


def lensed_reset_profile(h):
    _check(lib().lensed_reset_profile(h), h)


def lensed_set_refine(h, gain):
    _check(lib().lensed_set_refine(h, float(gain)), h)


def lensed_set_fg_expansion(h, tau):
    _check(lib().lensed_set_fg_expansion(h, float(tau)), h)


def lensed_get_refined(h):
    """-> pixels re-traced in FP64 since the last lensed_reset_profile."""
    n = ctypes.c_longlong()
    _check(lib().lensed_get_refined(h, ctypes.byref(n)), h)
    return n.value


def lensed_debug_fill_frames(h, value):
    """overwrite every cell of the handle's scratch frames (lensed_tune.h): uninitialised-read check"""
    _check(lib().lensed_debug_fill_frames(h, float(value)), h)


def lensed_set_chunk_bytes(h, nbytes):
    _check(lib().lensed_set_chunk_bytes(h, int(nbytes)), h)


def lensed_frame_bytes(h):
    return lib().lensed_frame_bytes(h)


CONV_SHAPES = ("narrow", "wide", "strip", "half")     # lensed_set_conv_shape / lensed_get_conv_shape: 0, 1, 2, 3


def lensed_set_conv_shape(h, shape):
    _check(lib().lensed_set_conv_shape(h, int(shape)), h)


def lensed_get_conv_shape(h):
    return lib().lensed_get_conv_shape(h)


def lensed_uses_global_taps(h):
    return lib().lensed_uses_global_taps(h)


def lensed_debug_force_global_taps(on):
    lib().lensed_debug_force_global_taps(int(bool(on)))


def lensed_set_static_tracer(h, on):
    _check(lib().lensed_set_static_tracer(h, int(bool(on))), h)


def lensed_get_static_tracer(h):
    return lib().lensed_get_static_tracer(h)


def lensed_debug_jit_compile(models, n_quad):
    """-> (cubin bytes or -1, log): the NVRTC step of the run-time specialisation alone (no device needed)"""
    m = _np(models, np.int32).reshape(-1)
    log = ctypes.create_string_buffer(2048)
    n = lib().lensed_debug_jit_compile(_hp(m), len(m), int(n_quad), log, len(log))
    return n, log.value.decode(errors="replace")


class NsOptions(ctypes.Structure):
    _fields_ = [("n_live", _i), ("batch", _i), ("max_rounds", _i), ("tol", _d), ("enlarge", _d),
                ("seed", ctypes.c_ulonglong), ("tied_to", _p)]


class NsResult(ctypes.Structure):
    _fields_ = [("ln_z", _d), ("ln_z_err", _d), ("information", _d), ("n_rounds", _ll), ("n_likelihood", _ll),
                ("n_dead", _ll), ("n_samples", _ll), ("converged", _i)]


def lensed_ns_run(h, prior_lo, prior_hi, n_live=400, batch=256, tol=1e-3, enlarge=1.2, seed=1, max_rounds=100000,
                  image_plane_sources=None, tied_to=None, samples_dev=None, logl_dev=None, logw_dev=None, stream=None):
    """-> dict of the lensed_ns_result fields.  prior_lo / prior_hi: host arrays [P]; the three
    output tensors (float32 CUDA, [cap][P], [cap], [cap]) are optional."""
    lo, hi = _np(prior_lo, np.float32), _np(prior_hi, np.float32)
    P = lensed_num_params(h)
    if lo.shape != (P,) or hi.shape != (P,):
        raise LensedError(EINVAL, "priors must be [%d]" % P)
    ip = None if image_plane_sources is None else _np(image_plane_sources, np.int32).reshape(-1)
    cap = 0
    if samples_dev is not None:
        cap = int(samples_dev.shape[0])
        _check_out(samples_dev, cap, cap * P)
        _check_out(logl_dev, cap, cap)
        _check_out(logw_dev, cap, cap)
    tied = None if tied_to is None else _np(tied_to, np.int32).reshape(-1)
    if tied is not None and tied.shape != (P,):
        raise LensedError(EINVAL, "tied_to must be [%d]" % P)
    opt = NsOptions(int(n_live), int(batch), int(max_rounds), float(tol), float(enlarge), int(seed), _hp(tied))
    res = NsResult()
    ptr = lambda t: None if t is None else ctypes.c_void_p(t.data_ptr())
    _check(lib().lensed_ns_run(h, _hp(lo), _hp(hi), _hp(ip), 0 if ip is None else len(ip), ctypes.byref(opt),
                               ctypes.byref(res), ptr(samples_dev), ptr(logl_dev), ptr(logw_dev), cap,
                               _stream(stream)), h)
    return {k: getattr(res, k) for k, _ in NsResult._fields_}


def lensed_ns_philox(counter, key):
    c = (ctypes.c_uint * 4)(*[int(x) for x in counter])
    k = (ctypes.c_uint * 2)(*[int(x) for x in key])
    out = (ctypes.c_uint * 4)()
    lib().lensed_ns_philox(c, k, out)
    return [int(x) for x in out]


def lensed_fma_peak(device=0, iters=4096):
    t = ctypes.c_double()
    _check(lib().lensed_fma_peak(int(device), int(iters), ctypes.byref(t)))
    return t.value


def lensed_issue_probe(device=0, kind=0, n_extra=0, warps=2):
    """-> SM cycles per body of 64 FFMA2 + n_extra instructions of `kind` (include/lensed.h)"""
    out = ctypes.c_double()
    _check(lib().lensed_issue_probe(int(device), int(kind), int(n_extra), int(warps), ctypes.byref(out)))
    return out.value


def lensed_last_error(h=None):
    t = lib().lensed_last_error(h)
    return t.decode() if t else ""


def lensed_destroy(h):
    if h is not None and h.value:
        lib().lensed_destroy(h)
        h.value = None


def _check_dev(h, params_dev):
    P = lensed_num_params(h)
    if not (params_dev.is_cuda and params_dev.is_contiguous() and str(params_dev.dtype) == "torch.float32"):
        raise LensedError(EINVAL, "params must be a contiguous float32 CUDA tensor")
    if params_dev.dim() != 2 or params_dev.shape[1] != P:
        raise LensedError(EINVAL, "params must be [B][%d]" % P)
    return int(params_dev.shape[0])


def _check_out(t, B, numel):
    if not (t.is_cuda and t.is_contiguous() and str(t.dtype) == "torch.float32" and t.dim() >= 1
            and t.shape[0] == B and t.numel() == numel):
        raise LensedError(EINVAL, "output must be a contiguous float32 CUDA tensor of %d elements with leading dim %d"
                          % (numel, B))


def _host_ptr(a, P):
    if isinstance(a, np.ndarray):
        if a.dtype != np.float32 or not a.flags["C_CONTIGUOUS"]:
            raise LensedError(EINVAL, "host arrays must be contiguous float32")
        B = a.shape[0] if P is None else a.size // P
        return ctypes.c_void_p(a.ctypes.data), int(B)
    if a.is_cuda or not a.is_contiguous() or str(a.dtype) != "torch.float32":
        raise LensedError(EINVAL, "host tensors must be contiguous float32 CPU tensors")
    B = a.shape[0] if P is None else a.numel() // P
    return ctypes.c_void_p(a.data_ptr()), int(B)
