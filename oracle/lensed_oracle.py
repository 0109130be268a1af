"""ctypes loader for oracle/lensed_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It marshals numpy arrays into the plain-C oracle and
holds no arithmetic of the method itself; every formula lives in lensed_oracle.c
with its PAPER.md citation.  It shares nothing with paper_1505_07674_b200/.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lensed_oracle.c")
_LIB = os.path.join(_HERE, "liblensed_oracle.so")

# Model kinds, the enum of lensed_oracle.c (order of the paper's object list,
# PAPER.md:37, 351; parameter order PAPER.md:345, 254).
LENS_SIS, LENS_SIE, LENS_POINT, LENS_SHEAR = 0, 1, 2, 3
SRC_SERSIC, SRC_GAUSS, FG_SERSIC, FG_GAUSS, FG_SKY = 4, 5, 6, 7, 8


_SAN = os.environ.get("LENSED_ORACLE_SANITIZE") == "1"
if _SAN:
    _LIB = os.path.join(_HERE, "liblensed_oracle_san.so")


def build(force=False):
    """gcc -O2 (no fast-math) build of the oracle, the command its header states.  With
    LENSED_ORACLE_SANITIZE=1 in the environment: an -fsanitize=address,undefined build beside it
    (tests/test_oracle_sanitized.py runs the pins on it; the process must preload libasan)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        flags = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
                 "-fno-omit-frame-pointer"] if _SAN else ["-O2"]
        subprocess.check_call(
            ["gcc"] + flags + ["-std=c99", "-fopenmp", "-fPIC", "-shared", _SRC, "-o", _LIB, "-lm"])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        d, i, p = ctypes.c_double, ctypes.c_int, ctypes.c_void_p
        L.oracle_kind_num_params.restype = i
        L.oracle_kind_num_params.argtypes = [i]
        L.oracle_num_params.restype = i
        L.oracle_num_params.argtypes = [p, i]
        L.oracle_gamma_p.restype = d
        L.oracle_gamma_p.argtypes = [d, d]
        L.oracle_sersic_bn.restype = d
        L.oracle_sersic_bn.argtypes = [d]
        L.oracle_deflection.restype = None
        L.oracle_deflection.argtypes = [i, p, d, d, p, p]
        L.oracle_potential.restype = d
        L.oracle_potential.argtypes = [i, p, d, d]
        L.oracle_brightness.restype = d
        L.oracle_brightness.argtypes = [i, p, d, d, d, d]
        L.oracle_render_raw.restype = i
        L.oracle_render_raw.argtypes = [i, i, d, p, i, p, i, d, p, p]
        L.oracle_convolve.restype = None
        L.oracle_convolve.argtypes = [p, i, i, p, i, i, p]
        L.oracle_chi2_loglike.restype = d
        L.oracle_chi2_loglike.argtypes = [p, p, p, p, ctypes.c_long]
        L.oracle_render.restype = i
        L.oracle_render.argtypes = [i, i, d, p, i, i, p, i, p, i, d, p, i, p, i]
        L.oracle_loglike.restype = i
        L.oracle_loglike.argtypes = [i, i, d, p, p, p, p, i, i, p, i, p, i, d, p, i, p, p, i]
        L.oracle_source_position.restype = i
        L.oracle_source_position.argtypes = [p, i, p, p, i, p]
        L.oracle_estimate_weights.restype = ctypes.c_long
        L.oracle_estimate_weights.argtypes = [ctypes.c_long, p, p, d, p, d, p, p, p]
        L.oracle_threads.restype = i
        L.oracle_threads.argtypes = []
        _lib = L
    return _lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _kinds(kinds):
    return np.ascontiguousarray(kinds, dtype=np.int32)


def num_params(kinds):
    k = _kinds(kinds)
    return lib().oracle_num_params(_ptr(k), len(k))


def gamma_p(a, x):
    return lib().oracle_gamma_p(float(a), float(x))


def sersic_bn(n):
    return lib().oracle_sersic_bn(float(n))


def deflection(kind, p, x, y):
    p = _f64(p)
    ax, ay = ctypes.c_double(), ctypes.c_double()
    lib().oracle_deflection(int(kind), _ptr(p), float(x), float(y),
                            ctypes.addressof(ax), ctypes.addressof(ay))
    return ax.value, ay.value


def potential(kind, p, x, y):
    p = _f64(p)
    return lib().oracle_potential(int(kind), _ptr(p), float(x), float(y))


def brightness(kind, p, x, y, scale=1.0, zp=0.0):
    p = _f64(p)
    return lib().oracle_brightness(int(kind), _ptr(p), float(x), float(y), float(scale), float(zp))


def source_position(kinds, params, xy):
    """y(x) = x - sum_lenses alpha(x) (eq. 1) for the K image-plane points xy[K][2] of ONE
    parameter vector; NaN if a lens of the vector is outside the domain."""
    k, params = _kinds(kinds), _f64(params)
    xy = _f64(xy).reshape(-1, 2)
    out = np.empty_like(xy)
    lib().oracle_source_position(_ptr(k), len(k), _ptr(params), _ptr(xy), len(xy), _ptr(out))
    return out


def estimate_weights(image, gain, offset=0.0, extra=None, want_variance=False):
    """w_i = x_i g_i / (d_i + b_i) (eqs. 18-21); gain / offset: scalars or maps."""
    img = _f64(image)
    g = None if np.isscalar(gain) else _f64(gain)
    b = None if np.isscalar(offset) else _f64(offset)
    x = None if extra is None else _f64(extra)
    w = np.empty_like(img)
    var = np.empty_like(img) if want_variance else None
    rc = lib().oracle_estimate_weights(img.size, _ptr(img), _ptr(g), float(gain) if g is None else 0.0,
                                       _ptr(b), float(offset) if b is None else 0.0, _ptr(x), _ptr(w), _ptr(var))
    if rc < 0:
        raise ValueError("oracle_estimate_weights: input outside the domain")
    return (w, var) if want_variance else w


def render_raw(H, W, scale, quad, kinds, params, zp=0.0):
    """Unconvolved pixel luminosities L[H][W] of ONE parameter vector (eq. 14)."""
    quad, k, params = _f64(quad).reshape(-1, 3), _kinds(kinds), _f64(params)
    out = np.empty((H, W), dtype=np.float64)
    lib().oracle_render_raw(H, W, float(scale), _ptr(quad), len(quad), _ptr(k), len(k),
                            float(zp), _ptr(params), _ptr(out))
    return out


def error_map(H, W, scale, quad, w_embedded, kinds, params, zp=0.0):
    """Per-pixel error estimate of the pixel quadrature: the definition written
    out with render_raw,  | sum_k w_k I(x_k) - sum_k w'_k I(x_k) |,  w' = the embedded rule's
    weights at the same abscissae (render_raw renormalises each weight set to sum 1, R6)."""
    quad = _f64(quad).reshape(-1, 3)
    emb = quad.copy()
    emb[:, 2] = _f64(w_embedded)
    return np.abs(render_raw(H, W, scale, quad, kinds, params, zp)
                  - render_raw(H, W, scale, emb, kinds, params, zp))


def convolve(L, psf):
    """eq. 15 with replicate padding and automatic PSF normalisation."""
    L = _f64(L)
    H, W = L.shape
    out = np.empty_like(L)
    if psf is None:
        lib().oracle_convolve(_ptr(L), H, W, None, 1, 1, _ptr(out))
    else:
        psf = _f64(psf)
        lib().oracle_convolve(_ptr(L), H, W, _ptr(psf), psf.shape[0], psf.shape[1], _ptr(out))
    return out


def chi2_loglike(model, image, weight, mask=None):
    model, image, weight = _f64(model), _f64(image), _f64(weight)
    m = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    return lib().oracle_chi2_loglike(_ptr(model), _ptr(image), _ptr(weight), _ptr(m), model.size)


def render(H, W, scale, psf, quad, kinds, params, zp=0.0, nthreads=0):
    """Model images L*[B][H][W] (double) for params[B][P]."""
    quad, k = _f64(quad).reshape(-1, 3), _kinds(kinds)
    params = _f64(params)
    params = params.reshape(1, -1) if params.ndim == 1 else params
    B = params.shape[0]
    ps = None if psf is None else _f64(psf)
    ph, pw = (1, 1) if ps is None else ps.shape
    out = np.empty((B, H, W), dtype=np.float64)
    rc = lib().oracle_render(H, W, float(scale), _ptr(ps), ph, pw, _ptr(quad), len(quad),
                             _ptr(k), len(k), float(zp), _ptr(params), B, _ptr(out), int(nthreads))
    if rc != 0:
        raise RuntimeError("oracle_render failed: %d" % rc)
    return out


def loglike(H, W, scale, image, weight, mask, psf, quad, kinds, params, zp=0.0,
            want_model=False, nthreads=0):
    """logL[B] (double) and, if asked, the B convolved model images."""
    quad, k = _f64(quad).reshape(-1, 3), _kinds(kinds)
    params = _f64(params)
    params = params.reshape(1, -1) if params.ndim == 1 else params
    B = params.shape[0]
    image, weight = _f64(image), _f64(weight)
    m = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    ps = None if psf is None else _f64(psf)
    ph, pw = (1, 1) if ps is None else ps.shape
    logl = np.empty(B, dtype=np.float64)
    model = np.empty((B, H, W), dtype=np.float64) if want_model else None
    rc = lib().oracle_loglike(H, W, float(scale), _ptr(image), _ptr(weight), _ptr(m), _ptr(ps),
                              ph, pw, _ptr(quad), len(quad), _ptr(k), len(k), float(zp),
                              _ptr(params), B, _ptr(logl), _ptr(model), int(nthreads))
    if rc != 0:
        raise RuntimeError("oracle_loglike failed: %d" % rc)
    return (logl, model) if want_model else logl


def threads():
    return lib().oracle_threads()
