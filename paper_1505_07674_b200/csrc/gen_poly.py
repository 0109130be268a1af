"""Writes the minimax polynomial tables of trace_math.cuh (output pasted there; tests/test_gen_poly.py regenerates and compares).

atan(z)/z and atanh(z)/z as polynomials in t = z^2 on [0, T], fitted in relative error by
Lawson's iteratively reweighted least squares on Chebyshev nodes (float64).  'centred'
tables are monomials in s = (2/T) t - 1, which FP32 Horner evaluates without the
cancellation the t-monomials suffer for T >~ 1; the others are monomials in t.
The atanh tables are multiplied by 2/ln 2 (the tracer carries atanh in lg2 units).
`python gen_poly.py` prints C arrays, highest degree first, and the fitted / FP32 errors.
"""
import numpy as np
from numpy.polynomial import chebyshev as C, polynomial as P


def f_atan(t):
    r = np.sqrt(np.maximum(t, 1e-300))
    return np.where(t > 1e-12, np.arctan(r) / r, 1 - t / 3)


def f_atanh(t):
    r = np.sqrt(np.maximum(t, 1e-300))
    return np.where(t > 1e-12, np.arctanh(r) / r, 1 + t / 3)


def lawson(f, T, deg, iters=40, n=4000):
    x = 0.5 * T * (1 + np.cos(np.pi * (np.arange(n) + 0.5) / n))
    s = 2 * x / T - 1
    y = f(x)
    w = np.ones(n)
    V = C.chebvander(s, deg)
    for _ in range(iters):
        sw = np.sqrt(w) / np.abs(y)
        c = np.linalg.lstsq(V * sw[:, None], y * sw, rcond=None)[0]
        e = np.abs(V @ c - y) / np.abs(y)
        w = w * e
        w /= w.sum()
    return C.cheb2poly(c), e.max()


def to_t(ms, T):
    out = np.zeros(1)
    for k in range(len(ms) - 1, -1, -1):
        out = P.polyadd(P.polymul(out, [-1.0, 2.0 / T]), [ms[k]])
    return out


def horner32(m, x):
    x = x.astype(np.float32)
    p = np.full_like(x, np.float32(m[-1]))
    for k in range(len(m) - 2, -1, -1):
        p = (p.astype(np.float64) * x + np.float32(m[k])).astype(np.float32)
    return p


TABLES = (  # name, function, T, degree, centred, scale
    ("kAtan019", f_atan, 0.16 / 0.84, 4, False, 1.0),
    ("kAtan056", f_atan, 0.36 / 0.64, 6, False, 1.0),
    ("kAtan1", f_atan, 1.0, 8, False, 1.0),
    ("kAtan2", f_atan, 2.0, 10, True, 1.0),
    ("kAtan3", f_atan, 3.0, 12, True, 1.0),
    ("kAtanh016", f_atanh, 0.16, 4, False, 2 / np.log(2)),
    ("kAtanh036", f_atanh, 0.36, 6, False, 2 / np.log(2)),
    ("kAtanh050", f_atanh, 0.50, 8, False, 2 / np.log(2)),
    ("kAtanh067", f_atanh, 2.0 / 3.0, 10, True, 2 / np.log(2)),
    ("kAtanh075", f_atanh, 0.75, 12, True, 2 / np.log(2)),
)

def generate():
    """[(name, T, degree, centred, coefficients highest degree first, fit error, FP32 Horner error)]"""
    out = []
    for name, f, T, deg, centred, scale in TABLES:
        ms, e = lawson(f, T, deg)
        m = ms if centred else to_t(ms, T)
        t = np.linspace(0, T, 200001)
        x = 2 * t / T - 1 if centred else t
        e32 = np.max(np.abs(horner32(m, x).astype(np.float64) - f(t)) / f(t))
        out.append((name, T, deg, centred, (m * scale)[::-1], e, e32))
    return out


if __name__ == "__main__":
    for name, T, deg, centred, coef, e, e32 in generate():
        print("// %s: t in [0, %.4g], degree %d, %s; fit %.2e, FP32 Horner %.2e"
              % (name, T, deg, "in s = %.9g t - 1" % (2 / T) if centred else "in t", e, e32))
        print("__device__ constexpr float %s[%d] = {%s};"
              % (name, deg + 1, ", ".join("%.10ef" % v for v in coef)))
