"""Nested sampling on the CPU -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

The textbook algorithm (Skilling 2004, 2006; cited PAPER.md:170), step by step in plain numpy
(float64), for checking the device-resident driver of the CUDA library (lensed_ns_run).  Only
tests/ may import this module; it shares no code with paper_1505_07674_b200/.

What the paper fixes (PAPER.md:134-139 steps iii-vii, 170, 184-186): parameters are drawn from
the prior (iii), their likelihood is computed (iv-v), the posterior is accumulated (vi), and
this repeats "until the parameter space is sufficiently sampled" (vii); the sampler is Nested
Sampling, which also yields the evidence (eq. 13).  The paper delegates the
sampler to the MultiNest library, which is not here; what follows is the base algorithm with
MultiNest's single-ellipsoid bound for the constrained prior draw (one ellipsoid, no
clustering -- reading N1 in DESIGN.md).

Algorithm (N live points, K candidates per round):
  0. u_i ~ U[0,1]^d, theta_i = lo + u_i (hi - lo) [+ image-plane map], L_i = loglike(theta_i).
  1. Bound: mean m and covariance C of the live u_i; C = G G^T (Cholesky); the ellipsoid
     {m + s G y : |y| <= 1} with s = enlarge * max_i |G^-1 (u_i - m)| holds every live point.
  2. Candidates j = 0..K-1: up to TRIES draws x = m + s r^(1/d) G z/|z| (z normal, r uniform),
     the first inside the unit cube is taken (none: the candidate is void).
  3. Their likelihoods, in one batch.
  4. In order j = 0..K-1: let L* = min_i L_i.  If L_j > L*: the worst live point dies with
     weight w = X_(k-1) - X_k, X_k = exp(-k/N) (k counts the dead), Z += L* w, the
     information H is updated (Skilling 2006 eq. 2.11), and candidate j takes its place.
     A candidate drawn uniformly inside a region that holds {L > L*_0} is, given L_j > L*,
     uniform inside {L > L*}: consuming the batch in order against the rising threshold is
     the sequential algorithm.
  5. Stop when max_i L_i X_k < tol Z; else back to 1.
  6. The live points join the dead with weight X_k / N each.
Random numbers: the counter-based generator Philox4x32-10 (Salmon et al. 2011), restated
here; the CUDA driver states it again on its side, so both draw the same numbers from
(seed, stream, round, candidate, try).
"""
import math

import numpy as np

TRIES = 16
_M0, _M1 = np.uint64(0xD2511F53), np.uint64(0xCD9E8D57)
_W0, _W1 = np.uint32(0x9E3779B9), np.uint32(0xBB67AE85)
_MASK = np.uint64(0xFFFFFFFF)


def philox4x32(c0, c1, c2, c3, k0, k1):
    """Philox4x32-10; every argument a uint32 array of one shape (or scalar); -> 4 uint32 arrays."""
    c = [np.asarray(x, dtype=np.uint32) for x in np.broadcast_arrays(c0, c1, c2, c3)]
    k0, k1 = np.uint32(k0), np.uint32(k1)
    with np.errstate(over="ignore"):
        for _ in range(10):
            p0 = _M0 * c[0].astype(np.uint64)
            p1 = _M1 * c[2].astype(np.uint64)
            hi0, lo0 = (p0 >> np.uint64(32)).astype(np.uint32), (p0 & _MASK).astype(np.uint32)
            hi1, lo1 = (p1 >> np.uint64(32)).astype(np.uint32), (p1 & _MASK).astype(np.uint32)
            c = [hi1 ^ c[1] ^ k0, lo1, hi0 ^ c[3] ^ k1, lo0]
            k0, k1 = np.uint32(k0 + _W0), np.uint32(k1 + _W1)
    return c


def _unit(x):
    """uint32 -> double in (0, 1)"""
    return (x.astype(np.float64) + 0.5) * 2.0 ** -32


def uniforms4(seed, stream, a, b, c):
    """4 uniforms in (0, 1) per counter (a, b, c, stream), key = the 64-bit seed"""
    w = philox4x32(a, b, c, stream, seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF)
    return [_unit(x) for x in w]


def normals4(seed, stream, a, b, c):
    """4 standard normals per counter: Box-Muller on the pairs (u0, u1), (u2, u3)"""
    u = uniforms4(seed, stream, a, b, c)
    r0, r1 = np.sqrt(-2.0 * np.log(u[0])), np.sqrt(-2.0 * np.log(u[2]))
    t0, t1 = 2.0 * math.pi * u[1], 2.0 * math.pi * u[3]
    return [r0 * np.cos(t0), r0 * np.sin(t0), r1 * np.cos(t1), r1 * np.sin(t1)]


STREAM_INIT, STREAM_DIR, STREAM_RADIUS = 0, 1, 2


def initial_points(seed, n_live, d):
    u = np.empty((n_live, d))
    i = np.arange(n_live, dtype=np.uint32)
    for blk in range((d + 3) // 4):
        w = uniforms4(seed, STREAM_INIT, i, blk, 0)
        for e in range(4):
            if 4 * blk + e < d:
                u[:, 4 * blk + e] = w[e]
    return u


def bound(u, enlarge):
    """(mean, Cholesky factor G, scale s) of the ellipsoid m + s G y, |y| <= 1, around the live points"""
    n, d = u.shape
    m = u.mean(axis=0)
    x = u - m
    C = x.T @ x / n
    C[np.diag_indices(d)] += 1e-30
    G = np.linalg.cholesky(C)
    y = np.linalg.solve(G, x.T)                              # G^-1 (u_i - m), triangular system
    s = enlarge * math.sqrt(float((y * y).sum(axis=0).max()))
    return m, G, s


def propose(seed, rnd, K, m, G, s):
    """K candidates of round rnd; void candidates come back as NaN rows"""
    d = len(m)
    out = np.full((K, d), np.nan)
    todo = np.ones(K, dtype=bool)
    j = np.arange(K, dtype=np.uint32)
    for t in range(TRIES):
        z = np.empty((K, d))
        for blk in range((d + 3) // 4):
            w = normals4(seed, STREAM_DIR, rnd, j, t * 64 + blk)
            for e in range(4):
                if 4 * blk + e < d:
                    z[:, 4 * blk + e] = w[e]
        r = uniforms4(seed, STREAM_RADIUS, rnd, j, t)[0] ** (1.0 / d)
        y = z / np.sqrt((z * z).sum(axis=1))[:, None] * r[:, None]
        x = m + s * (y @ G.T)
        ok = todo & np.all((x > 0.0) & (x < 1.0), axis=1)
        out[ok] = x[ok]
        todo &= ~ok
        if not todo.any():
            break
    return out


def run(loglike, lo, hi, n_live=400, batch=256, tol=1e-3, enlarge=1.2, seed=1, max_rounds=100000,
        transform=None):
    """loglike(theta[B][P]) -> logL[B].  lo == hi fixes a parameter.  transform(theta) -> theta,
    applied after the box prior (the image-plane map).  Returns a dict: ln_z, ln_z_err,
    information, n_rounds, n_likelihood, n_dead, converged, samples[M][P], logl[M], logw[M]
    (logw normalised: sum exp(logw) = 1), and first_candidates (round 0, for parity checks)."""
    lo, hi = np.asarray(lo, dtype=np.float64), np.asarray(hi, dtype=np.float64)
    free = np.flatnonzero(hi > lo)
    d, N = len(free), n_live

    def theta_of(u):
        t = np.tile(lo, (len(u), 1))
        t[:, free] = lo[free] + u * (hi[free] - lo[free])
        t = t.astype(np.float32).astype(np.float64)          # the likelihood takes float32 vectors
        return transform(t) if transform is not None else t

    u = initial_points(seed, N, d)
    theta = theta_of(u)
    logl = np.asarray(loglike(theta), dtype=np.float64).copy()
    n_like = N
    ln_z, ln_x, info = -np.inf, 0.0, 0.0
    ln_shell = math.log(1.0 - math.exp(-1.0 / N))           # ln (X_(k-1) - X_k) - ln X_(k-1)
    dead_theta, dead_logl, dead_logw = [], [], []
    converged, first = False, None
    rnd = 0
    while rnd < max_rounds and not converged:
        m, G, s = bound(u, enlarge)
        cu = propose(seed, rnd, batch, m, G, s)
        void = np.isnan(cu[:, 0])
        ct = theta_of(np.where(void[:, None], 0.5, cu))
        cl = np.asarray(loglike(ct), dtype=np.float64).copy()
        cl[void] = -np.inf
        n_like += batch
        if rnd == 0:
            first = (cu.copy(), ct.copy())
        for j in range(batch):
            worst = int(np.argmin(logl))
            if not cl[j] > logl[worst]:
                continue
            ls, lw = logl[worst], ln_x + ln_shell
            ln_z_new = np.logaddexp(ln_z, ls + lw)
            # Skilling (2006) eq. 2.11:  H <- e^(L* w)/Z' ln L* + Z/Z' (H + ln Z) - ln Z'
            info = (math.exp(ls + lw - ln_z_new) * ls
                    + (math.exp(ln_z - ln_z_new) * (info + ln_z) if np.isfinite(ln_z) else 0.0) - ln_z_new)
            ln_z = ln_z_new
            dead_theta.append(theta[worst].copy()); dead_logl.append(ls); dead_logw.append(lw)
            ln_x -= 1.0 / N
            u[worst], theta[worst], logl[worst] = cu[j], ct[j], cl[j]
        rnd += 1
        converged = bool(logl.max() + ln_x < ln_z + math.log(tol))
    lw_live = ln_x - math.log(N)
    for i in np.argsort(logl):                                # the live points join, lowest first
        ln_z_new = np.logaddexp(ln_z, logl[i] + lw_live)
        info = (math.exp(logl[i] + lw_live - ln_z_new) * logl[i]
                + (math.exp(ln_z - ln_z_new) * (info + ln_z) if np.isfinite(ln_z) else 0.0) - ln_z_new)
        ln_z = ln_z_new
        dead_theta.append(theta[i].copy()); dead_logl.append(logl[i]); dead_logw.append(lw_live)
    dead_logl, dead_logw = np.array(dead_logl), np.array(dead_logw)
    return dict(ln_z=float(ln_z), ln_z_err=math.sqrt(max(info, 0.0) / N), information=float(info), n_rounds=rnd,
                n_likelihood=n_like, n_dead=len(dead_logl) - N, converged=converged,
                samples=np.array(dead_theta), logl=dead_logl, logw=dead_logl + dead_logw - ln_z,
                first_candidates=first)


def posterior_moments(res):
    w = np.exp(res["logw"])
    w /= w.sum()
    mean = (w[:, None] * res["samples"]).sum(axis=0)
    var = (w[:, None] * (res["samples"] - mean) ** 2).sum(axis=0)
    return mean, np.sqrt(var)
