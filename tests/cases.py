"""Test-side glue: build one problem from a synth.Config for BOTH sides.

The oracle (tests only) renders the noiseless truth, synth.observe() adds the seeded noise,
and the same host arrays go to oracle.loglike and to lensed_create.  No arithmetic of the
method lives here.
"""
import numpy as np

from oracle import lensed_oracle as orc
from paper_1505_07674_b200 import synth

PIXEL_RTOL = 1e-4      # north_star: relative 1e-4 per rendered pixel ...
PIXEL_FLOOR = 1e-3     # ... for pixels above 1e-3 of the image peak
LOGL_RTOL = 1e-5       # north_star: 1e-5 relative on logL


class Problem:
    def __init__(self, cfg, image=None, weight=None):
        self.cfg = cfg
        self.kinds = synth.kind_ids(cfg.models)
        if image is None:
            truth = orc.render(cfg.H, cfg.W, cfg.scale, cfg.psf, cfg.quad, self.kinds,
                               cfg.truth.astype(np.float32), zp=cfg.zp)[0]
            image, weight = cfg.observe(truth)
        self.image, self.weight = image, weight

    def oracle_loglike(self, params, want_model=True):
        c = self.cfg
        return orc.loglike(c.H, c.W, c.scale, self.image, self.weight, c.mask, c.psf, c.quad,
                           self.kinds, params, zp=c.zp, want_model=want_model)

    def create(self, device=0):
        from paper_1505_07674_b200 import lensed
        c = self.cfg
        return lensed.lensed_create(self.image, self.weight, c.mask, c.psf, c.quad, self.kinds,
                                    c.scale, c.zp, device)


def pixel_errors(model_gpu, model_ref):
    """max relative error over pixels above PIXEL_FLOOR of each image's peak, per vector."""
    out = []
    for g, r in zip(model_gpu, model_ref):
        peak = np.abs(r).max()
        sel = np.abs(r) > PIXEL_FLOOR * peak
        out.append(float(np.max(np.abs(g[sel] - r[sel]) / np.abs(r[sel]))) if sel.any() else 0.0)
    return np.array(out)


def logl_errors(logl_gpu, logl_ref):
    return np.abs(np.asarray(logl_gpu, dtype=np.float64) - logl_ref) / np.maximum(np.abs(logl_ref), 1e-300)


# ---------------------------------------------------------------------------- parameter domain
# Hand-written expectations for the parameter domain, shared by the CPU pin of the oracle
# (test_oracle_pins.py) and the GPU test (test_parity_gpu.py): neither side's code wrote them.
# SURVEY.md section 8(b) "Errors" fixes: q outside (0, 1], r <= 0 (Sersic), sigma <= 0, n <= 0 and
# non-finite values are outside the domain.  DESIGN.md section 2 "Domain" adds this build's two
# readings: 0.02 <= n <= 20, and r = 0 allowed for the lenses (a lens of zero mass deflects nothing).
DOMAIN_BASE = {
    "sis": [0.01, -0.02, 0.3], "point": [0.01, -0.02, 0.05], "sie": [0.01, -0.02, 0.3, 0.7, 30.0],
    "shear": [0.03, -0.02],
    "src_sersic": [0.02, 0.01, 0.1, -1.0, 1.5, 0.7, 40.0], "fg_sersic": [0.02, 0.01, 0.1, -1.0, 1.5, 0.7, 40.0],
    "src_gauss": [0.02, 0.01, 0.08, -1.0, 0.7, 40.0], "fg_gauss": [0.02, 0.01, 0.08, -1.0, 0.7, 40.0],
    "sky": [0.1],
}
_DOMAIN_EDGES = {                      # kind -> (slot, value, inside the domain?)
    "sis": [(2, -1e-3, False), (2, 0.0, True)],
    "point": [(2, -1e-3, False), (2, 0.0, True)],
    "sie": [(2, -1e-3, False), (2, 0.0, True), (3, 0.0, False), (3, -0.5, False), (3, 1e-3, True), (3, 1.0, True),
            (3, 1.0001, False)],
    "shear": [(0, 5.0, True), (1, -5.0, True)],
    "src_sersic": [(2, 0.0, False), (2, -0.1, False), (2, 1e-3, True), (4, 0.0, False), (4, 0.0199, False), (4, 0.0201, True),
                   (4, 20.0, True), (4, 20.01, False), (5, 0.0, False), (5, 1.0, True), (5, 1.0001, False)],
    "src_gauss": [(2, 0.0, False), (2, -0.1, False), (2, 1e-3, True), (4, 0.0, False), (4, 1.0, True), (4, 1.0001, False)],
    "sky": [(0, -3.0, True)],
}
_DOMAIN_EDGES["fg_sersic"] = _DOMAIN_EDGES["src_sersic"]
_DOMAIN_EDGES["fg_gauss"] = _DOMAIN_EDGES["src_gauss"]


def domain_cases():
    """-> [(models, params float32, valid)]: for every kind one vector just inside and one just
    outside every bound, and NaN / +inf / -inf in every slot.  A lens comes with a Gaussian source
    behind it so that there is something to render."""
    out = []
    for kind, base in DOMAIN_BASE.items():
        lens = kind in ("sis", "point", "sie", "shear")
        models = (kind, "src_gauss") if lens else (kind,)
        tail = DOMAIN_BASE["src_gauss"] if lens else []
        rows = list(_DOMAIN_EDGES[kind]) + [(s, v, False) for s in range(len(base)) for v in (np.nan, np.inf, -np.inf)]
        rows.append((0, base[0], True))                          # the base vector itself
        for slot, value, valid in rows:
            p = np.array(list(base) + list(tail), dtype=np.float32)
            p[slot] = value
            out.append((models, p, valid))
    return out
