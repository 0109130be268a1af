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
