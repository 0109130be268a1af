// trace_sig_c.cu -- static ray tracer for the model list of the SLACS-like config: SIE + shear, 2 Sersic sources, Sersic lens light
// (trace_static.cuh; signature = shear, SIE, SIS, point | source Sersic, source Gaussian,
// foreground Sersic, foreground Gaussian).
#include "trace_static.cuh"

namespace lensed {
#ifndef LENSED_MINB_C
#define LENSED_MINB_C 3
#endif
LENSED_DEFINE_STATIC_TRACER(trace_static_c, LENSED_MINB_C, 1, 1, 0, 0, 2, 0, 1, 0)
}  // namespace lensed
