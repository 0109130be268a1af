// trace_sig_b.cu -- static ray tracer for the model list of the HST-like and Euclid-scale configs: SIE + shear, Sersic source, Sersic lens light
// (trace_static.cuh; signature = shear, SIE, SIS, point | source Sersic, source Gaussian,
// foreground Sersic, foreground Gaussian).
#include "trace_static.cuh"

namespace lensed {
#ifndef LENSED_MINB_B
#define LENSED_MINB_B 3
#endif
LENSED_DEFINE_STATIC_TRACER(trace_static_b, LENSED_MINB_B, 1, 1, 0, 0, 1, 0, 1, 0)
}  // namespace lensed
