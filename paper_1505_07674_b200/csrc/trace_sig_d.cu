// trace_sig_d.cu -- static ray tracer for the model list of the multi-lens config: 2 SIE + point mass + shear, 2 Sersic + 1 Gaussian source, Sersic lens light
// (trace_static.cuh; signature = shear, SIE, SIS, point | source Sersic, source Gaussian,
// foreground Sersic, foreground Gaussian).
#include "trace_static.cuh"

namespace lensed {
#ifndef LENSED_MINB_D
#define LENSED_MINB_D 2
#endif
LENSED_DEFINE_STATIC_TRACER(trace_static_d, LENSED_MINB_D, 1, 2, 0, 1, 2, 1, 1, 0)
}  // namespace lensed
