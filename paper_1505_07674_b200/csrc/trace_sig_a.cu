// trace_sig_a.cu -- static ray tracer for the model list of BASELINE.json's `tiny` config: SIS + Gaussian source
// (trace_static.cuh; signature = shear, SIE, SIS, point | source Sersic, source Gaussian,
// foreground Sersic, foreground Gaussian).
#include "trace_static.cuh"

namespace lensed {
#ifndef LENSED_MINB_A
#define LENSED_MINB_A 3
#endif
LENSED_DEFINE_STATIC_TRACER(trace_static_a, LENSED_MINB_A, 0, 0, 1, 0, 0, 1, 0, 0)
}  // namespace lensed
