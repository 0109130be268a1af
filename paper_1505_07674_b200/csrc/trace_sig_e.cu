// trace_sig_e.cu -- static ray tracer for the model list of the paper's mock scenario
// (PAPER.md:220-232, 254): SIE, Sersic source, de Vaucouleurs / Sersic host
// (trace_static.cuh; signature = shear, SIE, SIS, point | source Sersic, source Gaussian,
// foreground Sersic, foreground Gaussian).
#include "trace_static.cuh"

namespace lensed {
#ifndef LENSED_MINB_E
#define LENSED_MINB_E 3
#endif
LENSED_DEFINE_STATIC_TRACER(trace_static_e, LENSED_MINB_E, 0, 1, 0, 0, 1, 0, 1, 0)
}  // namespace lensed
