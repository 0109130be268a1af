// trace_sig_g.cu -- static ray tracer for a common list outside BASELINE.json's configs:
// SIE + shear and a Sersic source (no lens light)
// (trace_static.cuh; signature = shear, SIE, SIS, point | source Sersic, source Gaussian,
// foreground Sersic, foreground Gaussian; any number of sky components).
#include "trace_static.cuh"

namespace lensed {
#ifndef LENSED_MINB_G
#define LENSED_MINB_G 3
#endif
LENSED_DEFINE_STATIC_TRACER(trace_static_g, LENSED_MINB_G, 1, 1, 0, 0, 1, 0, 0, 0)
}  // namespace lensed
