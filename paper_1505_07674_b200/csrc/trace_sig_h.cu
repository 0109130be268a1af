// trace_sig_h.cu -- static ray tracer for a common list outside BASELINE.json's configs:
// a single SIS and a Sersic source
// (trace_static.cuh; signature = shear, SIE, SIS, point | source Sersic, source Gaussian,
// foreground Sersic, foreground Gaussian; any number of sky components).
#include "trace_static.cuh"

namespace lensed {
#ifndef LENSED_MINB_H
#define LENSED_MINB_H 3
#endif
LENSED_DEFINE_STATIC_TRACER(trace_static_h, LENSED_MINB_H, 0, 0, 1, 0, 1, 0, 0, 0)
}  // namespace lensed
