// trace_sig_i.cu -- static ray tracer for the paper's largest fitted model, SDSS J0808+4706
// (PAPER.md:357): two SIE lenses, three Sersic components for the foreground galaxies, two
// Sersic components for the background source (+ sky, which does not enter a signature)
// (trace_static.cuh; signature = shear, SIE, SIS, point | source Sersic, source Gaussian,
// foreground Sersic, foreground Gaussian).
#include "trace_static.cuh"

namespace lensed {
#ifndef LENSED_MINB_I
#define LENSED_MINB_I 2
#endif
LENSED_DEFINE_STATIC_TRACER(trace_static_i, LENSED_MINB_I, 0, 2, 0, 0, 2, 0, 3, 0)
}  // namespace lensed
