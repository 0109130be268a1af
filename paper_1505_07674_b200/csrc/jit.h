// jit.h -- run-time specialisation of the ray tracer (jit.cu); host side only.
#pragma once
#include "lensed_internal.h"
#include <string>

namespace lensed {

struct JitTracer;
constexpr unsigned kJitThreads = 256;           // = kTraceThreads of the default build (trace_block.cuh)

bool jit_wanted(const int (&counts)[K_COUNT]);
const JitTracer *jit_get(const int (&counts)[K_COUNT], int np, int device, std::string *why);
cudaError_t jit_launch(const JitTracer *t, const Program &prog, const TraceArgs &a, int nvec, cudaStream_t st);

}  // namespace lensed
