// jit.h -- run-time specialisation of the ray tracer (jit.cu); host side only.
#pragma once
#include "lensed_internal.h"
#include <string>
#include <vector>

namespace lensed {

struct JitTracer;
constexpr unsigned kJitThreads = 256;           // = kTraceThreads of the default build (trace_block.cuh)

std::string jit_compile(const int (&counts)[K_COUNT], int np, int minb, std::vector<char> *cubin, std::string *name);
bool jit_wanted(const int (&counts)[K_COUNT]);
const JitTracer *jit_get(const int (&counts)[K_COUNT], int np, int device, std::string *why);
cudaError_t jit_launch(const JitTracer *t, const Program &prog, const TraceArgs &a, int nvec, cudaStream_t st);

}  // namespace lensed
