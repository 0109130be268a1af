// jit.cu -- a specialised ray tracer for ANY model list, compiled at run time.
//
// The paper builds its device code at run time from the objects of the configuration file
// (the OpenCL kernel is compiled "at run-time", which is what lets a reconstruction
// use any combination of lens and source objects at full speed).  The B200-native equivalent: the
// specialised tracer (trace_static.cuh: model list fixed at compile time, straight-line ray loop,
// direct frames, foreground expansion, pixel pairs) is a template over the list's per-kind counts,
// so for a list that has none of the built-in signatures (trace_sig_[a-i].cu) lensed_create
// instantiates that template with NVRTC for sm_100a and loads the cubin through the driver API.
// Same source as the built-in signatures -- the headers are embedded in the library as text
// (build.py writes jit_sources.inc) -- so the arithmetic is identical; only the counts differ.
// A few seconds per new signature, once per process and device.
//
// Everything here is optional: NVRTC is looked up with dlopen (libnvrtc.so.12 of the CUDA
// toolkit); when it is missing, compilation fails or LENSED_JIT=0 is set, the list runs the
// interpreting tracer (trace.cu) as before.
#include "lensed_internal.h"
#include "jit.h"

#include <cuda.h>
#include <cudaTypedefs.h>
#include <dlfcn.h>
#include <stdio.h>
#include <stdlib.h>

#include <map>
#include <mutex>
#include <string>
#include <vector>

namespace lensed {
namespace {

#include "jit_sources.inc"        // kJitHeaderNames[], kJitHeaderTexts[], kJitHeaderCount

struct Nvrtc {
    void *lib = nullptr;
    int (*CreateProgram)(void **, const char *, const char *, int, const char *const *, const char *const *) = nullptr;
    int (*DestroyProgram)(void **) = nullptr;
    int (*AddNameExpression)(void *, const char *) = nullptr;
    int (*CompileProgram)(void *, int, const char *const *) = nullptr;
    int (*GetProgramLogSize)(void *, size_t *) = nullptr;
    int (*GetProgramLog)(void *, char *) = nullptr;
    int (*GetCUBINSize)(void *, size_t *) = nullptr;
    int (*GetCUBIN)(void *, char *) = nullptr;
    int (*GetLoweredName)(void *, const char *, const char **) = nullptr;
    bool ok = false;
};

const Nvrtc &nvrtc()
{
    static Nvrtc n;
    static std::once_flag once;
    std::call_once(once, [] {
        for (const char *name : {"libnvrtc.so.12", "libnvrtc.so", "/usr/local/cuda/lib64/libnvrtc.so.12"}) {
            n.lib = dlopen(name, RTLD_NOW | RTLD_LOCAL);
            if (n.lib) break;
        }
        if (!n.lib) return;
#define LENSED_SYM(field, sym) *(void **)(&n.field) = dlsym(n.lib, sym); if (!n.field) return;
        LENSED_SYM(CreateProgram, "nvrtcCreateProgram")
        LENSED_SYM(DestroyProgram, "nvrtcDestroyProgram")
        LENSED_SYM(AddNameExpression, "nvrtcAddNameExpression")
        LENSED_SYM(CompileProgram, "nvrtcCompileProgram")
        LENSED_SYM(GetProgramLogSize, "nvrtcGetProgramLogSize")
        LENSED_SYM(GetProgramLog, "nvrtcGetProgramLog")
        LENSED_SYM(GetCUBINSize, "nvrtcGetCUBINSize")
        LENSED_SYM(GetCUBIN, "nvrtcGetCUBIN")
        LENSED_SYM(GetLoweredName, "nvrtcGetLoweredName")
#undef LENSED_SYM
        n.ok = true;
    });
    return n;
}

struct Driver {
    PFN_cuModuleLoadData_v2000 ModuleLoadData = nullptr;
    PFN_cuModuleGetFunction_v2000 ModuleGetFunction = nullptr;
    PFN_cuModuleUnload_v2000 ModuleUnload = nullptr;
    PFN_cuFuncSetAttribute_v9000 FuncSetAttribute = nullptr;
    PFN_cuFuncGetAttribute_v2020 FuncGetAttribute = nullptr;
    PFN_cuLaunchKernel_v4000 LaunchKernel = nullptr;
    bool ok = false;
};

const Driver &driver()
{
    static Driver d;
    static std::once_flag once;
    std::call_once(once, [] {
        auto get = [](const char *name, void **fn) {
            cudaDriverEntryPointQueryResult qr;
            return cudaGetDriverEntryPoint(name, fn, cudaEnableDefault, &qr) == cudaSuccess && *fn &&
                   qr == cudaDriverEntryPointSuccess;
        };
        d.ok = get("cuModuleLoadData", (void **)&d.ModuleLoadData) && get("cuModuleGetFunction", (void **)&d.ModuleGetFunction) &&
               get("cuModuleUnload", (void **)&d.ModuleUnload) && get("cuFuncSetAttribute", (void **)&d.FuncSetAttribute) &&
               get("cuFuncGetAttribute", (void **)&d.FuncGetAttribute) && get("cuLaunchKernel", (void **)&d.LaunchKernel);
    });
    return d;
}

}  // namespace

// Immutable once jit_get has published it: clones of a handle launch it from several threads.
struct JitTracer {
    CUfunction fn = nullptr;
    int np = 0;
    size_t smem_max = 48 * 1024;      // dynamic shared memory a launch may ask for (set once, in jit_get)
};

namespace {
struct CacheEntry {
    JitTracer *tracer = nullptr;      // NULL: this signature failed in this process ...
    std::string why;                  // ... for this reason (reported to every later handle too)
};
std::mutex g_mutex;
std::map<std::string, CacheEntry> g_cache;       // key: device, counts, points per pass, blocks per SM
}  // namespace

// Which lists are specialised at run time: at most one shear (TraceSig), and few enough positioned
// components that the unrolled ray loop stays a sensible kernel; beyond that the interpreter.
bool jit_wanted(const int (&c)[K_COUNT])
{
    const char *env = getenv("LENSED_JIT");
    if (env && env[0] == '0') return false;
    const int n_lens = c[K_SHEAR] + c[K_SIE] + c[K_SIS] + c[K_POINT];
    const int n_pos = c[K_SRC_SERSIC] + c[K_SRC_GAUSS] + c[K_FG_SERSIC] + c[K_FG_GAUSS];
#ifdef LENSED_JIT_NO_LIMITS             // tuning builds: how far does the specialised template carry?
    return c[K_SHEAR] <= 1 && n_lens + n_pos >= 1;
#endif
    return c[K_SHEAR] <= 1 && c[K_SIE] <= 3 && n_lens <= 6 && n_pos >= 0 && n_pos <= 8 && n_lens + n_pos >= 1;
}

// NVRTC: the explicit instantiation of trace_static_kernel for these counts -> cubin and the
// kernel's lowered name; returns an empty string, or what went wrong.  Needs no device.
std::string jit_compile(const int (&c)[K_COUNT], int np, int minb, std::vector<char> *cubin, std::string *name)
{
    const Nvrtc &rt = nvrtc();
    if (!rt.ok) return "NVRTC (libnvrtc.so.12) not found";
    char expr[256];
    snprintf(expr, sizeof expr, "lensed::trace_static_kernel<%d, lensed::TraceSig<%d, %d, %d, %d, %d, %d, %d, %d>, %d>", np,
             c[K_SHEAR], c[K_SIE], c[K_SIS], c[K_POINT], c[K_SRC_SERSIC], c[K_SRC_GAUSS], c[K_FG_SERSIC], c[K_FG_GAUSS], minb);
    const std::string src = std::string("#include \"trace_static.cuh\"\ntemplate __global__ void ") + expr +
                            "(lensed::Program, lensed::TraceArgs);\n";
    void *prog = nullptr;
    if (rt.CreateProgram(&prog, src.c_str(), "lensed_jit.cu", kJitHeaderCount, kJitHeaderTexts, kJitHeaderNames) != 0)
        return "nvrtcCreateProgram failed";
    const char *opts[] = {"--gpu-architecture=sm_100a", "-std=c++17", "-lineinfo"};
    std::string msg;
    const char *lowered = nullptr;
    if (rt.AddNameExpression(prog, expr) != 0) msg = "nvrtcAddNameExpression failed";
    else if (rt.CompileProgram(prog, 3, opts) != 0) {
        size_t n = 0;
        rt.GetProgramLogSize(prog, &n);
        std::string log(n, '\0');
        if (n) rt.GetProgramLog(prog, &log[0]);
        msg = "nvrtcCompileProgram failed: " + log.substr(0, 600);
    } else {
        size_t n = 0;
        if (rt.GetCUBINSize(prog, &n) != 0 || n == 0) msg = "no cubin";
        else {
            cubin->resize(n);
            if (rt.GetCUBIN(prog, cubin->data()) != 0) msg = "nvrtcGetCUBIN failed";
            else if (rt.GetLoweredName(prog, expr, &lowered) != 0 || !lowered) msg = "nvrtcGetLoweredName failed";
            else *name = lowered;
        }
    }
    rt.DestroyProgram(&prog);
    return msg;
}

// The tracer for these per-kind counts with np rule points per pass on the current device: from the
// cache, else compiled now.  NULL (and a line in *why) when NVRTC or the driver entry points are
// missing or the compilation fails.
const JitTracer *jit_get(const int (&c)[K_COUNT], int np, int device, std::string *why)
{
    const int n_models = c[K_SHEAR] + c[K_SIE] + c[K_SIS] + c[K_POINT] + c[K_SRC_SERSIC] + c[K_SRC_GAUSS] + c[K_FG_SERSIC] + c[K_FG_GAUSS];
    const int minb = n_models <= 5 ? 3 : 2;      // resident blocks per SM: 80 or 128 registers (as the built-in signatures)
    char key[160];
    snprintf(key, sizeof key, "%d:%d,%d,%d,%d,%d,%d,%d,%d:%d:%d", device, c[K_SHEAR], c[K_SIE], c[K_SIS], c[K_POINT],
             c[K_SRC_SERSIC], c[K_SRC_GAUSS], c[K_FG_SERSIC], c[K_FG_GAUSS], np, minb);
    std::lock_guard<std::mutex> lock(g_mutex);
    auto it = g_cache.find(key);
    if (it != g_cache.end()) {
        if (!it->second.tracer && why) *why = it->second.why;
        return it->second.tracer;
    }
    auto fail = [&](const std::string &msg) -> const JitTracer * {
        if (why) *why = msg;
        g_cache[key] = CacheEntry{nullptr, msg};     // do not try again in this process; keep the reason
        return nullptr;
    };
    const Driver &drv = driver();
    if (!drv.ok) return fail("driver entry points not available");

    std::vector<char> cubin;
    std::string name;
    const std::string msg = jit_compile(c, np, minb, &cubin, &name);
    if (!msg.empty()) return fail(msg);

    if (cudaSetDevice(device) != cudaSuccess || cudaFree(nullptr) != cudaSuccess) return fail("no current context");
    CUmodule mod = nullptr;
    CUfunction fn = nullptr;
    if (drv.ModuleLoadData(&mod, cubin.data()) != CUDA_SUCCESS) return fail("cuModuleLoadData failed");
    if (drv.ModuleGetFunction(&fn, mod, name.c_str()) != CUDA_SUCCESS) {
        drv.ModuleUnload(mod);
        return fail("cuModuleGetFunction failed");
    }
    // the dynamic shared memory any launch may need, allowed once and here (under g_mutex): everything the
    // device lets a block opt in to beyond the kernel's own static arrays.  jit_launch only reads it.
    int optin = 0, fixed = 0;
    if (cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, device) != cudaSuccess ||
        drv.FuncGetAttribute(&fixed, CU_FUNC_ATTRIBUTE_SHARED_SIZE_BYTES, fn) != CUDA_SUCCESS || optin - fixed < 48 * 1024 ||
        drv.FuncSetAttribute(fn, CU_FUNC_ATTRIBUTE_MAX_DYNAMIC_SHARED_SIZE_BYTES, optin - fixed) != CUDA_SUCCESS) {
        drv.ModuleUnload(mod);
        return fail("cuFuncSetAttribute(max dynamic shared memory) failed");
    }
    JitTracer *t = new JitTracer;
    t->fn = fn;
    t->np = np;
    t->smem_max = (size_t)(optin - fixed);
    g_cache[key] = CacheEntry{t, std::string()};     // the module stays loaded for the life of the process
    return t;
}

// same launch as trace_block.cuh launch_trace_kernel, through the driver API
cudaError_t jit_launch(const JitTracer *t, const Program &prog, const TraceArgs &a0, int nvec, cudaStream_t st)
{
    const Driver &drv = driver();
    TraceArgs a = a0;
    a.quad = a0.quad_pp;
    a.nq_pad = a0.nq_pp;
    const size_t smem = trace_smem_bytes(prog, a.nq_pad);
    if (smem > t->smem_max) return cudaErrorInvalidValue;
    Program p = prog;
    void *params[2] = {&p, &a};
    const unsigned gx = (unsigned)((a.npix + a.pix_per_block - 1) / a.pix_per_block);
    const CUresult r = drv.LaunchKernel(t->fn, gx, (unsigned)nvec, 1, kJitThreads, 1, 1, (unsigned)smem, (CUstream)st, params, nullptr);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorLaunchFailure;
}

}  // namespace lensed
