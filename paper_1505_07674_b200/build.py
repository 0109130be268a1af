"""Build step of the CUDA library: nvcc -> paper_1505_07674_b200/liblensed_b200.so (in-tree).

sm_100a only, -lineinfo so that ncu's source page maps to the .cu files.  Each .cu is
compiled to an object (in parallel) and linked into one shared library with the static CUDA
runtime, so the library has no dependency beyond the driver.  `python -m
paper_1505_07674_b200.build [--force] [--verbose]`.
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "liblensed_b200.so")
SOURCES = ("api.cu", "prep.cu", "trace.cu", "trace_sig_a.cu", "trace_sig_b.cu", "trace_sig_c.cu",
           "trace_sig_d.cu", "trace_sig_e.cu", "trace_sig_f.cu", "trace_sig_g.cu", "trace_sig_h.cu", "trace_sig_i.cu", "refine.cu", "deflect.cu", "nested.cu", "conv.cu",
           "peak.cu")
HEADERS = tuple(os.path.join(CSRC, f) for f in ("lensed_internal.h", "f32x2.cuh", "trace_math.cuh",
                                                  "trace_block.cuh", "trace_static.cuh")) + (
           os.path.join(os.path.dirname(HERE), "include", "lensed.h"),)
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False, defines=(), lib=LIB, objdir=None):
    """Compile what is out of date; returns the path of the shared library.  `defines`
    (e.g. ("LENSED_TRACE_MIN_BLOCKS=3",)), `lib` and `objdir` make a differently tuned build
    beside the default one (load it with LENSED_B200_LIB=<path>)."""
    nvcc = _nvcc()
    objdir = objdir or os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    extra = (["-Xptxas", "-v"] if verbose else []) + ["-D" + d for d in defines]
    jobs = []
    for src in SOURCES:
        s = os.path.join(CSRC, src)
        o = os.path.join(objdir, src[:-3] + ".o")
        if force or _stale(o, (s,) + HEADERS + (os.path.abspath(__file__),)):
            jobs.append([nvcc] + NVCC_FLAGS + extra + ["-c", s, "-o", o])

    def run(cmd):
        r = subprocess.run(cmd, capture_output=True, text=True)
        return cmd, r

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        for cmd, r in ex.map(run, jobs):
            if verbose or r.returncode != 0:
                sys.stderr.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
            if r.returncode != 0:
                raise RuntimeError("nvcc failed: " + " ".join(cmd))
    objs = [os.path.join(objdir, s[:-3] + ".o") for s in SOURCES]
    if force or jobs or _stale(lib, objs):
        cmd = [nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", lib] + objs
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError("link failed: " + " ".join(cmd))
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
