"""In-tree build of libcomb.so (C ABI of include/comb.h) with nvcc for sm_100a.

    python paper_2602_01519_b200/build.py [--force] [-v]      (run as a file: importing the package needs the library)
    python paper_2602_01519_b200/build.py --trace[=1]         (libcomb_trace.so: the same sources with -DCOMB_TRACE, the
                                                               prefill timeline stamps of prefill_timeline.py; a
                                                               profiling aid, never loaded by the package by default)

One nvcc invocation per .cu (in parallel), then one link step.  cudart is linked statically and libcuda is
reached through cudaGetDriverEntryPoint, so the library loads on a machine without a GPU driver (the
"-m 'not gpu'" tests check that it loads and exports every symbol of comb.h).
"""
from __future__ import annotations

import concurrent.futures as cf
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libcomb.so")
LIB_TRACE = os.path.join(HERE, "libcomb_trace.so")
SOURCES = ["comb_host.cu", "store_kernel.cu", "decode_kernel.cu", "prefill_kernel.cu", "cascade_kernel.cu", "gemm_kernel.cu", "fp8_kernel.cu"]
HEADERS = [os.path.join(CSRC, "kernels.h"), os.path.join(CSRC, "ptx.cuh"), os.path.join(CSRC, "attn_core.cuh"),
           os.path.join(os.path.dirname(HERE), "include", "comb.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden", "--expt-relaxed-constexpr",
              "-DCOMB_BUILD"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _stale(target: str, deps) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def _compile(src: str, verbose: bool, obj_dir: str = OBJ, extra=()) -> str:
    obj = os.path.join(obj_dir, os.path.splitext(src)[0] + ".o")
    path = os.path.join(CSRC, src)
    if _stale(obj, [path] + HEADERS):
        cmd = [_nvcc()] + NVCC_FLAGS + list(extra) + (["-Xptxas", "-v"] if verbose else []) + ["-c", path, "-o", obj]
        p = subprocess.run(cmd, capture_output=True, text=True)
        if p.returncode != 0:
            raise RuntimeError("nvcc failed for %s:\n%s\n%s" % (src, p.stdout, p.stderr))
        if verbose:
            sys.stderr.write(p.stderr)
    return obj


def build(force: bool = False, verbose: bool = False, trace: int = 0) -> str:
    """trace: 0 = the product library; 2 = libcomb_trace.so (all stamps); 1 = libcomb_trace1.so (softmax stamps only)."""
    obj_dir, lib, extra = OBJ, LIB, []
    if trace:
        obj_dir, extra = OBJ + "_trace%d" % trace, ["-DCOMB_TRACE=%d" % trace]
        lib = LIB_TRACE if trace >= 2 else LIB_TRACE.replace("_trace", "_trace1")
    os.makedirs(obj_dir, exist_ok=True)
    if force:
        for f in os.listdir(obj_dir):
            os.remove(os.path.join(obj_dir, f))
        if os.path.exists(lib):
            os.remove(lib)
    with cf.ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        objs = list(ex.map(lambda s: _compile(s, verbose, obj_dir, extra), SOURCES))
    if _stale(lib, objs):
        cmd = [_nvcc(), "-shared", "-o", lib] + objs + ["-cudart", "static", "-Xlinker", "--no-undefined", "-ldl",
                                                        "-lpthread", "-lrt"]
        p = subprocess.run(cmd, capture_output=True, text=True)
        if p.returncode != 0:
            raise RuntimeError("link failed:\n%s\n%s" % (p.stdout, p.stderr))
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, trace=1 if "--trace=1" in sys.argv else 2 if "--trace" in sys.argv else 0))
