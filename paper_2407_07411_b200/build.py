"""Compile the C-ABI library (csrc/ -> paper_2407_07411_b200/libhpsi.so) for sm_100a with nvcc, and the separate
calibration probe library libhpsi_bench.so (csrc/bench/, include/hpsi_bench.h) that only bench.py loads.

In-tree build: the .so files are git-ignored but travel to the GPU box with the repo snapshot.  nvcc cross-compiles
without a GPU.  ``python -m paper_2407_07411_b200.build`` forces a rebuild (``-v`` adds -Xptxas -v).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libhpsi.so")
BENCH_LIB = os.path.join(HERE, "libhpsi_bench.so")
SOURCES = ["planner.cpp", "interp.cpp", "kernels.cu", "kernels_paired.cu", "kernels_fused.cu", "api.cu", "stream.cu",
           "davidson.cu", "rotate.cu", "svd.cu"]
HEADERS = ["plan.h", "plan_dev.h", "kernels.cuh", "kernels_common.cuh", os.path.join("..", "..", "include", "hpsi.h")]
BENCH_SOURCES = [os.path.join("bench", "fp64_pipe.cu")]
BENCH_HEADERS = [os.path.join("..", "..", "include", "hpsi_bench.h")]
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def _stale(lib, deps) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in deps)


def _compile_and_link(lib, sources, verbose):
    build_dir = os.path.join(HERE, "build")
    os.makedirs(build_dir, exist_ok=True)
    common = ARCH + ["-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC", "-Xcompiler", "-Wall"]
    if verbose:
        common += ["-Xptxas", "-v"]
    objs, procs = [], []
    for src in sources:
        obj = os.path.join(build_dir, os.path.splitext(os.path.basename(src))[0] + ".o")
        objs.append(obj)
        cmd = [_nvcc()] + common + ["-x", "cu", "-c", os.path.join(CSRC, src), "-o", obj]
        procs.append((cmd, subprocess.Popen(cmd)))
    for cmd, pr in procs:
        if pr.wait() != 0:
            raise RuntimeError("compile failed: " + " ".join(cmd))
    subprocess.check_call([_nvcc(), "-shared"] + ARCH + ["-cudart", "static", "-o", lib] + objs)
    return lib


def build(force: bool = False, verbose: bool = False) -> str:
    """The product library."""
    if not force and not _stale(LIB, SOURCES + HEADERS):
        return LIB
    return _compile_and_link(LIB, SOURCES, verbose)


def build_bench(force: bool = False, verbose: bool = False) -> str:
    """The calibration probes (bench.py only)."""
    if not force and not _stale(BENCH_LIB, BENCH_SOURCES + BENCH_HEADERS):
        return BENCH_LIB
    return _compile_and_link(BENCH_LIB, BENCH_SOURCES, verbose)


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
    print(build_bench(force=True, verbose="-v" in sys.argv))
