"""Build libsfft_b200.so in-tree with nvcc for sm_100a (no torch extension machinery needed:
the library has a plain C ABI and links only the CUDA runtime)."""
import glob
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsfft_b200.so")
BENCH_LIB = os.path.join(HERE, "libsfft_bench.so")      # measurement probes for bench.py only (csrc/bench/)
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
         "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _headers():
    return (glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(CSRC, "*.cuh")) +
            [os.path.join(HERE, "..", "include", "sfft.h")])


def _stale(lib=None, srcs=None):
    lib = LIB if lib is None else lib
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = (sources() if srcs is None else srcs) + _headers()
    return any(os.path.getmtime(d) > t for d in deps)


def build_library(force=False, verbose=False):
    """Compile every .cu under csrc/ into libsfft_b200.so.  Returns the library path."""
    if not force and not _stale():
        return LIB
    objs, procs = [], []
    os.makedirs(os.path.join(HERE, "build"), exist_ok=True)
    for src in sources():
        obj = os.path.join(HERE, "build", os.path.basename(src) + ".o")
        objs.append(obj)
        cmd = [NVCC] + [f for f in FLAGS if f != "-shared"] + (["-Xptxas", "-v"] if verbose else []) + ["-c", src, "-o", obj]
        procs.append((cmd, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    for cmd, pr in procs:
        out, _ = pr.communicate()
        if verbose or pr.returncode != 0:
            print(out)
        if pr.returncode != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    subprocess.run([NVCC, "-shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs,
                   check=True)
    return LIB


def build_bench_library(force=False):
    """Compile csrc/bench/*.cu into libsfft_bench.so (FP64 peak probes and flop counters for bench.py)."""
    srcs = sorted(glob.glob(os.path.join(CSRC, "bench", "*.cu")))
    if not force and not _stale(BENCH_LIB, srcs + glob.glob(os.path.join(CSRC, "bench", "*.h"))):
        return BENCH_LIB
    subprocess.run([NVCC] + FLAGS + srcs + ["-o", BENCH_LIB], check=True)
    return BENCH_LIB


if __name__ == "__main__":
    import sys
    print(build_library(force=True, verbose="-v" in sys.argv))
    print(build_bench_library(force=True))
