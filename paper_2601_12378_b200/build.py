"""Build libptefit.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libptefit.so")
SOURCES = ["ptefit.cu"]
DEPS = ["common.cuh", "fit_kernels.cuh", "search_kernels.cuh", "solve_kernels.cuh", "fused_solve.cuh", "tc_gemm.cuh", "tc_kernels.cuh", "tc_solve.cuh", "search_lean.cuh", "dmma_gemm.cuh", "dmma_kernels.cuh", "dm_host.inc", "tc_host.inc", "launch.inc", "ptefit.cu",
        os.path.join("..", "..", "include", "ptefit.h")]
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
         "-Xcompiler", "-fPIC", "-shared", "--use_fast_math=false"]


def _stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in DEPS if os.path.exists(os.path.join(CSRC, d)))


def build(force=False, verbose=False, tuning=False):
    """tuning=True adds -DPTEFIT_TUNING: in-kernel phase timers that print per-phase cycle counts (never
    the build that is measured or shipped)."""
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    flags = [f for f in FLAGS if not f.startswith("--use_fast_math")] + (["-DPTEFIT_TUNING"] if tuning else [])
    cmd = [nvcc] + flags + (["-Xptxas", "-v"] if verbose else []) + [os.path.join(CSRC, s) for s in SOURCES] + ["-o", LIB]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + r.stdout + r.stderr)
    if verbose:
        print(r.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, tuning="--tuning" in sys.argv))
