"""Build the C-ABI shared library (hand-written CUDA, sm_100a only) in-tree.

    python -m paper_1401_8060_b200.build [--force] [--checked | --microbench]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the
GPU box with the repo snapshot.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libstochtrack_b200.so")
MICRO = os.path.join(HERE, "st_microbench")
SOURCES = ["stochtrack_api.cu"]
HEADERS = ["st_kernels.cuh", "st_track.cuh", "st_ftmap.cuh", os.path.join("..", "..", "include", "stochtrack.h")]
# -ffp-contract=off: the host copy of the rasteriser arithmetic (st_track_params)
# must not be contracted into FMAs (G15); device code uses *_rn intrinsics.
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC,-ffp-contract=off"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps if os.path.exists(d))


LIB_CHECKED = os.path.join(HERE, "libstochtrack_b200_checked.so")


def build_checked(force=False):
    """The same library with -DST_CHECKED: device-side assertions on every index (for the GPU tests)."""
    srcs = [os.path.join(CSRC, s) for s in SOURCES]
    deps = srcs + [os.path.join(CSRC, h) for h in HEADERS]
    if force or _stale(LIB_CHECKED, deps):
        subprocess.check_call([_nvcc(), *NVCC_FLAGS, "-DST_CHECKED", "-shared", "-o", LIB_CHECKED, *srcs])
    return LIB_CHECKED


def build_microbench(force=False):
    """The issue-rate / gather-rate microbenchmarks behind profiles/microbench_*.md (not part of the library)."""
    micro_src = os.path.join(CSRC, "st_microbench.cu")
    if force or _stale(MICRO, [micro_src]):
        subprocess.check_call([_nvcc(), *NVCC_FLAGS, "-o", MICRO, micro_src])
    return MICRO


def build(force=False, verbose=False):
    """Compile libstochtrack_b200.so. Returns the .so path."""
    srcs = [os.path.join(CSRC, s) for s in SOURCES]
    deps = srcs + [os.path.join(CSRC, h) for h in HEADERS]
    if force or _stale(LIB, deps):
        cmd = [_nvcc(), *NVCC_FLAGS, "-shared", "-o", LIB, *srcs]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
            print(" ".join(cmd))
        subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    if "--checked" in sys.argv:
        print(build_checked(force="--force" in sys.argv))
    elif "--microbench" in sys.argv:
        print(build_microbench(force="--force" in sys.argv))
    else:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
