"""Build the C-ABI shared library (hand-written CUDA, sm_100a only) in-tree.

    python -m paper_1401_8060_b200.build [--force] [--checked | --microbench | --sass-summary | --ablate 1|2]

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


def build_ablate(which, force=False):
    """Measurement builds of the Chebyshev kernel (-DST_ABLATE=1: phase B alone, 2: phase A alone; st_kernels.cuh).
    Their results are meaningless; only `bench.py --lib <path>` loads them (profiles/r03_ablation.md)."""
    which = int(which)
    if which not in (1, 2):
        raise ValueError("--ablate takes 1 (phase B alone) or 2 (phase A alone)")
    out = os.path.join(HERE, f"libstochtrack_b200_ablate{which}.so")
    srcs = [os.path.join(CSRC, s) for s in SOURCES]
    deps = srcs + [os.path.join(CSRC, h) for h in HEADERS]
    if force or _stale(out, deps):
        subprocess.check_call([_nvcc(), *NVCC_FLAGS, f"-DST_ABLATE={which}", "-shared", "-o", out, *srcs])
    return out


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


def sass_summary(lib=None):
    """Markdown table of what the assembler made of every kernel in the built library: registers, local (spill)
    bytes and the counts of the sm_100 instructions the design leans on (packed FP32 FFMA2 / FADD2, warp REDUX,
    the float64 atomic of the template counter, float64 MUFU seeds), from `cuobjdump -res-usage` and `-sass`."""
    import collections
    import re
    lib = lib or build()
    cuobjdump = os.path.join(os.path.dirname(_nvcc()), "cuobjdump") if os.path.isabs(_nvcc()) else "cuobjdump"
    res = subprocess.run([cuobjdump, "-res-usage", lib], capture_output=True, text=True, check=True).stdout
    usage, cur = {}, None
    for line in res.splitlines():
        m = re.search(r"Function (\S+):", line)
        if m:
            cur = m.group(1)
            continue
        m = re.search(r"REG:(\d+).*?SHARED:(\d+).*?LOCAL:(\d+)", line)
        if m and cur:
            usage[cur], cur = tuple(int(x) for x in m.groups()), None
    pat = collections.OrderedDict([
        ("FFMA2", r"\bFFMA2\b"), ("FADD2", r"\bFADD2\b"), ("FFMA", r"\bFFMA\b"), ("REDUX", r"\bC?REDUX\b"),
        ("ATOMG.ADD.F64", r"ATOMG\.E\.ADD\.F64"), ("MUFU.*64H", r"MUFU\.\w+64H"), ("DFMA", r"\bDFMA\b"), ("LDS", r"\bLDS\b"),
        ("SHFL", r"\bSHFL\b"), ("instructions", r"^\s+/\*[0-9a-f]{4}\*/")])
    sass = subprocess.run([cuobjdump, "-sass", lib], capture_output=True, text=True, check=True).stdout
    counts, cur = collections.OrderedDict(), None
    for line in sass.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            cur = m.group(1)
            counts[cur] = collections.Counter()
            continue
        if cur is not None:
            for k, rx in pat.items():
                if re.search(rx, line):
                    counts[cur][k] += 1
    filt = os.path.join(os.path.dirname(cuobjdump), "cu++filt") if os.path.isabs(cuobjdump) else "cu++filt"
    names = subprocess.run([filt] + list(counts), capture_output=True, text=True, check=True).stdout.splitlines()
    rows, total = [], collections.Counter()
    for sym, name in zip(counts, names):
        name = re.sub(r"\((bool|int)\)", "", re.sub(r"^void ", "", name))         # <(bool)1, (int)2> -> <1, 2>
        name = re.sub(r"\(.*$", "", name).replace("st::", "")
        rows.append((name, usage.get(sym, (0, 0, 0)), counts[sym]))
        total.update(counts[sym])
    out = ["| kernel build | registers | local (spill) B | " + " | ".join(pat) + " |", "|---|---|---|" + "---|" * len(pat)]
    for name, u, c in sorted(rows):
        out.append(f"| `{name}` | {u[0]} | {u[2]} | " + " | ".join(str(c[k]) for k in pat) + " |")
    out.append(f"| **all {len(rows)} kernel builds** | | | " + " | ".join(str(total[k]) for k in pat) + " |")
    return "\n".join(out)


if __name__ == "__main__":
    if "--sass-summary" in sys.argv:
        print(sass_summary())
    elif "--ablate" in sys.argv:
        print(build_ablate(sys.argv[sys.argv.index("--ablate") + 1], force="--force" in sys.argv))
    elif "--checked" in sys.argv:
        print(build_checked(force="--force" in sys.argv))
    elif "--microbench" in sys.argv:
        print(build_microbench(force="--force" in sys.argv))
    else:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
