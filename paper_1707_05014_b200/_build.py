"""Build libpct.so in-tree with nvcc for sm_100a (no torch involved: the library links cudart only)."""
import hashlib
import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libpct.so")
_STAMP = LIB + ".stamp"
SOURCES = ["pct_api.cu", "pct_kernels.cu", "pct_exact.cu", "pct_tvs.cu", "pct_peaks.cu", "pct_noalloc.cu"]
HEADERS = ["pct_rule.cuh", "pct_walk.cuh", "pct_walk16.cuh", "pct_internal.h", os.path.join("..", "..", "include", "pct.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    # the voxel-index rule is written with explicit rounding intrinsics; -fmad=false additionally
    # keeps nvcc from contracting anything else (BASELINE.json north_star: "compiled without FMA
    # contraction for the index math"); IEEE division and square root are nvcc's defaults
    "-fmad=false", "-prec-div=true", "-prec-sqrt=true", "-ftz=false",
    "-Xcompiler", "-fPIC,-O2,-ffp-contract=off,-fno-fast-math",
    "-shared", "-cudart", "static",
]


def nvcc_path():
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA extension cannot be built (there is no CPU fallback)")


def _tag():
    h = hashlib.sha256(" ".join(NVCC_FLAGS).encode())
    for f in SOURCES + HEADERS:
        with open(os.path.join(CSRC, f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def build(force=False, verbose=False):
    """Compile csrc/*.cu -> paper_1707_05014_b200/libpct.so (rebuilt when sources or flags change)."""
    if os.environ.get("PCT_LIB"):  # a prebuilt library (a checking or profiling build of the same sources)
        return os.environ["PCT_LIB"]
    tag = _tag()
    if not force and os.path.exists(LIB) and os.path.exists(_STAMP):
        with open(_STAMP) as f:
            if f.read().strip() == tag:
                return LIB
    tmp = LIB + ".tmp%d" % os.getpid()
    cmd = [nvcc_path(), *NVCC_FLAGS, "-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed:\n%s\n%s" % (" ".join(cmd), res.stderr))
    if verbose:
        print(res.stderr)
    os.replace(tmp, LIB)
    with open(_STAMP, "w") as f:
        f.write(tag)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
