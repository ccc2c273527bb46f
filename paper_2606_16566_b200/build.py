"""Builds paper_2606_16566_b200/libgs.so (the C-ABI library of include/gs.h) with nvcc for sm_100a.

Each translation unit gets its own floating-point flags:
  preprocess.cu   -fmad=false, IEEE div/sqrt, no fast-math  (bit-exact integers)
  render*.cu      -use_fast_math                            (PAPER.md:302 builds its kernels this way)
  binning.cu/api  integer / host code
The library is built IN-TREE so that it travels to the GPU box with the repository snapshot.
"""
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libgs.so")
LIB_DBG = os.path.join(HERE, "libgs_dbg.so")   # -DGS_DEBUG_BOUNDS: device-side checks of every workspace / output index
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-I", os.path.join(ROOT, "include")]
UNITS = {
    "api.cu": [],
    "preprocess.cu": ["-fmad=false", "-prec-div=true", "-prec-sqrt=true", "-ftz=false"],
    "binning.cu": [],
    "selftest.cu": [],
    "noalloc.cu": [],
    "render.cu": ["-use_fast_math"],
    "render_b200.cu": ["-use_fast_math"],
}
HEADERS = ["common.cuh", "render_common.cuh", "render_blend.cuh"]


def _nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: the CUDA extension cannot be built (there is no CPU fallback)")
    return exe


def _deps():
    d = [os.path.join(CSRC, h) for h in HEADERS] + [os.path.join(ROOT, "include", "gs.h"), os.path.abspath(__file__)]
    return d


def build(force: bool = False, verbose: bool = False, debug_bounds: bool = False) -> str:
    """Builds libgs.so (or, with debug_bounds, libgs_dbg.so: the same sources with -DGS_DEBUG_BOUNDS, objects in build/dbg)."""
    obj_dir = os.path.join(OBJ, "dbg") if debug_bounds else OBJ
    lib = LIB_DBG if debug_bounds else LIB
    extra = ["-DGS_DEBUG_BOUNDS"] if debug_bounds else []
    os.makedirs(obj_dir, exist_ok=True)
    nvcc = _nvcc()
    objs, rebuilt = [], False
    for src, flags in UNITS.items():
        flags = flags + extra
        s = os.path.join(CSRC, src)
        o = os.path.join(obj_dir, src.replace(".cu", ".o"))
        objs.append(o)
        newest = max(os.path.getmtime(x) for x in [s] + _deps())
        if force or not os.path.exists(o) or os.path.getmtime(o) < newest:
            cmd = [nvcc] + ARCH + COMMON + flags + (["-Xptxas", "-v"] if verbose else []) + ["-c", s, "-o", o]
            subprocess.run(cmd, check=True)
            rebuilt = True
    if rebuilt or not os.path.exists(lib):
        subprocess.run([nvcc] + ARCH + ["-shared", "-o", lib] + objs, check=True)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, debug_bounds="--debug-bounds" in sys.argv))
