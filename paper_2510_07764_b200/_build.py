"""Build paper_2510_07764_b200/libppm_b200.so (the C-ABI library of include/ppm.h) in-tree with nvcc
for sm_100a.  `python -m paper_2510_07764_b200._build` or `_build.build()`; rebuilt only when a source
is newer than the library.  nvcc cross-compiles without a GPU."""
import glob
import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(_HERE)
CSRC = os.path.join(_HERE, "csrc")
# PPM_BOUNDS=1 in the environment selects the debug build (-DPPM_BOUNDS: every shared-memory access of the table cell
# kernel is checked against the block's allocation and traps outside it); it lives beside the product library.
BOUNDS = os.environ.get("PPM_BOUNDS", "") not in ("", "0")
LIB = os.path.join(_HERE, "libppm_b200_bounds.so" if BOUNDS else "libppm_b200.so")
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cuh")) +
                  [os.path.join(ROOT, "include", "ppm.h")])


def nvcc_path():
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: cannot build libppm_b200.so (there is no CPU fallback)")


def build(force: bool = False, verbose: bool = False) -> str:
    srcs = sources()
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= max(os.path.getmtime(s) for s in srcs):
        return LIB
    cmd = [nvcc_path()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + (["-DPPM_BOUNDS"] if BOUNDS else []) + \
          ["-I", os.path.join(ROOT, "include"), "-I", CSRC, "-o", LIB + ".tmp", os.path.join(CSRC, "ppm.cu")]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + res.stdout + res.stderr)
    if verbose:
        print(res.stderr)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
