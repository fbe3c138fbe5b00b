"""Build paper_2510_07764_b200/libppm_b200.so (the C-ABI library of include/ppm.h) in-tree with nvcc
for sm_100a.  `python -m paper_2510_07764_b200._build` or `_build.build()`; rebuilt only when a source
is newer than the library.  nvcc cross-compiles without a GPU.  The translation units (ppm.cu and the
cell-kernel launchers launch_*.cu) are compiled in parallel and linked into one shared library."""
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
              "-Xcompiler", "-fPIC"]
LINK_FLAGS = ["-shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a"]


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
    nvcc = nvcc_path()
    units = sorted(glob.glob(os.path.join(CSRC, "*.cu")))
    objdir = os.path.join(_HERE, "build", "bounds" if BOUNDS else "obj")
    os.makedirs(objdir, exist_ok=True)
    common = NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + (["-DPPM_BOUNDS"] if BOUNDS else []) + \
             ["-I", os.path.join(ROOT, "include"), "-I", CSRC]
    procs = []
    for u in units:
        obj = os.path.join(objdir, os.path.basename(u)[:-3] + ".o")
        logf = open(obj + ".log", "w+")                      # a file, not a pipe: no unit ever blocks on a full pipe
        procs.append((logf, obj, subprocess.Popen([nvcc] + common + ["-c", "-o", obj, u], stdout=logf, stderr=subprocess.STDOUT)))
    log, failed = "", False
    for logf, obj, pr in procs:
        pr.wait()
        logf.seek(0)
        log += logf.read()
        logf.close()
        failed = failed or pr.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed:\n" + log)
    res = subprocess.run([nvcc] + LINK_FLAGS + ["-o", LIB + ".tmp"] + [obj for _, obj, _ in procs],
                         capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("nvcc link failed:\n" + res.stdout + res.stderr)
    if verbose:
        print(log)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
