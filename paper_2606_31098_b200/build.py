"""In-tree build of the CUDA C-ABI library for sm_100a (nvcc cross-compiles without a GPU)."""
import glob
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
# PILOT_REFINE_LIB: load another build of the same sources (kernel-tuning experiments); default = the in-tree library
LIB = os.environ.get("PILOT_REFINE_LIB") or os.path.join(CSRC, "libpilot_refine.so")
SOURCES = sorted(glob.glob(os.path.join(CSRC, "*.cu")))
HEADERS = [os.path.join(HERE, "..", "include", "pilot_refine.h")] + sorted(glob.glob(os.path.join(CSRC, "*.cuh")))
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC"]


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(f) > t for f in deps)


def build(force=False, verbose=False):
    """Compile every csrc/*.cu to an object (in parallel, only the stale ones) and link libpilot_refine.so."""
    if os.environ.get("PILOT_REFINE_LIB"):
        return LIB                      # an explicitly chosen build is used as it is
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    extra = ["-Xptxas", "-v"] if verbose else []
    objs, jobs = [], []
    for src in SOURCES:
        obj = src[:-3] + ".o"
        objs.append(obj)
        if force or _stale(obj, [src] + HEADERS):
            jobs.append([nvcc] + NVCC_FLAGS + extra + ["-c", "-o", obj, src])
    if jobs:
        with ThreadPoolExecutor(max_workers=len(jobs)) as ex:
            for r in ex.map(lambda c: subprocess.run(c, check=False), jobs):
                if r.returncode != 0:
                    raise subprocess.CalledProcessError(r.returncode, r.args)
    if jobs or _stale(LIB, objs):
        subprocess.run([nvcc, "-shared", "-o", LIB] + objs, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
