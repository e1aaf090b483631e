"""Build libsph_b200.so (the C-ABI CUDA library, include/sph.h) in-tree with nvcc for sm_100a.

    python -m paper_2507_21684_b200.build [--force] [--verbose] [--bounds]

--bounds: debug build with -DSPH_BOUNDS (checked shared-memory indices in the tile kernels, sph_internal.cuh); it
replaces the library in place; the next plain build (or __graft_entry__.build()) notices and rebuilds the normal one.

nvcc cross-compiles without a GPU.  No --use_fast_math: the neighbour predicate and the position wrap
are fixed sequences of IEEE operations (readings R3/R4); fast approximations are used
explicitly (sqrt.approx / rcp.approx) only inside the pair sums.
"""
from __future__ import annotations
import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsph_b200.so")
STAMP = os.path.join(HERE, "_obj", "flavour.txt")     # "normal" or "bounds": what the library in place was built as


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _stale():
    if not os.path.exists(LIB):
        return True
    try:
        if open(STAMP).read().strip() != "normal":        # a --bounds debug library was left in place
            return True
    except OSError:
        return True
    t = os.path.getmtime(LIB)
    deps = sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(HERE, "..", "include", "sph.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, bounds: bool = False) -> str:
    if not force and not bounds and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    flags = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xcompiler", "-fPIC"]
    if verbose:
        flags = ["-Xptxas", "-v"] + flags
    if bounds:
        flags = flags + ["-DSPH_BOUNDS"]
    objdir = os.path.join(HERE, "_obj_bounds" if bounds else "_obj")
    os.makedirs(objdir, exist_ok=True)
    srcs = sources()
    objs = [os.path.join(objdir, os.path.basename(f)[:-3] + ".o") for f in srcs]

    def compile_one(pair):
        src, obj = pair
        return subprocess.run([nvcc] + flags + ["-c", src, "-o", obj], capture_output=True, text=True)

    # one nvcc per translation unit, in parallel (no device code crosses a file: no -rdc)
    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(max_workers=min(len(srcs), os.cpu_count() or 1)) as ex:
        results = list(ex.map(compile_one, zip(srcs, objs)))
    for r in results:
        if verbose or r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
        if r.returncode != 0:
            raise subprocess.CalledProcessError(r.returncode, r.args)
    subprocess.run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs, check=True)
    os.makedirs(os.path.dirname(STAMP), exist_ok=True)
    with open(STAMP, "w") as f:
        f.write("bounds\n" if bounds else "normal\n")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, bounds="--bounds" in sys.argv))
