"""Build csrc/*.cu into csrc/libgrinqh.so for sm_100a (in-tree, so the .so travels with gpurun).

Every .cu is compiled to an object file of its own, in parallel, then linked (the kernel templates take a minute each).
GQ_NVCC_EXTRA adds flags (e.g. -DGQ_TIMING for a build that prints per-phase clocks)."""
import glob
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(CSRC, "libgrinqh.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _deps():
    return glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(HERE, "..", "include", "grinqh.h")]


def _tag() -> str:
    return "_".join(e.strip("-") for e in os.environ.get("GQ_NVCC_EXTRA", "").split())


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    try:  # the library on disk was linked from objects built with other extra flags
        if open(LIB + ".tag").read() != _tag():
            return True
    except OSError:
        if _tag():
            return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in sources() + _deps())


def build(force: bool = False, verbose: bool = False) -> str:
    if not (force or needs_build()):
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    extra = os.environ.get("GQ_NVCC_EXTRA", "").split()
    tag = _tag()
    hdr_t = max(os.path.getmtime(d) for d in _deps())

    def compile_one(src):
        obj = os.path.join(OBJ, os.path.basename(src)[:-3] + (("." + tag) if tag else "") + ".o")
        if (not force) and os.path.exists(obj) and os.path.getmtime(obj) > max(os.path.getmtime(src), hdr_t):
            return obj
        cmd = [NVCC] + FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, src]
        subprocess.check_call(cmd)
        return obj

    with ThreadPoolExecutor(max_workers=8) as ex:
        objs = list(ex.map(compile_one, sources()))
    subprocess.check_call([NVCC, "--shared", "-cudart", "static", "-o", LIB] + objs)
    with open(LIB + ".tag", "w") as f:
        f.write(tag)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
