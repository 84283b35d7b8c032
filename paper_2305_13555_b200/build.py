"""Compile the CUDA sources for sm_100a, in-tree:

    csrc/*.cu          -> liboci_b200.so    the C-ABI library of include/oci.h (the product)
    csrc/probe/*.cu    -> liboci_probe.so   measurement probe (fp64 tensor-pipe issue rate; bench.py's roofline
                                            denominator), deliberately NOT part of the product ABI

    python -m paper_2305_13555_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  Every .cu is compiled to an object of its own (in parallel, only when
stale), then linked.  The .so files and objects are git-ignored but travel to the GPU box with gpurun.
"""
import glob
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "liboci_b200.so")
PROBE_LIB = os.path.join(HERE, "liboci_probe.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "-fmad=true",
]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def probe_sources():
    return sorted(glob.glob(os.path.join(CSRC, "probe", "*.cu")))


def _headers():
    return glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(CSRC, "*.cuh")) + \
        [os.path.join(ROOT, "include", "oci.h"), os.path.abspath(__file__)]


def _newer(deps, target):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def _compile(src, obj, verbose):
    nvcc = os.environ.get("NVCC", "nvcc")
    cmd = [nvcc] + NVCC_FLAGS + ["-I", os.path.join(ROOT, "include"), "-I", CSRC, "-c", src, "-o", obj]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += os.environ.get("OCI_NVCC_EXTRA", "").split()
    subprocess.check_call(cmd)


def _link(objs, lib):
    nvcc = os.environ.get("NVCC", "nvcc")
    subprocess.check_call([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", lib] + objs)


def _build_lib(srcs, lib, tag, force, verbose):
    os.makedirs(OBJ, exist_ok=True)
    hdrs = _headers()
    objs, jobs = [], []
    for src in srcs:
        obj = os.path.join(OBJ, tag + "_" + os.path.basename(src)[:-3] + ".o")
        objs.append(obj)
        if force or _newer([src] + hdrs, obj):
            jobs.append((src, obj))
    if jobs:
        with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as ex:
            list(ex.map(lambda so: _compile(so[0], so[1], verbose), jobs))
    if jobs or _newer(objs, lib):
        _link(objs, lib)
    return lib


def build(force: bool = False, verbose: bool = False) -> str:
    _build_lib(probe_sources(), PROBE_LIB, "probe", force, verbose)
    return _build_lib(sources(), LIB, "oci", force, verbose)


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
