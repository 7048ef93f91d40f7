"""Build libmg.so (the C-ABI CUDA library of include/mg.h) in-tree with nvcc for sm_100a.

    python -m paper_2412_20522_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  Each .cu is compiled to an object under csrc/build/ (in parallel,
only when stale), then linked.  The .so is git-ignored but travels to the GPU box with gpurun.
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "libmg.so")
# The test build: the same objects, except that binsort.cu is compiled with -DMG_TESTING, which adds the failure-injection
# hook mg_debug_set_lookback_spin_limit (include/mg.h).  Only tests load it; the product binding loads libmg.so.
LIB_TESTING = os.path.join(HERE, "libmg_testing.so")
TESTING_SOURCES = ["binsort.cu"]
SOURCES = ["api.cu", "preprocess.cu", "binsort.cu", "render_fwd.cu", "render_bwd.cu", "preprocess_bwd.cu", "maskhead.cu", "renderloss.cu", "optimizer.cu", "peak.cu"]
HEADERS = ["mg_common.cuh", "render_common.cuh"]


def _deps():
    return [os.path.join(CSRC, f) for f in HEADERS] + [os.path.join(ROOT, "include", "mg.h"), os.path.abspath(__file__)]


def _compile(src: str, force: bool, verbose: bool, testing: bool = False) -> str:
    obj = os.path.join(OBJ, src[:-3] + ("_testing.o" if testing else ".o"))
    path = os.path.join(CSRC, src)
    if not force and os.path.exists(obj):
        t = os.path.getmtime(obj)
        if all(os.path.getmtime(d) <= t for d in [path] + _deps()):
            return obj
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
           "-Xcompiler", "-fPIC", "-I", os.path.join(ROOT, "include"), "-I", CSRC, "-c", path, "-o", obj]
    if testing:
        cmd.insert(1, "-DMG_TESTING")
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    subprocess.check_call(cmd)
    return obj


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    jobs = [(s, False) for s in SOURCES] + [(s, True) for s in TESTING_SOURCES]
    with ThreadPoolExecutor(max_workers=len(jobs)) as ex:
        built = list(ex.map(lambda j: _compile(j[0], force, verbose, j[1]), jobs))
    objs = built[:len(SOURCES)]
    swap = dict(zip(TESTING_SOURCES, built[len(SOURCES):]))
    objs_testing = [swap.get(s, o) for s, o in zip(SOURCES, objs)]
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    for lib, os_ in ((LIB, objs), (LIB_TESTING, objs_testing)):
        if force or not os.path.exists(lib) or any(os.path.getmtime(o) > os.path.getmtime(lib) for o in os_):
            subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", lib] + os_)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
