"""Build liblqcd.so in-tree with nvcc for sm_100a (no torch linkage; cudart is linked statically).

csrc/*.cu are independent translation units (lqcd.cu: host side, pack and BLAS-1 kernels; inst_*.cu: the dslash
kernel instantiations of one storage type x link format each); they are compiled in parallel and linked."""
from __future__ import annotations

import concurrent.futures
import glob
import os
import shlex
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
OBJ = os.path.join(_HERE, "build")
LIB = os.path.join(_HERE, "liblqcd.so")
HEADER = os.path.join(os.path.dirname(_HERE), "include", "lqcd.h")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC"]


def units():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def sources():
    return units() + sorted(glob.glob(os.path.join(CSRC, "*.cuh"))) + [HEADER, os.path.abspath(__file__)]


STAMP = LIB + ".flags"   # the flag string liblqcd.so was compiled with (git-ignored, travels with the library)


def wanted_flags() -> str:
    """What a build started now would pass to nvcc: the fixed flags plus $LQCD_NVCC_FLAGS (-D switches of a sweep)."""
    return " ".join(NVCC_FLAGS + shlex.split(os.environ.get("LQCD_NVCC_FLAGS", "")))


def built_flags():
    """The flags of the library on disk, or None if it was built before the stamp existed / is missing."""
    try:
        with open(STAMP) as f:
            return f.read().strip()
    except OSError:
        return None


def stale() -> bool:
    """Rebuild if the library is missing, older than a source, or was compiled with other flags than this process asks
    for -- a library left behind by a tuning sweep (-DLQCD_...=...) must not be picked up by a default test or bench run."""
    if not os.path.exists(LIB):
        return True
    if built_flags() != wanted_flags():
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(s) > t for s in sources())


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile every unit (extra flags, e.g. -D switches of a tuning sweep, from $LQCD_NVCC_FLAGS) and link."""
    if not (force or stale()):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    extra = shlex.split(os.environ.get("LQCD_NVCC_FLAGS", ""))
    os.makedirs(OBJ, exist_ok=True)
    tag = os.getpid()

    def compile_unit(src):
        obj = os.path.join(OBJ, f"{os.path.splitext(os.path.basename(src))[0]}.{tag}.o")
        cmd = [nvcc, *NVCC_FLAGS, *extra, *(["-Xptxas=-v"] if verbose else []), "-c", src, "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src}:\n{r.stderr[-4000:]}")
        return obj, r.stderr

    objs = []
    try:
        with concurrent.futures.ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as pool:
            for obj, log in pool.map(compile_unit, units()):
                objs.append(obj)
                if verbose:
                    print(log)
        tmp = LIB + f".tmp{tag}"
        subprocess.check_call([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp, *objs])
        os.replace(tmp, LIB)
        with open(STAMP + f".tmp{tag}", "w") as f:
            f.write(" ".join(NVCC_FLAGS + extra) + "\n")
        os.replace(STAMP + f".tmp{tag}", STAMP)
    finally:
        for o in glob.glob(os.path.join(OBJ, f"*.{tag}.o")):
            os.remove(o)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
