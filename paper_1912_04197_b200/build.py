"""Compile csrc/*.cu into paper_1912_04197_b200/libbh.so with nvcc for sm_100a (in-tree)."""
from __future__ import annotations

import glob
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
LIB = os.path.join(HERE, "libbh.so")
MICRO_LIB = os.path.join(HERE, "libbh_microbench.so")   # measurement-only kernels, loaded by bench.py alone
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "--fmad=true", "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


PER_FILE_FLAGS = {}    # extra nvcc flags of single translation units (none at present)


def sources():
    return sorted(glob.glob(os.path.join(HERE, "csrc", "*.cu")))


def micro_sources():
    return sorted(glob.glob(os.path.join(HERE, "csrc", "bench", "*.cu")))


def _deps():
    return sources() + micro_sources() + glob.glob(os.path.join(HERE, "csrc", "*.cuh")) + \
        glob.glob(os.path.join(ROOT, "include", "*.h"))


def build(force: bool = False, verbose: bool = False) -> str:
    deps = _deps()
    if not sources():
        raise FileNotFoundError('no CUDA sources under csrc/')
    if not force and all(os.path.exists(lib) and all(os.path.getmtime(lib) >= os.path.getmtime(d) for d in deps)
                         for lib in (LIB, MICRO_LIB)):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    flags = [f for f in NVCC_FLAGS if f != "-shared"] + (["-Xptxas", "-v"] if verbose else []) + \
        ["-I", os.path.join(ROOT, "include")]
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    # one nvcc per translation unit, all at once (no relocatable device code: kernels share nothing but headers)
    jobs = []
    for src in sources() + micro_sources():
        obj = os.path.join(objdir, os.path.basename(src)[:-3] + ".o")
        jobs.append((src, obj, subprocess.Popen([nvcc] + flags + PER_FILE_FLAGS.get(os.path.basename(src), []) +
                                                ["-c", "-o", obj, src])))
    if any(j.wait() != 0 for _, _, j in jobs):
        raise RuntimeError("nvcc failed")
    objs = {src: obj for src, obj, _ in jobs}
    link = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static", "-Xcompiler", "-fPIC"]
    subprocess.run(link + ["-o", LIB] + [objs[x] for x in sources()], check=True)
    subprocess.run(link + ["-o", MICRO_LIB] + [objs[x] for x in micro_sources()], check=True)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
