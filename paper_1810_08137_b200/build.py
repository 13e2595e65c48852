"""Build libugks.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1810_08137_b200.build [--force] [--verbose] [--developer]

--developer compiles with -DUGKS_DEVELOPER: the library then honours the UGKS_* environment overrides used for experiments and
SASS dumps (see csrc/ugks_jit.cu).  The default build reads no environment variable.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libugks.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "--use_fast_math=false"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _deps():
    return sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(HERE, "..", "include", "ugks.h")]


def build(force: bool = False, verbose: bool = False, developer: bool = False) -> str:
    stale = force or not os.path.exists(SO) or any(os.path.getmtime(s) > os.path.getmtime(SO) for s in _deps())
    if not stale:
        return SO
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    flags = [f for f in NVCC_FLAGS if not f.startswith("--use_fast_math")]
    if verbose:
        flags += ["-Xptxas", "-v"]
    if developer:
        flags += ["-DUGKS_DEVELOPER"]
    tmp = SO + f".tmp{os.getpid()}"
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    hdrs = [d for d in _deps() if not d.endswith(".cu")]

    def compile_one(src):                      # one translation unit -> build/<name>.o, skipped when up to date
        obj = os.path.join(objdir, os.path.basename(src)[:-3] + ".o")
        if not force and os.path.exists(obj) and all(os.path.getmtime(d) <= os.path.getmtime(obj) for d in [src, *hdrs]):
            return obj
        subprocess.run([nvcc, *flags, "-c", "-o", obj, src], check=True, cwd=CSRC)
        return obj

    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(max_workers=max(1, min(len(sources()), os.cpu_count() or 1))) as ex:
        objs = list(ex.map(compile_one, sources()))
    cuda_lib = os.path.join(os.path.dirname(os.path.dirname(os.path.realpath(nvcc))), "lib64")
    # NVRTC compiles the two f-sized kernels at ugks_init (csrc/ugks_jit.cu); libnvrtc is found through the rpath
    link = ["-L" + cuda_lib, "-lnvrtc", "-ldl", "-Xlinker", "-rpath", "-Xlinker", cuda_lib]
    subprocess.run([nvcc, *[f for f in flags if f not in ("-lineinfo",)], "-shared", "-o", tmp, *objs, *link], check=True, cwd=CSRC)
    os.replace(tmp, SO)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv or "--developer" in sys.argv, verbose="--verbose" in sys.argv, developer="--developer" in sys.argv))
