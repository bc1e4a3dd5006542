"""In-tree build of libvelo.so (the CUDA path + its C-ABI) with nvcc for sm_100a only.

The built library sits beside this file so that it travels with the repository snapshot; there
is no JIT cache and no other architecture.
"""
from __future__ import annotations

import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(_HERE), "include")
LIB = os.path.join(_HERE, "libvelo.so")
SOURCES = ["velo_api.cu", "velo_kernels.cu", "velo_sort.cu", "velo_track.cu", "velo_fit.cu", "velo_next.cu",
           "velo_scheduler.cu"]
HEADERS = ["velo_device.cuh", "velo_internal.h", "velo_pool.cuh"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "--expt-relaxed-constexpr", "-Xcompiler", "-fPIC"]
OBJ_DIR = os.path.join(_HERE, "build")


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.join(INCLUDE, "velo.h")]
    return any(os.path.getmtime(d) > t for d in deps)


LIB_TIMELINE = os.path.join(_HERE, "libvelo_timeline.so")


def _compile(lib: str, extra: list[str], tag: str, verbose: bool = False) -> str:
    """nvcc -c every source (in parallel: they are independent translation units), then link."""
    from concurrent.futures import ThreadPoolExecutor

    # objects and the linked library are private to this process until an atomic rename: several ranks
    # (torchrun) or forked test workers may find the library stale at the same moment
    obj_dir = os.path.join(OBJ_DIR, f"{tag}_{os.getpid()}")
    os.makedirs(obj_dir, exist_ok=True)
    objs = [os.path.join(obj_dir, f"{f[:-3]}.o") for f in SOURCES]

    def one(src, obj):
        cmd = [_nvcc(), *NVCC_FLAGS, *extra, "-I", INCLUDE, "-c", "-o", obj, os.path.join(CSRC, src)]
        if verbose:
            cmd[1:1] = ["-Xptxas", "-v"]
        subprocess.run(cmd, check=True)

    with ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 1)) as ex:
        list(ex.map(one, SOURCES, objs))
    tmp = f"{lib}.{os.getpid()}.tmp"
    subprocess.run([_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", tmp, *objs], check=True)
    os.replace(tmp, lib)
    shutil.rmtree(obj_dir, ignore_errors=True)
    return lib


def build_timeline() -> str:
    """The same library with -DVELO_TIMELINE: every pipeline kernel records the window in which its
    CTAs ran (GPU global timer), for `bench.py --timeline`. Never used by the product path."""
    return _compile(LIB_TIMELINE, ["-DVELO_TIMELINE"], "tl")


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile libvelo.so if missing or older than its sources. Returns its path."""
    if force or _stale():
        _compile(LIB, [], "velo", verbose)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
