"""Build libmhd_b200.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2402_05478_b200.build [--force] [-v]

nvcc cross-compiles without a GPU; the .so is git-ignored but travels to the GPU box with the tree.
Each translation unit is compiled to an object under build/ (in parallel, only when stale), then linked.
"""
from __future__ import annotations

import hashlib
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libmhd_b200.so")
OBJDIR = os.path.join(HERE, "build")
SOURCES = ["fft_kernels.cu", "xfused_kernel.cu", "planefft_kernel.cu", "mhd_kernels.cu", "peaks_kernel.cu",
           "mhd_api.cu", "fft_c2r_static.cu"]
HEADERS = ["fft_core.cuh", "xteam.cuh", "bulk_copy.cuh", "mhd_internal.h"]

NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "--compiler-options", "-fPIC", "-cudart", "static"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _extra() -> list:
    return os.environ.get("MHD_NVCC_EXTRA", "").split()     # tuning experiments, e.g. -DMHD_XF_THREADS=320


def _sources() -> list:
    return [f for f in SOURCES if os.path.exists(os.path.join(CSRC, f))]


def _deps(src: str) -> list:
    return [os.path.join(CSRC, src)] + [os.path.join(CSRC, h) for h in HEADERS] + [os.path.join(INCLUDE, "mhd.h")]


def _obj(src: str) -> str:
    tag = hashlib.sha1(" ".join(NVCC_FLAGS + _extra()).encode()).hexdigest()[:8]     # objects built with other flags are stale
    return os.path.join(OBJDIR, f"{os.path.splitext(src)[0]}.{tag}.o")


def _stale(target: str, deps: list) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def _flag_stamp() -> str:
    return os.path.join(OBJDIR, "flags.txt")


def is_stale() -> bool:
    """the library is older than a source, or was built with other flags (objects need not exist: they do not travel)"""
    deps = sorted({d for s in _sources() for d in _deps(s)})
    if _stale(LIB, deps):
        return True
    if _extra():
        try:
            return open(_flag_stamp()).read() != " ".join(_extra())
        except OSError:
            return True
    return os.path.exists(_flag_stamp()) and open(_flag_stamp()).read() != ""


def _compile(src: str, verbose: bool) -> None:
    cmd = [_nvcc()] + NVCC_FLAGS + _extra() + (["-Xptxas", "-v"] if verbose else []) + \
          ["-I", INCLUDE, "-c", "-o", _obj(src), os.path.join(CSRC, src)]
    subprocess.run(cmd, check=True)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not is_stale():
        return LIB
    os.makedirs(OBJDIR, exist_ok=True)
    todo = [s for s in _sources() if force or _stale(_obj(s), _deps(s))]
    if todo:
        with ThreadPoolExecutor(max_workers=min(len(todo), os.cpu_count() or 1)) as ex:
            list(ex.map(lambda s: _compile(s, verbose), todo))
    objs = [_obj(s) for s in _sources()]
    subprocess.run([_nvcc(), "-shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs, check=True)
    with open(_flag_stamp(), "w") as f:
        f.write(" ".join(_extra()))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
