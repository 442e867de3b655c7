"""Build the CUDA libraries (sm_100a) in-tree with nvcc.  `python -m paper_2311_18737_b200.build`.

libplspec.so        the product: the C ABI of include/plspec.h (no cuFFT, no cuBLAS); plspec_api.cu + plspec_static.cu
                    (the entry point that allocates nothing, with its file-scope device workspace)
libplspec_cufft.so  comparison point only (csrc/cufft_pipeline.cu: the paper's multiply -> cuFFT -> accumulate
                    structure); loaded by bench.py alone, never by the binding
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libplspec.so")
LIB_CUFFT = os.path.join(HERE, "libplspec_cufft.so")
SOURCES = ["plspec_api.cu", "plspec_static.cu"]
HEADERS = ["plspec_common.cuh", "plspec_kernels.cuh", "plspec_fused.cuh", os.path.join("..", "..", "include", "plspec.h")]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA library cannot be built (there is no CPU fallback)")


def _stale(lib: str, deps: list[str]) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(d) > t for d in deps + [os.path.abspath(__file__)])


def stale() -> bool:
    return _stale(LIB, [os.path.join(CSRC, s) for s in SOURCES + HEADERS])


def _run(lib: str, sources: list[str], extra: list[str], verbose: bool) -> str:
    tmp = lib + f".tmp{os.getpid()}"
    cmd = [_nvcc(), *NVCC_FLAGS, *os.environ.get("PLSPEC_NVCC_EXTRA", "").split(), *(["-Xptxas", "-v"] if verbose else []),
           "-o", tmp, *sources, *extra]
    subprocess.check_call(cmd)
    os.replace(tmp, lib)
    return lib


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not stale():
        return LIB
    return _run(LIB, [os.path.join(CSRC, s) for s in SOURCES], [], verbose)


def build_cufft_pipeline(force: bool = False, verbose: bool = False) -> str:
    """The comparison pipeline, linked against the toolkit's cuFFT (the same one on the GPU box's image)."""
    src = os.path.join(CSRC, "cufft_pipeline.cu")
    if not force and not _stale(LIB_CUFFT, [src]):
        return LIB_CUFFT
    libdir = os.path.join(os.path.dirname(os.path.dirname(os.path.realpath(_nvcc()))), "lib64")
    return _run(LIB_CUFFT, [src], ["-lcufft", f"-L{libdir}", "-Xlinker", f"-rpath={libdir}"], verbose)


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
    print(build_cufft_pipeline(force="--force" in sys.argv, verbose="-v" in sys.argv))
