"""In-tree build of libvx.so (the C-ABI CUDA library) for sm_100a with nvcc."""
from __future__ import annotations

import os
import shutil
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libvx.so")
SOURCES = ["vx_api.cu", "vx_stage1.cu", "vx_stage2.cu", "vx_egress.cu", "vx_probe.cu", "vx_noalloc.cu"]
HEADERS = ["vx_internal.h", "vx_blake3.cuh", os.path.join("..", "..", "include", "vx.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC", "--cudart", "shared"]


def _nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: libvx.so cannot be built (there is no CPU fallback)")
    return exe


STAMP = LIB + ".flags"      # the VX_NVCC_EXTRA string libvx.so was built with


def _extra() -> str:
    return " ".join(os.environ.get("VX_NVCC_EXTRA", "").split())      # e.g. -DVX_DEBUG_BOUNDS=1


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    try:
        with open(STAMP) as f:
            built_with = f.read()
    except OSError:
        built_with = None
    if built_with != _extra():     # a debug build must not stay behind as the product build, or vice versa
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/*.cu into paper_2606_14007_b200/libvx.so; returns its path."""
    if force or is_stale():
        extra = _extra().split()
        cmd = [_nvcc(), *NVCC_FLAGS, *extra, *(["-Xptxas", "-v"] if verbose else []), "-o", LIB,
               *[os.path.join(CSRC, s) for s in SOURCES]]
        subprocess.check_call(cmd, cwd=CSRC)
        with open(STAMP, "w") as f:
            f.write(_extra())
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
