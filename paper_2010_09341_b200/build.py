"""Build step: nvcc -> paper_2010_09341_b200/libvegas_b200.so (in-tree, sm_100a only).

``python -m paper_2010_09341_b200.build [--force]`` or ``build()`` from Python.  nvcc cross-compiles
without a GPU.  The library is rebuilt when any source under csrc/ or include/ is newer than it.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
CSRC = os.path.join(_HERE, "csrc")
INCLUDE = os.path.join(_ROOT, "include")
LIB = os.path.join(_HERE, "libvegas_b200.so")
SOURCES = [os.path.join(CSRC, "vegas_api.cu"), os.path.join(CSRC, "pipe_bench.cu"), os.path.join(CSRC, "vegas_rtc.cu"),
           os.path.join(CSRC, "vegas_static.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "vegas_kernels.cuh"), os.path.join(CSRC, "vegas_device.cuh"),
                  os.path.join(CSRC, "vegas_user.cuh"), os.path.join(CSRC, "vegas_rtc.h"),
                  os.path.join(INCLUDE, "vegas_b200.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",   # B200 only; no PTX fallback for other archs
    "-lineinfo", "-O3", "-std=c++17", "--expt-extended-lambda",
    # no -use_fast_math; every fused multiply-add in the per-event code is an explicit intrinsic and
    # the host-side constant setup must not be contracted either
    "-Xcompiler", "-fPIC,-ffp-contract=off",
    "-shared",
    "-lnvrtc",                                       # run-time compilation of user integrands (vegas_create_custom)
]


def kernel_source_sha() -> str:
    """First 16 hex digits of sha256 over the two headers that hold the device code of the iterate kernel.  Stored
    with the per-event counts an ncu capture yields (ncu_counts.py) so that bench.py can tell whether those counts
    still describe the kernels it is running."""
    import hashlib
    h = hashlib.sha256()
    for name in ("vegas_device.cuh", "vegas_kernels.cuh"):
        with open(os.path.join(CSRC, name), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def nvcc_path() -> str:
    cand = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(cand):
        raise RuntimeError("nvcc not found (needed to build libvegas_b200.so)")
    return cand


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(p) > t for p in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or is_stale():
        tmp = LIB + ".tmp.%d" % os.getpid()
        cmd = [nvcc_path(), *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-I", INCLUDE, "-o", tmp, *SOURCES]
        subprocess.run(cmd, check=True)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
