"""Builds paper_2607_02630_b200/libaesoff.so in-tree with nvcc for sm_100a.

    python -m paper_2607_02630_b200.build [--force]

The shared library is the product (the C ABI of include/aesoff.h); it links the
CUDA runtime statically and nothing else, and it travels to the GPU box with the
repository snapshot.  nvcc cross-compiles without a GPU.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

_PKG = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_PKG)
CSRC = os.path.join(_PKG, "csrc")
SO = os.path.join(_PKG, "libaesoff.so")
SOURCES = ["aesoff_kernels.cu", "aesoff_calib.cu", "aesoff_runtime.cpp", "aesoff_keys.cpp", "aesoff_router.cpp"]
HEADERS = ["aesoff_shared.h", "aesoff_internal.h", "aesoff_cipher.cuh", "aesoff_bitslice.cuh", os.path.join(_ROOT, "include", "aesoff.h")]

NVCC_FLAGS = [
    "-O3", "-std=c++17", "-lineinfo",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-Xcompiler", "-fPIC,-O2,-Wall,-fvisibility=hidden",
    "-Xptxas", "-v",
    "--shared", "-cudart", "static",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA extension cannot be built (there is no CPU fallback)")


def _stale() -> bool:
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + [h if os.path.isabs(h) else os.path.join(CSRC, h) for h in HEADERS]
    deps.append(os.path.abspath(__file__))
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return SO
    tmp = SO + ".%d.tmp" % os.getpid()
    extra = os.environ.get("AESOFF_NVCC_EXTRA", "").split()  # e.g. -DAESOFF_NB=8 for tuning experiments
    cmd = [_nvcc()] + NVCC_FLAGS + extra + ["-I", os.path.join(_ROOT, "include"), "-I", CSRC, "-o", tmp]
    cmd += ["-x", "cu"] + [os.path.join(CSRC, s) for s in SOURCES]
    cmd += ["-lpthread", "-ldl", "-lrt"]
    proc = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if proc.returncode != 0:
        sys.stderr.write(proc.stdout)
        raise RuntimeError("nvcc failed (exit %d)" % proc.returncode)
    if verbose:
        sys.stderr.write(proc.stdout)
    os.replace(tmp, SO)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
