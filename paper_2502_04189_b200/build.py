"""Build step for libfizzy.so (the C-ABI product, include/fizzy.h): one nvcc call, sm_100a only.

`python -m paper_2502_04189_b200.build` or `build()`; the library is written IN-TREE next to
this file so that it travels to the GPU box with the repository snapshot."""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libfizzy.so")
SOURCES = ["fizzy_api.cu", "fizzy_static.cu"]
HEADERS = ["fz_common.cuh", "fz_stencil.cuh", "fz_momentum.cuh", "fz_fft.cuh", "fz_fftx.cuh", "fz_spectral.cuh", "fz_linefft.cuh", "fz_iface.cuh", "fz_diag.cuh", "fz_mg.cuh"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-std=c++17", "-O3", "-lineinfo",
              "-shared", "-Xcompiler", "-fPIC", "-cudart", "static"]


def _newest_source() -> float:
    inc = os.path.join(os.path.dirname(_HERE), "include", "fizzy.h")
    files = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [inc]
    return max(os.path.getmtime(f) for f in files)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile libfizzy.so if missing or older than its sources.  Returns its path."""
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= _newest_source():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + \
          [os.path.join(CSRC, f) for f in SOURCES]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + res.stdout + res.stderr)
    if verbose:
        print(res.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
