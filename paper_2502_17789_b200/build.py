"""Build the C-ABI shared library (libidg_b200.so) in-tree with nvcc for sm_100a.

    python -m paper_2502_17789_b200.build [--force]

nvcc cross-compiles without a GPU.  The library lands next to this file so that it travels to
the GPU box with the source tree.
"""
from __future__ import annotations

import concurrent.futures
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
BUILD = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libidg_b200.so")

SOURCES = ["plan.cpp", "api.cu", "gridder.cu", "gridder_tc.cu", "degridder.cu", "degridder_tc.cu", "direct_f64.cu", "fft.cu", "adder.cu", "closure.cu", "peaks.cu", "no_alloc.cu"]
NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC", "-Xcompiler", "-ffp-contract=off", "-Xcompiler", "-fvisibility=hidden",
    "-I", INCLUDE, "-I", CSRC,
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found (set NVCC or put it on PATH)")


def _deps():
    out = [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    out += [os.path.join(INCLUDE, f) for f in os.listdir(INCLUDE)]
    out.append(os.path.abspath(__file__))
    return out


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in _deps())


def _compile(src: str, verbose: bool, extra=(), tag: str = "", objdir: str = BUILD) -> str:
    obj = os.path.join(objdir, os.path.splitext(src)[0] + tag + ".o")
    cmd = [_nvcc(), *NVCC_FLAGS, *extra, "-c", os.path.join(CSRC, src), "-o", obj]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed on {src}:\n{r.stdout}\n{r.stderr}")
    if verbose:
        sys.stderr.write(r.stderr)
    return obj


def build(force: bool = False, verbose: bool = False, extra_flags=(), out: str | None = None) -> str:
    """Compile if needed; returns the path of the shared library.  `extra_flags` / `out` build a
    differently configured copy (e.g. -D tuning macros); its object files go beside `out`, not into the
    in-tree build directory (which every gpurun call ships to the GPU box)."""
    lib = out or LIB
    if out is None and not force and not is_stale():
        return LIB
    objdir = BUILD if out is None else os.path.dirname(os.path.abspath(out))
    os.makedirs(objdir, exist_ok=True)
    tag = "" if out is None else "." + os.path.splitext(os.path.basename(out))[0]
    with concurrent.futures.ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        objs = list(ex.map(lambda s: _compile(s, verbose, tuple(extra_flags), tag, objdir), SOURCES))
    cmd = [_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", lib, *objs,
           "-lcufft", "-Xlinker", "-rpath=/usr/local/cuda/lib64"]     # cuFFT: master-grid FFT of the closure only
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
