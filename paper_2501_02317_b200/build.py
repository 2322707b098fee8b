"""Build the C-ABI library ``libkratos_hydro.so`` in-tree with nvcc for sm_100a.

    python -m paper_2501_02317_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The built .so is git-ignored but travels to the GPU box
with the repository snapshot.  The ptxas resource report (registers, spills, shared memory per
kernel) of the last build is left next to it in ``build_ptxas.log`` (git-ignored too).

Supported option: the environment variable ``KH_NVCC_EXTRA`` holds extra nvcc flags, e.g.
``KH_NVCC_EXTRA="-DKH_TMA_UNROLL=2 -DKH_TMA_MAIN_REGS=200"`` -- the tuning macros the kernel
headers define under ``#ifndef``.  The default build uses none.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libkratos_hydro.so")
SOURCES = ["kh_api.cu"]
HEADERS = ["kh_device.cuh", "kh_simple.cuh", "kh_tiled.cuh", "kh_pair.cuh", "kh_tma.cuh", "kh_strip.cuh", "kh_vanleer.cuh", "kh_reduce.cuh",
           os.path.join("..", "..", "include", "kratos_hydro.h")]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "--shared", "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden",
              "--fmad=true", "-Xptxas", "-v"]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    extra = os.environ.get("KH_NVCC_EXTRA", "").split()  # supported option, see the module docstring
    cmd = [nvcc_path()] + NVCC_FLAGS + extra + ["-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed (exit %d)" % res.returncode)
    os.replace(tmp, LIB)
    with open(os.path.join(HERE, "build_ptxas.log"), "w") as f:
        # (the temporary output name carries the pid: log the final name so that rebuilding leaves the file unchanged)
        log = (res.stdout + res.stderr).replace(tmp, LIB)
        log = "\n".join(l for l in log.split("\n") if "Compile time" not in l)
        f.write(" ".join(cmd).replace(tmp, LIB) + "\n" + log)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
