"""Build the native libraries in-tree (sm_100a only).

  libmg.so          C ABI of include/mg.h          (CUDA: csrc/mg_*.cu + csrc/relabel.cpp)
  libmg_builder.so  C ABI of include/mg_builder.h  (host C++: csrc/builder/*.cpp + csrc/relabel.cpp)
  libmg_synth.so    GPU versions of the synth.py volume generators (CUDA: csrc/synth_kernels.cu)

nvcc cross-compiles without a GPU.  A library is rebuilt when any of its sources is newer.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INC = os.path.join(os.path.dirname(HERE), "include")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC,-fopenmp,-O3,-Wall", "--shared", "-I", INC, "-lgomp"]
GXX_FLAGS = ["-O3", "-std=c++17", "-fPIC", "-fopenmp", "-shared", "-Wall", "-Wextra", "-I", INC]


def _stale(target: str, sources: list[str]) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    deps = sources + glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(CSRC, "builder", "*.h")) + \
        glob.glob(os.path.join(INC, "*.h")) + [os.path.abspath(__file__)]
    return any(os.path.getmtime(s) > t for s in deps)


def _run(cmd: list[str], verbose: bool) -> None:
    if verbose:
        print(" ".join(cmd), flush=True)
    subprocess.check_call(cmd)


def lib_path(name: str) -> str:
    return os.path.join(HERE, name)


def build(force: bool = False, verbose: bool = False, extra_nvcc: list[str] | None = None) -> dict:
    out = {}
    cu = sorted(glob.glob(os.path.join(CSRC, "mg_*.cu"))) + [os.path.join(CSRC, "relabel.cpp")]
    tgt = lib_path("libmg.so")
    if force or _stale(tgt, cu):
        tmp = tgt + f".tmp{os.getpid()}"
        _run(["nvcc"] + NVCC_FLAGS + (extra_nvcc or []) + ["-o", tmp] + cu, verbose)
        os.replace(tmp, tgt)
    out["libmg"] = tgt

    bsrc = sorted(glob.glob(os.path.join(CSRC, "builder", "*.cpp")))
    if bsrc:
        bsrc.append(os.path.join(CSRC, "relabel.cpp"))
        tgt = lib_path("libmg_builder.so")
        if force or _stale(tgt, bsrc):
            tmp = tgt + f".tmp{os.getpid()}"
            _run(["g++"] + GXX_FLAGS + ["-o", tmp] + bsrc, verbose)
            os.replace(tmp, tgt)
        out["libmg_builder"] = tgt

    ssrc = os.path.join(CSRC, "synth_kernels.cu")
    if os.path.exists(ssrc):
        tgt = lib_path("libmg_synth.so")
        if force or _stale(tgt, [ssrc]):
            tmp = tgt + f".tmp{os.getpid()}"
            _run(["nvcc"] + NVCC_FLAGS + ["-o", tmp, ssrc], verbose)
            os.replace(tmp, tgt)
        out["libmg_synth"] = tgt
    return out


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True,
                extra_nvcc=["-Xptxas", "-v"] if "--ptxas-v" in sys.argv else None))
