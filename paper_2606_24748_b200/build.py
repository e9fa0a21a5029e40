"""Build the native pieces in-tree.

  python -m paper_2606_24748_b200.build            # generator (g++) + CUDA library (nvcc, sm_100a)
  python -m paper_2606_24748_b200.build --gen      # generator only

The CUDA library is compiled for sm_100a only (`-gencode arch=compute_100a,code=sm_100a -lineinfo`).
Outputs: gen/libelastgen.so and csrc/libbsramg.so next to their sources (git-ignored, shipped by gpurun).
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
GEN_SRC = os.path.join(HERE, "gen", "elasticity_gen.cpp")
GEN_LIB = os.path.join(HERE, "gen", "libelastgen.so")
CSRC = os.path.join(HERE, "csrc")
CUDA_LIB = os.path.join(CSRC, "libbsramg.so")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")


def _stale(target: str, sources: list[str]) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(s) > t for s in sources)


def _run(cmd: list[str]) -> None:
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
        raise RuntimeError("build failed: " + os.path.basename(cmd[-1]))
    if r.stderr.strip() and os.environ.get("BSRAMG_VERBOSE"):
        sys.stderr.write(r.stderr)


def build_gen(force: bool = False) -> str:
    if force or _stale(GEN_LIB, [GEN_SRC]):
        _run(["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-fopenmp", "-o", GEN_LIB, GEN_SRC])
    return GEN_LIB


def cuda_sources() -> list[str]:
    return sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cu", ".cpp")))


def cuda_headers() -> list[str]:
    hs = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))]
    hs += [os.path.join(INCLUDE, f) for f in os.listdir(INCLUDE) if f.endswith(".h")]
    return sorted(hs)


def build_cuda(force: bool = False, verbose: bool = False) -> str:
    srcs = cuda_sources()
    if not srcs:
        raise RuntimeError("no CUDA sources under " + CSRC)
    if force or _stale(CUDA_LIB, srcs + cuda_headers()):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
               "-Xcompiler", "-fPIC,-fopenmp", "-shared", "-I", INCLUDE, "-I", CSRC]
        if verbose:
            cmd += ["-Xptxas", "-v"]
        cmd += ["-o", CUDA_LIB] + srcs + ["-lgomp"]
        _run(cmd)
    return CUDA_LIB


def main() -> None:
    only_gen = "--gen" in sys.argv
    force = "--force" in sys.argv
    print(build_gen(force))
    if not only_gen:
        print(build_cuda(force, verbose="-v" in sys.argv))


if __name__ == "__main__":
    main()
