"""Build the CUDA library libsldg.so in-tree for sm_100a (B200).

    python -m paper_1907_08316_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so sits beside the sources (git-ignored) so that
it travels to the GPU box with the repository snapshot.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsldg.so")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")


def _deps():
    deps = [os.path.join(INCLUDE, "sldg.h")]
    for name in sorted(os.listdir(CSRC)):
        if name.endswith((".cu", ".cuh", ".hpp", ".h")):
            deps.append(os.path.join(CSRC, name))
    return deps


def build(force=False, verbose=False):
    deps = _deps()
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
           "--fmad=false",            # every FMA in the sweep is explicit (O7 contract)
           "-Xcompiler", "-fPIC", "-shared", "-I", INCLUDE,
           "-o", LIB + ".tmp", os.path.join(CSRC, "sldg.cu")]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    subprocess.run(cmd, check=True, cwd=CSRC)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
