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


SOURCES = ("sldg.cu", "rho_noalloc.cu")     # one object each; rho_noalloc.cu holds sldg_rho_noalloc and its scratch


def _headers():
    deps = [os.path.join(INCLUDE, "sldg.h")]
    for name in sorted(os.listdir(CSRC)):
        if name.endswith((".cuh", ".hpp", ".h")):
            deps.append(os.path.join(CSRC, name))
    return deps


def _stale(target, deps):
    return not os.path.exists(target) or any(os.path.getmtime(target) < os.path.getmtime(d) for d in deps)


def build(force=False, verbose=False):
    headers = _headers()
    if not force and not _stale(LIB, headers + [os.path.join(CSRC, n) for n in SOURCES]):
        return LIB                                      # up to date, whether or not the objects are still there
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    flags = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
             "--fmad=false",            # every FMA in the sweep is explicit (O7 contract)
             "-Xcompiler", "-fPIC", "-I", INCLUDE]
    if verbose:
        flags.insert(0, "-Xptxas=-v")
    objs, jobs = [], []
    for name in SOURCES:
        src = os.path.join(CSRC, name)
        obj = os.path.join(CSRC, name[:-3] + ".o")     # beside the source, git-ignored
        objs.append(obj)
        if force or _stale(obj, headers + [src]):
            jobs.append((obj, subprocess.Popen([nvcc] + flags + ["-c", "-o", obj + ".tmp", src], cwd=CSRC)))
    for obj, proc in jobs:                              # the translation units compile side by side
        if proc.wait() != 0:
            raise subprocess.CalledProcessError(proc.returncode, proc.args)
        os.replace(obj + ".tmp", obj)
    if force or jobs or _stale(LIB, objs):
        subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB + ".tmp"] + objs,
                       check=True, cwd=CSRC)
        os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
