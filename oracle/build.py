"""Build the CPU oracle shared library (TEST INFRASTRUCTURE, not the product).

    python oracle/build.py

compiles oracle/sldg_oracle.c into oracle/liboracle_sldg.so with gcc.  Flags:
-O2, hardware FMA for fma()/fmaf() (-mfma when the host has it), no FP contraction
or fast-math (the O7 chain order is part of the contract), OpenMP over lines.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "sldg_oracle.c")
DEPS = [SRC, os.path.join(HERE, "sldg_oracle_real.inc"), os.path.join(HERE, "sldg_oracle.h")]
LIB = os.path.join(HERE, "liboracle_sldg.so")


def _host_has_fma():
    try:
        with open("/proc/cpuinfo") as fh:
            return " fma " in fh.read().replace("\n", " ")
    except OSError:
        return False


def build(force=False):
    if not force and os.path.exists(LIB):
        if all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
            return LIB
    cmd = ["gcc", "-std=c11", "-O2", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
           "-fno-fast-math", "-Wall", "-Wextra", "-Wno-unknown-pragmas"]
    if _host_has_fma():
        cmd.append("-mfma")
    cmd += ["-o", LIB + ".tmp", SRC, "-lm"]
    subprocess.run(cmd, check=True, cwd=HERE)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
