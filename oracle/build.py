"""Build the ORACLE shared library (test infrastructure, CPU only).

    python oracle/build.py

gcc -O2 -ffp-contract=off (no FMA contraction: plain IEEE fp64 in source order), OpenMP over
primaries.  Called by __graft_entry__.build(), tests/conftest.py and bench.py's cpu_baseline leg.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = ["emo_philox.c", "emo_xs.c", "emo_problem.c", "emo_geom.c", "emo_field.c", "emo_interact.c", "emo_transport.c"]
LIB = os.path.join(HERE, "libemo.so")


def build(force=False):
    srcs = [os.path.join(HERE, s) for s in SRC]
    deps = srcs + [os.path.join(HERE, "emo.h")]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    cmd = ["gcc", "-std=c11", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-o", LIB] + srcs + ["-lm"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
