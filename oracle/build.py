"""Builds the C part of the oracle (oracle/alg1.c) with gcc.  Test infrastructure only."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))


def build_alg1(force=False):
    src = os.path.join(HERE, "alg1.c")
    out = os.path.join(HERE, "liboracle_alg1.so")
    if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", out, src])
    return out


if __name__ == "__main__":
    print(build_alg1(force=True))
