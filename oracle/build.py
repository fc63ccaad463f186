"""Builds the C part of the oracle (oracle/alg1.c) with gcc.  Test infrastructure only.

Flags: `-O3 -march=native -fopenmp` as SURVEY 8(d) / BASELINE.md state for the timed CPU baseline; `-ffp-contract=off`
keeps the arithmetic as written (no fused multiply-adds).  `-march=native` binds the library to the CPU it was built
on, and built `.so` files travel with the tree to other machines, so the flags of the building CPU are recorded beside
the library and a different CPU rebuilds it."""
import hashlib
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
FLAGS = ["-O3", "-march=native", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared"]


def _host_tag():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    return hashlib.sha1(line.encode()).hexdigest()
    except OSError:
        pass
    return "unknown"


def build_alg1(force=False):
    src = os.path.join(HERE, "alg1.c")
    out = os.path.join(HERE, "liboracle_alg1.so")
    tag_file = out + ".host"
    tag = _host_tag() + " " + " ".join(FLAGS)
    try:
        with open(tag_file) as f:
            same_host = f.read() == tag
    except OSError:
        same_host = False
    if force or not same_host or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(src):
        subprocess.check_call(["gcc", *FLAGS, "-o", out, src])
        with open(tag_file, "w") as f:
            f.write(tag)
    return out


if __name__ == "__main__":
    print(build_alg1(force=True))
