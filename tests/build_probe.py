"""Build tests/libcosenu_probe.so: a host compilation of the product's stencil arithmetic (csrc/weno7_math.h) for the CPU tests."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "host_probe.cpp")
HDR = os.path.join(os.path.dirname(HERE), "paper_2203_12866_b200", "csrc", "weno7_math.h")
OUT = os.path.join(HERE, "libcosenu_probe.so")


def build(force=False):
    if not force and os.path.exists(OUT) and all(os.path.getmtime(OUT) >= os.path.getmtime(d) for d in (SRC, HDR)):
        return OUT
    subprocess.run(["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fPIC", "-shared", "-o", OUT, SRC], check=True)
    return OUT


if __name__ == "__main__":
    print(build(force=True))
