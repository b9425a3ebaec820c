"""Build tests/libcosenu_probe.so: a host compilation of the product's stencil arithmetic (csrc/weno7_math.h) for the CPU tests,
and tests/libcosenu_device_probe.so: a device compilation of its per-beam constants for one GPU test."""
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


DEV_SRC = os.path.join(HERE, "device_probe.cu")
DEV_OUT = os.path.join(HERE, "libcosenu_device_probe.so")


def build_device(force=False):
    """nvcc for sm_100a (cross-compiles without a GPU); returns None when there is no nvcc to build it with."""
    if not force and os.path.exists(DEV_OUT) and all(os.path.getmtime(DEV_OUT) >= os.path.getmtime(d) for d in (DEV_SRC, HDR)):
        return DEV_OUT
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    if not os.path.exists(nvcc):
        return DEV_OUT if os.path.exists(DEV_OUT) else None
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-Xcompiler", "-fPIC", "-shared",
                    "-cudart", "static", "-o", DEV_OUT, DEV_SRC], check=True)
    return DEV_OUT


if __name__ == "__main__":
    print(build(force=True))
    print(build_device(force=True))
