"""Build the CUDA library of cosenu-b200 in-tree for sm_100a.

    python -m paper_2203_12866_b200.build [--force] [--verbose]
        -> paper_2203_12866_b200/libcosenu_b200.so     (the product: kernels + C ABI, include/cosenu.h)

nvcc cross-compiles without a GPU.  -lineinfo keeps the ncu source page mapped to csrc/.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
ROOT = os.path.dirname(HERE)
LIB = os.path.join(HERE, "libcosenu_b200.so")

# translation units of the library: the handle-based API with all stage kernels, and the allocation-free
# cosenu_beam_sums_static, which keeps its file-scope scratch array and the host code that looks its address up in one file
UNITS = ["cosenu_api.cu", "beam_sums_static.cu"]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def source_id():
    """sha1 (12 hex digits) over the sources the library is built from, in a fixed order.  Compiled into the library
    (cosenu_build_id) so that a bench line and an ncu capture can name the binary they ran, not the tree they sat in."""
    import hashlib
    h = hashlib.sha1()
    for f in sorted(os.listdir(CSRC)):
        with open(os.path.join(CSRC, f), "rb") as fh:
            h.update(fh.read())
    with open(os.path.join(ROOT, "include", "cosenu.h"), "rb") as fh:
        h.update(fh.read())
    return h.hexdigest()[:12]


def _newer(out, deps):
    return os.path.exists(out) and all(os.path.getmtime(out) >= os.path.getmtime(d) for d in deps)


def build(force=False, verbose=False):
    srcs = [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC))]
    deps = srcs + [os.path.join(ROOT, "include", "cosenu.h"), os.path.abspath(__file__)]
    if force or not _newer(LIB, deps):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc] + NVCC_FLAGS + ['-DCOSENU_BUILD_ID="%s"' % source_id()] + (["-Xptxas", "-v"] if verbose else []) + \
              ["-o", LIB] + [os.path.join(CSRC, f) for f in UNITS]
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
