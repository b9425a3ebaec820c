"""Build the CPU oracle shared library (test infrastructure, not the product).

    python oracle/build_oracle.py        ->  oracle/libcosenu_ref.so

-ffp-contract=off keeps the arithmetic exactly as written in cosenu_ref.cpp (no FMA fusion);
-fopenmp parallelises over z only (the per-cell arithmetic and its order are unchanged).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "cosenu_ref.cpp")
OUT = os.path.join(HERE, "libcosenu_ref.so")


def build(force: bool = False) -> str:
    deps = [SRC, os.path.join(HERE, "cosenu_ref.h")]
    if (not force and os.path.exists(OUT)
            and all(os.path.getmtime(OUT) >= os.path.getmtime(d) for d in deps)):
        return OUT
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", OUT, SRC]
    subprocess.run(cmd, check=True)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
