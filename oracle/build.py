"""Build the CPU oracle shared library (test infrastructure; see sa_oracle.cpp header).

    python -m oracle.build        # or oracle.build.build()

Plain g++; no CUDA, no torch. The product (paper_2606_23019_b200) never imports this package.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "sa_oracle.cpp")
LIB = os.path.join(HERE, "libsa_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-pthread", "-Wall", "-Wextra",
           "-o", LIB, SRC]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
