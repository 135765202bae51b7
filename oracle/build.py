"""Build the oracle shared library (TEST INFRASTRUCTURE; see rt_oracle.cpp header).

    python -m oracle.build

g++ only, -O2 -ffp-contract=off so that no product-sum is fused: every fp64 operation in
rt_oracle.cpp is one IEEE round-to-nearest operation in source order.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "rt_oracle.cpp")
LIB = os.path.join(HERE, "librt_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math",
           "-shared", "-fPIC", "-pthread", "-o", LIB, SRC]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
