"""ORACLE — TEST INFRASTRUCTURE ONLY.  Builds oracle/liboracle.so from oracle/cavity_oracle.cpp.

Plain g++, no CUDA, no torch.  -ffp-contract=off keeps the PLAIN arithmetic mode free of fused
multiply-adds; std::fma in the FMA mode is exact either way.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "cavity_oracle.cpp")
LIB = os.path.join(HERE, "liboracle.so")


def build(force: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fvisibility=hidden", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", tmp, SRC]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
