"""TEST INFRASTRUCTURE.  Compile the CPU oracle (oracle/taiga_oracle.cpp) into
oracle/libtaiga_oracle.so.  -ffp-contract=off: fma only where std::fma is written."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "taiga_oracle.cpp")
HDR = os.path.join(HERE, "taiga_oracle.h")
LIB = os.path.join(HERE, "libtaiga_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(SRC), os.path.getmtime(HDR))):
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
           "-Wall", "-o", LIB, SRC]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
