"""Compile the CPU oracle (oracle.cpp -> liboracle.so) with g++.  Test infrastructure only.

Flags: -O2 -ffp-contract=off (canonical arithmetic); -mfma so that std::fma is the
hardware instruction (correctly rounded either way)."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "oracle.cpp")
LIB = os.path.join(HERE, "liboracle.so")


def build(force: bool = False) -> str:
    deps = [SRC, os.path.join(HERE, "oracle.h")]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-mfma", "-mavx2", "-fPIC", "-shared",
           "-Wall", "-Wextra"] + os.environ.get("ORACLE_CXXFLAGS", "").split() + ["-o", LIB, SRC]      # e.g. -fsanitize=address,undefined -g
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
