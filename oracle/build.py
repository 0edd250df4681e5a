"""ORACLE — test infrastructure only.  Builds oracle/liboracle_dlo.so with g++ (no CUDA, no torch)."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "liboracle_dlo.so")
SOURCES = ["dlo_oracle.cpp", "rod_step.hpp", "tape.hpp"]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(HERE, s)) > t for s in SOURCES)


def build(force: bool = False) -> str:
    if force or needs_build():
        cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", LIB + ".tmp",
               os.path.join(HERE, "dlo_oracle.cpp")]
        subprocess.run(cmd, check=True, cwd=HERE)
        os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
