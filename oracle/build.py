"""Build the CPU oracle (test infrastructure) into oracle/liboracle_tnlm.so with gcc.

Run as `python -m oracle.build` or call `build()`; `oracle/__init__.py` calls it on first use
when the shared object is missing or older than the source.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "tnlm_oracle.c")
LIB = os.path.join(HERE, "liboracle_tnlm.so")


def needs_build() -> bool:
    return (not os.path.exists(LIB)) or os.path.getmtime(LIB) < os.path.getmtime(SRC)


def build(force: bool = False) -> str:
    if force or needs_build():
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-fno-fast-math",
               "-o", LIB, SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
