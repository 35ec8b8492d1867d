"""Build step for the oracle's C part (TEST INFRASTRUCTURE, not the product).

`build_oracle()` compiles oracle/attention_ref.c into oracle/liboracle_attention.so with gcc.
Building the checker is not using it: __graft_entry__.build() calls this, the product never does.
"""
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(_HERE, "attention_ref.c")
LIB = os.path.join(_HERE, "liboracle_attention.so")


def build_oracle(force: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-Wall", "-Wextra", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build_oracle(force=True))
