"""Build the CPU oracle (test infrastructure) as oracle/liborc_uniboost.so with gcc."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "orc_uniboost.c")
LIB = os.path.join(HERE, "liborc_uniboost.so")


def build(force: bool = False) -> str:
    deps = [SRC, os.path.join(HERE, "orc_uniboost.h")]
    if (not force and os.path.exists(LIB)
            and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps)):
        return LIB
    cmd = ["gcc", "-O2", "-std=c11", "-Wall", "-Wextra", "-fPIC", "-shared", "-o", LIB, SRC, "-lm"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
