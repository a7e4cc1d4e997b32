"""Builds inputs/libgen.so (plain C + OpenMP) in-tree."""
import fcntl
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "gen.c")
LIB = os.path.join(HERE, "libgen.so")


def _build(force: bool = False) -> str:
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < os.path.getmtime(SRC):
        cmd = ["gcc", "-O2", "-fPIC", "-shared", "-fopenmp", "-o", LIB, SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return LIB


def build(*args, **kwargs) -> str:
    """Serialised across processes (torchrun ranks share the tree) with a lock file."""
    with open(os.path.join(HERE, ".build.lock"), "w") as lk:
        fcntl.flock(lk, fcntl.LOCK_EX)
        try:
            return _build(*args, **kwargs)
        finally:
            fcntl.flock(lk, fcntl.LOCK_UN)


if __name__ == "__main__":
    print(build(force=True))
