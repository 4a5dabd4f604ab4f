"""Builds harness/libamr_host.so (native clustering / nesting mask / flag unpacking of the AMR harness) in-tree with gcc.

    python -m harness.build
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "amr_host.c")
LIB = os.path.join(HERE, "libamr_host.so")


def build(force=False):
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    subprocess.check_call(["gcc", "-O2", "-std=c11", "-Wall", "-Wno-misleading-indentation", "-shared", "-fPIC", "-o", LIB, SRC])
    return LIB


if __name__ == "__main__":
    print(build(force=True))
