"""Build the CPU oracle's shared object (gcc -O2 -fopenmp, no -ffast-math).

TEST INFRASTRUCTURE: see ck_oracle.h.  `python -m oracle.build` or oracle.build.build().
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "ck_oracle.c")
SRC_JAC = os.path.join(HERE, "ck_oracle_jac.c")
HDR = os.path.join(HERE, "ck_oracle.h")
LIB = os.path.join(HERE, "libck_oracle.so")


def build(force: bool = False) -> str:
    newest = max(os.path.getmtime(SRC), os.path.getmtime(SRC_JAC), os.path.getmtime(HDR))
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-o", LIB + ".tmp", SRC, SRC_JAC, "-lm"]
    subprocess.run(cmd, check=True, cwd=HERE)
    os.replace(LIB + ".tmp", LIB)
    return LIB


def build_sanitized(outdir: str) -> str:
    """The same sources with AddressSanitizer and UndefinedBehaviorSanitizer, into `outdir` (SURVEY.md
    section 5): loaded instead of the normal build when CK_ORACLE_LIB names it, in a process that has
    libasan preloaded (tests/test_oracle_sanitized.py)."""
    lib = os.path.join(outdir, "libck_oracle_san.so")
    cmd = ["gcc", "-O1", "-g", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer",
           "-o", lib, SRC, SRC_JAC, "-lm"]
    subprocess.run(cmd, check=True, cwd=HERE)
    return lib


if __name__ == "__main__":
    print(build(force=True))
