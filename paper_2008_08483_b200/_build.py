"""Builds libck.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

`python -m paper_2008_08483_b200._build` or paper_2008_08483_b200._build.build().
nvcc cross-compiles without a GPU, so this also runs on the CPU-only build box.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libck.so")
SOURCES = ["ck_api.cu", "ck_kernels.cu", "ck_jit.cu", "ck_rk4.cu", "ck_jac.cu", "ck_peaks.cu", "ck_nu.cu", "ck_jacj.cu", "ck_static.cu"]
HEADERS = ["ck_internal.h", "ck_program.h", "ck_jit_kernel.cuh", "ck_jit_math.cuh", "ck_nu_kernel.cuh", "ck_jac_v2.cuh", "ck_jacj_kernel.cuh"]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC"]


def _newest_source() -> float:
    files = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.join(INCLUDE, "ck.h")]
    return max(os.path.getmtime(f) for f in files)


def _embed_jit_source() -> None:
    """ck_jit_kernel.cuh, ck_nu_kernel.cuh (+ the shared ck_jit_math.cuh pasted in at their
    //@@CK_MATH@@ line) -> ck_jit_source.inc, ck_nu_source.inc: the kernel texts as C++ raw string
    literals (what NVRTC compiles at ck_mech_create time)."""
    math = open(os.path.join(CSRC, "ck_jit_math.cuh")).read()
    for src, dst in (("ck_jit_kernel.cuh", "ck_jit_source.inc"), ("ck_nu_kernel.cuh", "ck_nu_source.inc"),
                     ("ck_jacj_kernel.cuh", "ck_jacj_source.inc")):
        text = open(os.path.join(CSRC, src)).read()
        assert text.count("//@@CK_MATH@@") == 1
        line = [l for l in text.splitlines() if l.startswith("//@@CK_MATH@@")][0]
        text = text.replace(line, math)
        assert ')CKJIT"' not in text
        chunks = [text[i:i + 8000] for i in range(0, len(text), 8000)]
        out = "".join('R"CKJIT(' + c + ')CKJIT"\n' for c in chunks)
        path = os.path.join(CSRC, dst)
        if not os.path.exists(path) or open(path).read() != out:      # (keeps the object cache valid)
            with open(path, "w") as fh:
                fh.write(out)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= _newest_source():
        return LIB
    _embed_jit_source()
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    newest_header = max(os.path.getmtime(f) for f in
                        [os.path.join(CSRC, h) for h in HEADERS + ["ck_jit_source.inc", "ck_nu_source.inc", "ck_jacj_source.inc"]] +
                        [os.path.join(INCLUDE, "ck.h")])

    def compile_one(src):
        obj = os.path.join(objdir, src.replace(".cu", ".o"))
        path = os.path.join(CSRC, src)
        if not force and os.path.exists(obj) and os.path.getmtime(obj) >= max(os.path.getmtime(path), newest_header):
            return obj
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, path]
        subprocess.run(cmd, check=True, cwd=CSRC)
        return obj

    # the translation units compile side by side (the Jacobian kernel's templates dominate)
    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(max_workers=len(SOURCES)) as pool:
        objs = list(pool.map(compile_one, SOURCES))
    subprocess.run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB + ".tmp"] + objs + ["-ldl"],
                   check=True, cwd=CSRC)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
