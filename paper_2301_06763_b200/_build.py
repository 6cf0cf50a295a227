"""Build libcm.so in-tree with nvcc for sm_100a (no JIT cache, no torch extension)."""
from __future__ import annotations

import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libcm.so")
# translation units, compiled side by side and linked into one library
SOURCES = ["cm_lib.cu", "cm_static.cu"]
DEPS = SOURCES + ["cm_kernels.cuh", "cm_zconv.cuh", "cm_expand.cuh", "cm_fft.cuh", os.path.join("..", "..", "include", "cm.h")]

# no --use_fast_math: fp64 parity needs IEEE division and sqrt
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC"]


def needs_build() -> bool:
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    return any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in DEPS)


def _run(cmd):
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + r.stdout + r.stderr)
    return r.stderr


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        objs = [os.path.join(HERE, "_" + os.path.splitext(s)[0] + ".o") for s in SOURCES]
        cmds = [[nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", o, os.path.join(CSRC, s)]
                for s, o in zip(SOURCES, objs)]
        try:
            with ThreadPoolExecutor(len(cmds)) as ex:
                logs = list(ex.map(_run, cmds))
            _run([nvcc, "-shared", "-o", SO] + objs)
        finally:
            for o in objs:
                if os.path.exists(o):
                    os.remove(o)
        if verbose:
            print("\n".join(logs))
    return SO
