"""Build libcm.so in-tree with nvcc for sm_100a (no JIT cache, no torch extension)."""
from __future__ import annotations

import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libcm.so")
# translation units, compiled side by side and linked into one library
SOURCES = ["cm_lib.cu", "cm_lib_expand.cu", "cm_static.cu"]
DEPS = SOURCES + ["cm_plan.h", "cm_kernels.cuh", "cm_zconv.cuh", "cm_expand.cuh", "cm_fft.cuh", os.path.join("..", "..", "include", "cm.h")]

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
    """Compile the translation units side by side and link libcm.so.  Safe against concurrent callers (ranks of one job,
    parallel test workers): one builder at a time under a file lock, objects in a private directory, and the library
    moved into place atomically, so a process that has the old one mapped keeps a consistent file."""
    if not (force or needs_build()):
        return SO
    import fcntl
    import shutil
    import tempfile
    with open(os.path.join(HERE, ".build.lock"), "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        if not (force or needs_build()):          # another process built it while this one waited
            return SO
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = tempfile.mkdtemp(prefix=".build_", dir=HERE)
        try:
            objs = [os.path.join(tmp, os.path.splitext(s)[0] + ".o") for s in SOURCES]
            cmds = [[nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", o, os.path.join(CSRC, s)]
                    for s, o in zip(SOURCES, objs)]
            with ThreadPoolExecutor(len(cmds)) as ex:
                logs = list(ex.map(_run, cmds))
            out = os.path.join(tmp, "libcm.so")
            _run([nvcc, "-shared", "-o", out] + objs)
            os.replace(out, SO)
        finally:
            shutil.rmtree(tmp, ignore_errors=True)
        if verbose:
            print("\n".join(logs))
    return SO
