"""In-tree build of libchfsi.so (the C-ABI library of include/chfsi.h) with nvcc for sm_100a.

    python -m paper_2203_07820_b200.build [--force] [--verbose]

The shared object is written next to this file so that it travels with the source tree; it links only
against the CUDA runtime (no torch, no Python).
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libchfsi.so")
SOURCES = ["api.cu", "apply_kernels.cu", "rr_kernels.cu", "rr_dense.cu", "rr_umma.cu", "part_kernels.cu", "setup_kernels.cu", "host_setup.cpp", "peak_fp64.cu"]
HEADERS = sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".h", ".cuh"))) + \
    [os.path.join(HERE, "..", "include", "chfsi.h")]
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]


def _nvcc() -> str:
    cand = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(cand):
        raise RuntimeError("nvcc not found: libchfsi cannot be built (there is no CPU fallback)")
    return cand


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile (if stale) and return the path of libchfsi.so.  Safe under torchrun: concurrent callers serialise on
    a file lock (the first one builds, the others find a fresh library), and the library is moved into place
    atomically, so no rank ever dlopens a half-written file."""
    if not force and not _stale():
        return LIB
    import fcntl
    os.makedirs(os.path.join(HERE, "build"), exist_ok=True)
    with open(os.path.join(HERE, "build", ".lock"), "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        try:
            if not force and not _stale():          # another process built it while we waited
                return LIB
            return _build_locked(verbose)
        finally:
            fcntl.flock(lock, fcntl.LOCK_UN)


def _build_locked(verbose: bool) -> str:
    nvcc = _nvcc()
    objs = []
    procs = []
    for s in SOURCES:
        obj = os.path.join(HERE, "build", s + ".o")
        cmd = [nvcc, "-O3", "-std=c++17", "-lineinfo", *ARCH, "-Xcompiler", "-fPIC", "-x", "cu",
               "-c", os.path.join(CSRC, s), "-o", obj]
        cmd[1:1] = os.environ.get("CHFSI_NVCC_FLAGS", "").split()     # extra flags, e.g. -Xptxas=-v
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        procs.append((s, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(obj)
    failed = False
    for s, pr in procs:
        out, _ = pr.communicate()
        if pr.returncode != 0:
            failed = True
            sys.stderr.write(f"--- nvcc failed on {s}\n{out}\n")
        elif verbose:
            sys.stderr.write(f"--- {s}\n{out}\n")
    if failed:
        raise RuntimeError("libchfsi build failed")
    tmp = LIB + f".tmp{os.getpid()}"
    cmd = [nvcc, "-shared", *ARCH, "-o", tmp, *objs, "-cudart", "shared"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
