"""Builds paper_2604_20295_b200/libetac.so (C-ABI, include/etac.h) with nvcc for sm_100a.

    python -m paper_2604_20295_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The .so is kept in-tree (git-ignored) so that it travels to
the GPU box with the repository snapshot."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libetac.so")
SOURCES = ["etac_api.cu", "k_build.cu", "k_sdf.cu", "k_gather_fp32.cu", "k_pointnet_fp32.cu", "k_fused.cu", "k_backward.cu", "k_backward_pointnet.cu", "k_backward_pose.cu", "k_peaks.cu", "k_noalloc.cu", "k_mesh.cu"]
HEADERS = ["etac_internal.h", "sm100_prims.cuh", "pointnet_fp32.cuh", "sdf_device.cuh", os.path.join("..", "..", "include", "etac.h"),
           os.path.join("..", "..", "include", "etac_bench.h"), os.path.join("..", "..", "include", "etac_noalloc.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
         "-Xcompiler", "-fPIC", "--expt-relaxed-constexpr", "-cudart", "static"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compiles the library if it is missing or older than a source.  Several processes may call this at once (one
    rank per GPU under torchrun): an exclusive lock on a file beside the library serialises them, the check is repeated
    under the lock, and the link goes to a temporary name that is renamed into place."""
    if not force and not _stale():
        return LIB
    import fcntl
    with open(LIB + ".lock", "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        try:
            if not force and not _stale():          # another process built it while this one waited
                return LIB
            return _build_locked(verbose)
        finally:
            fcntl.flock(lock, fcntl.LOCK_UN)


def _build_locked(verbose: bool) -> str:
    objs = []
    procs = []
    for s in SOURCES:
        o = os.path.join(CSRC, s.replace(".cu", ".o"))
        cmd = [NVCC, *FLAGS, "-c", os.path.join(CSRC, s), "-o", o]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
            print(" ".join(cmd), flush=True)
        procs.append((s, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(o)
    failed = False
    for s, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0 or verbose:
            sys.stderr.write(f"--- {s}\n{out}\n")
        failed |= p.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed")
    tmp = LIB + f".tmp{os.getpid()}"
    cmd = [NVCC, "-shared", "-cudart", "static", "-o", tmp, *objs]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
