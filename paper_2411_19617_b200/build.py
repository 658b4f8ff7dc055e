"""Build libmala_snap.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2411_19617_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with the snapshot.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmala_snap.so")
SOURCES = ["mala_snap.cu", "mala_mlp.cu"]
DEPS = ["mala_snap.cu", "mala_mlp.cu", "snap_common.cuh", "snap_internal.h", "snap_tables.h", "snap_ui.cuh", "snap_ui_dft.cuh", "snap_ui_pipe.cuh", "snap_dedr_dft.cuh", "snap_yi_fix.cuh", "snap_zi.cuh", "snap_zi_coop.cuh",
        "snap_zi_diag.cuh", "snap_zi_block.cuh", "snap_gauss.cuh", "snap_force.cuh", "snap_yi_block.cuh", os.path.join("..", "..", "include", "mala_snap.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "--expt-relaxed-constexpr", "-std=c++17",
              "-Xcompiler", "-fPIC", "-diag-suppress", "177"]


def nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def build(force: bool = False, verbose: bool = False) -> str:
    newest = max(os.path.getmtime(os.path.join(CSRC, d)) for d in DEPS)
    newest = max(newest, os.path.getmtime(os.path.abspath(__file__)))
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    procs, objs = [], []
    for src in SOURCES:   # one nvcc per translation unit, side by side
        obj = os.path.join(objdir, os.path.splitext(src)[0] + ".o")
        objs.append(obj)
        cmd = [nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, src]
        procs.append((cmd, subprocess.Popen(cmd, cwd=CSRC)))
    for cmd, p in procs:
        if p.wait() != 0:
            raise subprocess.CalledProcessError(p.returncode, cmd)
    subprocess.check_call([nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
