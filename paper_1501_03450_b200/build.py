"""Compile the CUDA C-ABI library in-tree: paper_1501_03450_b200/libgst.so (sm_100a only).

The kernel instantiations of each split live in their own translation unit (csrc/track_split_*.cu) so that the
nvcc runs go in parallel; objects are kept under csrc/build/ (git-ignored)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
SRC = [os.path.join(CSRC, f) for f in ("gst_api.cu", "gst_diag.cu", "track_split_dk.cu", "track_split_bk.cu", "track_split_mk.cu")]
DEPS = SRC + [os.path.join(CSRC, f) for f in ("track_kernel.cuh", "track_chain_kernel.cuh", "track_launch.cuh",
                                              "reduce_kernel.cuh", "gst_internal.h")] + \
    [os.path.join(os.path.dirname(HERE), "include", f) for f in ("gst.h", "gst_diag.h")] + \
    [os.path.abspath(__file__)]   # the flags live in this file
OUT = os.path.join(HERE, "libgst.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC"]


def build(force: bool = False, verbose: bool = False) -> str:
    newest = max(os.path.getmtime(p) for p in DEPS)
    if not force and os.path.exists(OUT) and os.path.getmtime(OUT) >= newest:
        return OUT
    nvcc = os.environ.get("NVCC", "nvcc")
    os.makedirs(OBJ, exist_ok=True)
    jobs = []
    for src in SRC:
        obj = os.path.join(OBJ, os.path.basename(src)[:-3] + ".o")
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, src]
        jobs.append((obj, cmd, subprocess.Popen(cmd, cwd=CSRC, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    objs = []
    for obj, cmd, proc in jobs:
        out, _ = proc.communicate()
        if verbose or proc.returncode != 0:
            sys.stdout.write(out)
        if proc.returncode != 0:
            raise subprocess.CalledProcessError(proc.returncode, cmd)
        objs.append(obj)
    subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", OUT] + objs, cwd=CSRC)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
