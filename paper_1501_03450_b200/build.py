"""Compile the CUDA C-ABI library in-tree: paper_1501_03450_b200/libgst.so (sm_100a only).

The kernel instantiations are spread over nine translation units (csrc/track_inst.cu compiled with different
-DGST_TU_SPLIT / -DGST_TU_GROUP) so that the nvcc runs go in parallel on every host core; objects are kept under
csrc/build/ (git-ignored)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
# (object name, source, extra defines): the API, the diagnostics and nine units of kernel instantiations
UNITS = [("gst_api", "gst_api.cu", []), ("gst_diag", "gst_diag.cu", [])] + \
    [("track_inst_s%dg%d" % (sp, g), "track_inst.cu", ["-DGST_TU_SPLIT=%d" % sp, "-DGST_TU_GROUP=%d" % g])
     for g in (1, 2, 0) for sp in (2, 1, 0)]            # the slowest units first
DEPS = [os.path.join(CSRC, f) for f in ("gst_api.cu", "gst_diag.cu", "track_inst.cu", "track_kernel.cuh",
                                        "track_chain_kernel.cuh", "track_launch.cuh", "reduce_kernel.cuh",
                                        "gst_internal.h")] + \
    [os.path.join(os.path.dirname(HERE), "include", f) for f in ("gst.h", "gst_diag.h")] + \
    [os.path.abspath(__file__)]   # the flags live in this file
OUT = os.path.join(HERE, "libgst.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC"]


KERNEL_SOURCES = ("track_kernel.cuh", "track_chain_kernel.cuh", "track_launch.cuh", "track_inst.cu")


def kernel_source_hash() -> str:
    """Fingerprint of what the tracking kernels are compiled from (sources and flags): compiled into the library
    (gst_diag_kernel_source_hash) so that bench.py can tell whether its flop model was captured on this code."""
    import hashlib
    h = hashlib.sha1(" ".join(NVCC_FLAGS).encode())
    for f in KERNEL_SOURCES:
        h.update(open(os.path.join(CSRC, f), "rb").read())
    return h.hexdigest()[:16]


def build(force: bool = False, verbose: bool = False) -> str:
    newest = max(os.path.getmtime(p) for p in DEPS)
    if not force and os.path.exists(OUT) and os.path.getmtime(OUT) >= newest:
        return OUT
    nvcc = os.environ.get("NVCC", "nvcc")
    os.makedirs(OBJ, exist_ok=True)
    objs, pending, running = [], list(UNITS), []
    workers = max(1, min(len(UNITS), os.cpu_count() or 1))
    while pending or running:
        while pending and len(running) < workers:
            name, src, defs = pending.pop(0)
            obj = os.path.join(OBJ, name + ".o")
            if name == "gst_diag":
                defs = defs + ['-DGST_KERNEL_SOURCE_HASH="%s"' % kernel_source_hash()]
            cmd = [nvcc] + NVCC_FLAGS + defs + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, os.path.join(CSRC, src)]
            running.append((obj, cmd, subprocess.Popen(cmd, cwd=CSRC, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        obj, cmd, proc = running.pop(0)
        out, _ = proc.communicate()
        if verbose or proc.returncode != 0:
            sys.stdout.write(out)
        if proc.returncode != 0:
            for _, _, other in running:
                other.kill()
            raise subprocess.CalledProcessError(proc.returncode, cmd)
        objs.append(obj)
    subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", OUT] + objs, cwd=CSRC)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
