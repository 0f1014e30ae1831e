"""Compile the CUDA C-ABI library in-tree: paper_1501_03450_b200/libgst.so (sm_100a only).

The kernel instantiations are spread over nine translation units (csrc/track_inst.cu compiled with different
-DGST_TU_SPLIT / -DGST_TU_GROUP) so that the nvcc runs go in parallel on every host core; objects are kept under
csrc/build/ (git-ignored) and recompiled only when something their unit includes has changed."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
INC = os.path.join(os.path.dirname(HERE), "include")
TRACK_HEADERS = ["track_kernel.cuh", "track_chain_kernel.cuh", "track_split_kernel.cuh", "track_launch.cuh"]
# (object name, source, extra defines, headers it includes): the API, the diagnostics, the allocation-free entry point
# and nine units of kernel instantiations
UNITS = [("gst_api", "gst_api.cu", [], TRACK_HEADERS + ["reduce_kernel.cuh", "gst_internal.h", "gst.h", "gst_diag.h"]),
         ("gst_diag", "gst_diag.cu", [], TRACK_HEADERS + ["gst_internal.h", "gst.h", "gst_diag.h"]),
         ("gst_noalloc", "gst_noalloc.cu", [], ["gst_internal.h", "gst.h"])] + \
    [("track_inst_s%dg%d" % (sp, g), "track_inst.cu", ["-DGST_TU_SPLIT=%d" % sp, "-DGST_TU_GROUP=%d" % g], TRACK_HEADERS)
     for g in (1, 2, 0) for sp in (2, 1, 0)]            # the slowest units first


def _path(f):
    return os.path.join(INC if f in ("gst.h", "gst_diag.h") else CSRC, f)


def _unit_deps(src, headers):
    return [_path(src)] + [_path(h) for h in headers] + [os.path.abspath(__file__)]   # the flags live in this file


DEPS = sorted({d for _, src, _, hdrs in UNITS for d in _unit_deps(src, hdrs)})
OUT = os.path.join(HERE, "libgst.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC"]


KERNEL_SOURCES = ("track_kernel.cuh", "track_chain_kernel.cuh", "track_split_kernel.cuh", "track_launch.cuh", "track_inst.cu")


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
    objs, pending, running = [], [], []
    for unit in UNITS:          # an object is kept when it is newer than everything its unit is compiled from
        obj = os.path.join(OBJ, unit[0] + ".o")
        fresh = os.path.exists(obj) and os.path.getmtime(obj) >= max(os.path.getmtime(d) for d in _unit_deps(unit[1], unit[3]))
        if fresh and not force and not verbose:
            objs.append(obj)
        else:
            pending.append(unit)
    workers = max(1, min(len(UNITS), os.cpu_count() or 1))
    while pending or running:
        while pending and len(running) < workers:
            name, src, defs, _ = pending.pop(0)
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
