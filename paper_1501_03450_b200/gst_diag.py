"""ctypes binding over the diagnostics of libgst.so (include/gst_diag.h): roofline microbenchmarks, the accuracy
self-test of the kernels' reciprocals, kernel resource queries and the fault-injection hook of the tests.  Not part
of the tracking API (paper_1501_03450_b200.gst)."""
import ctypes as C

from . import gst

EXPORTS = ["gst_diag_fp64_peak", "gst_diag_fp64_peak_rrr", "gst_diag_selftest_math", "gst_diag_selftest_ring",
           "gst_diag_chain_poll_limit", "gst_diag_kernel_info", "gst_diag_kernel_source_hash"]
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)
_ready = False


def lib():
    global _ready
    L = gst.lib()
    if not _ready:
        L.gst_diag_fp64_peak.argtypes = [_dp, _dp]
        L.gst_diag_fp64_peak_rrr.argtypes = [_dp, _dp]
        L.gst_diag_selftest_math.argtypes = [_dp]
        L.gst_diag_selftest_ring.argtypes = [C.c_uint32, C.c_uint32, C.POINTER(C.c_int64)]
        L.gst_diag_chain_poll_limit.argtypes = [C.c_void_p, C.c_int64]
        L.gst_diag_kernel_info.argtypes = [C.c_int, C.c_int, C.c_int, _ip, _ip, _ip]
        for name in EXPORTS:
            getattr(L, name).restype = C.c_int
        L.gst_diag_kernel_source_hash.restype = C.c_char_p
        L.gst_diag_kernel_source_hash.argtypes = []
        _ready = True
    return L


def fp64_peak():
    """gst_diag_fp64_peak: measured DFMA peak of the current device (TFLOP/s) and the kernel time (ms)."""
    t = C.c_double(0)
    ms = C.c_double(0)
    gst._check(lib().gst_diag_fp64_peak(C.byref(t), C.byref(ms)))
    return t.value, ms.value


def fp64_peak_rrr():
    """gst_diag_fp64_peak_rrr: the same with three distinct register operands per DFMA (TFLOP/s, ms)."""
    t = C.c_double(0)
    ms = C.c_double(0)
    gst._check(lib().gst_diag_fp64_peak_rrr(C.byref(t), C.byref(ms)))
    return t.value, ms.value


def selftest_math():
    """gst_diag_selftest_math: max residuals of the kernels' rcp / rsqrt in units of 2^-53."""
    out = (C.c_double * 2)()
    gst._check(lib().gst_diag_selftest_math(out))
    return out[0], out[1]


def selftest_ring(start_count, n_entries):
    """gst_diag_selftest_ring: values that came out of the two-warp kernel's ring wrong (0 expected)."""
    bad = C.c_int64(-1)
    gst._check(lib().gst_diag_selftest_ring(int(start_count), int(n_entries), C.byref(bad)))
    return bad.value


def chain_poll_limit(bunch, polls):
    """gst_diag_chain_poll_limit: make the next rotating launches on `bunch` give up after `polls` polls (0: default)."""
    gst._check(lib().gst_diag_chain_poll_limit(bunch._h, int(polls)))


def kernel_source_hash():
    """gst_diag_kernel_source_hash: fingerprint of the kernel sources and flags this library was built from."""
    return lib().gst_diag_kernel_source_hash().decode()


KERNEL_VARIANTS = {"track_kernel": 0, "track_chain_kernel": 1, "track_kernel_fat": 2, "track_split_kernel": 3}


def kernel_info(split, depth, kernel="track_kernel"):
    """gst_diag_kernel_info: {registers, local_bytes, blocks_per_sm} of one tracking-kernel instantiation."""
    r, l, b = C.c_int(0), C.c_int(0), C.c_int(0)
    gst._check(lib().gst_diag_kernel_info(int(split), int(depth), KERNEL_VARIANTS[kernel], C.byref(r), C.byref(l), C.byref(b)))
    return {"registers": r.value, "local_bytes": l.value, "blocks_per_sm": b.value}
