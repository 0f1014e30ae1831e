"""Thin ctypes binding over the C-ABI library (include/gst.h).  Argument marshalling only: every
step of the hot path runs in the CUDA kernels of libgst.so.  PyTorch supplies device memory and
streams.  There is no CPU fallback: if libgst.so is missing or no CUDA device is present, the
calls raise.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgst.so")

OK, EINVAL, ENOMEM, ECUDA, ESTATE = range(5)
DRIFT, SBEND, QUAD, MULTIPOLE, THINMULT, RFCAV, SNAKE, MARKER, FRINGE, SOLENOID, RBEND = range(11)
SPLIT_DRIFT_KICK, SPLIT_BEND_KICK, SPLIT_MATRIX_KICK = range(3)


class GstError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("gst status %d: %s" % (status, msg))
        self.status = status


class gst_element(C.Structure):
    _fields_ = [("type", C.c_int32), ("slice_mult", C.c_int32), ("L", C.c_double), ("h", C.c_double),
                ("k0", C.c_double), ("kn", C.c_double * 4), ("ks", C.c_double * 4),
                ("volt_eV", C.c_double), ("harmonic", C.c_double), ("phi_s", C.c_double), ("sign", C.c_double),
                ("snake_mu", C.c_double), ("snake_phi", C.c_double)]


class gst_beam(C.Structure):
    _fields_ = [("G", C.c_double), ("mass_eV", C.c_double), ("gamma0", C.c_double)]


_lib = None
_dp = C.POINTER(C.c_double)

EXPORTS = ["gst_lattice_create", "gst_lattice_destroy", "gst_lattice_steps_per_turn", "gst_bunch_init",
           "gst_bunch_destroy", "gst_track", "gst_polarization", "gst_emittance", "gst_bunch_lost",
           "gst_bunch_reference", "gst_bunch_set_reference", "gst_track_host", "gst_last_error",
           "gst_bunch_set_launch", "gst_bunch_status", "gst_track_pwc", "gst_bunch_last_kernel",
           "gst_polarization_noalloc", "gst_moments", "gst_moments_finish"]
NOALLOC_MAX_PARTICLES = 1 << 20
MOMENTS_LEN = 20
LAUNCH_AUTO, LAUNCH_STATIC, LAUNCH_LEAN = 0, 1, 2


def lib():
    """Load libgst.so (built by paper_1501_03450_b200/build.py).  Fails loudly when it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libgst.so not built: run `python -m paper_1501_03450_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp = C.c_void_p
        L.gst_last_error.restype = C.c_char_p
        L.gst_lattice_create.argtypes = [C.POINTER(gst_element), C.c_size_t, C.POINTER(gst_beam), C.POINTER(vp)]
        L.gst_lattice_destroy.argtypes = [vp]
        L.gst_lattice_destroy.restype = None
        L.gst_lattice_steps_per_turn.argtypes = [vp, C.c_int]
        L.gst_lattice_steps_per_turn.restype = C.c_int64
        L.gst_bunch_init.argtypes = [vp] * 9 + [C.c_size_t, C.POINTER(vp)]
        L.gst_bunch_destroy.argtypes = [vp]
        L.gst_bunch_destroy.restype = None
        L.gst_track.argtypes = [vp, vp, C.c_int64, C.c_int, C.c_int, C.c_int, vp]
        L.gst_track_pwc.argtypes = [vp, vp, C.c_int64, C.c_int, C.c_int, C.c_int, vp]
        L.gst_track_pwc.restype = C.c_int
        L.gst_bunch_last_kernel.argtypes = [vp]
        L.gst_bunch_last_kernel.restype = C.c_char_p
        L.gst_polarization.argtypes = [vp, vp, _dp, C.POINTER(C.c_int64)]
        L.gst_emittance.argtypes = [vp, vp, _dp]
        L.gst_moments.argtypes = [vp, vp, _dp]
        L.gst_moments_finish.argtypes = [_dp, _dp, _dp, C.POINTER(C.c_int64)]
        L.gst_bunch_lost.argtypes = [vp, vp, C.POINTER(C.c_uint8)]
        L.gst_bunch_reference.argtypes = [vp, _dp, C.POINTER(C.c_int64)]
        L.gst_bunch_set_reference.argtypes = [vp, C.POINTER(gst_beam), C.c_int64]
        L.gst_track_host.argtypes = [vp, C.POINTER(_dp), C.c_size_t, C.c_int64, C.c_int, C.c_int, C.c_int, _dp,
                                     C.POINTER(C.c_int64)]
        L.gst_polarization_noalloc.argtypes = [vp, vp, vp, vp, C.c_size_t, vp, vp]
        L.gst_polarization_noalloc.restype = C.c_int
        L.gst_bunch_set_launch.argtypes = [vp, C.c_int]
        L.gst_bunch_status.argtypes = [vp, vp]
        for name in ("gst_lattice_create", "gst_bunch_init", "gst_track", "gst_polarization", "gst_emittance",
                     "gst_bunch_lost", "gst_bunch_reference", "gst_bunch_set_reference", "gst_track_host",
                     "gst_bunch_set_launch", "gst_bunch_status", "gst_moments", "gst_moments_finish"):
            getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def _check(status):
    if status != OK:
        raise GstError(status, lib().gst_last_error().decode())


def _elements(lattice):
    arr = (gst_element * len(lattice))()
    for i, e in enumerate(lattice):
        a = arr[i]
        a.type = int(e["type"]); a.slice_mult = int(e["slice_mult"])
        a.L = float(e["L"]); a.h = float(e["h"]); a.k0 = float(e["k0"])
        for k in range(4):
            a.kn[k] = float(e["kn"][k]); a.ks[k] = float(e["ks"][k])
        a.volt_eV = float(e["volt_eV"]); a.harmonic = float(e["harmonic"])
        a.phi_s = float(e["phi_s"]); a.sign = float(e["sign"])
        a.snake_mu = float(e["snake_mu"]); a.snake_phi = float(e["snake_phi"])
    return arr


def _host_ptr(a):
    if isinstance(a, np.ndarray):
        assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
        return a.ctypes.data, a.size
    assert not a.is_cuda and a.is_contiguous() and a.element_size() == 8
    return a.data_ptr(), a.numel()


class Lattice:
    """gst_lattice_create / gst_lattice_destroy."""

    def __init__(self, lattice, beam):
        self._h = C.c_void_p()
        els = _elements(lattice)
        b = gst_beam(float(beam["G"]), float(beam["mass_eV"]), float(beam["gamma0"]))
        _check(lib().gst_lattice_create(els, len(lattice), C.byref(b), C.byref(self._h)))

    def steps_per_turn(self, n_slices):
        return int(lib().gst_lattice_steps_per_turn(self._h, int(n_slices)))

    def track_host(self, host_state, n_turns, split, n_slices, depth):
        """gst_track_host: host_state = nine 1-D float64 CPU arrays/tensors, updated in place."""
        ptrs = (_dp * 9)()
        n = None
        for i, a in enumerate(host_state):
            addr, ln = _host_ptr(a)
            n = ln if n is None else n
            assert ln == n
            ptrs[i] = C.cast(addr, _dp)
        pol = (C.c_double * 4)()
        lost = C.c_int64(0)
        _check(lib().gst_track_host(self._h, ptrs, n, int(n_turns), int(split), int(n_slices), int(depth), pol,
                                    C.byref(lost)))
        return np.array(pol[:]), lost.value

    def close(self):
        if self._h:
            lib().gst_lattice_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Bunch:
    """gst_bunch_init over a [9, n] float64 CUDA tensor (rows X,Px,Y,Py,T,Pt,Sx,Sy,Ss) or nine tensors."""

    def __init__(self, state):
        import torch
        if isinstance(state, torch.Tensor):
            assert state.is_cuda and state.dtype == torch.float64 and state.dim() == 2 and state.shape[0] == 9
            assert state.is_contiguous()
            rows = [state[i] for i in range(9)]
        else:
            rows = list(state)
            for r in rows:
                assert r.is_cuda and r.dtype == torch.float64 and r.is_contiguous()
        self._keep = (state, rows)                      # the library borrows the memory
        self.n = rows[0].numel()
        self._h = C.c_void_p()
        _check(lib().gst_bunch_init(*[C.c_void_p(r.data_ptr()) for r in rows], self.n, C.byref(self._h)))

    @staticmethod
    def _stream(stream):
        import torch
        s = torch.cuda.current_stream() if stream is None else stream
        return C.c_void_p(s.cuda_stream)

    def track(self, lattice, n_turns, split, n_slices, depth, stream=None):
        _check(lib().gst_track(self._h, lattice._h, int(n_turns), int(split), int(n_slices), int(depth),
                               self._stream(stream)))

    def track_pwc(self, lattice, n_turns, split, n_slices, order, stream=None):
        """gst_track_pwc; `order` is workloads.PWC_HALF_SLICE (0) or workloads.PWC_DKSKD (-1)."""
        _check(lib().gst_track_pwc(self._h, lattice._h, int(n_turns), int(split), int(n_slices),
                                   0 if int(order) == 0 else 1, self._stream(stream)))

    def last_kernel(self):
        return lib().gst_bunch_last_kernel(self._h).decode()

    def set_launch(self, mode):
        """gst_bunch_set_launch: LAUNCH_AUTO (default), LAUNCH_STATIC (never the rotating launch) or LAUNCH_LEAN (nor the
        small-bunch kernel variant)."""
        _check(lib().gst_bunch_set_launch(self._h, int(mode)))

    def status(self, stream=None):
        """gst_bunch_status: synchronise and raise GstError(ECUDA) if a launch on this bunch failed."""
        _check(lib().gst_bunch_status(self._h, self._stream(stream)))

    def polarization(self, stream=None):
        out = (C.c_double * 4)()
        lost = C.c_int64(0)
        _check(lib().gst_polarization(self._h, self._stream(stream), out, C.byref(lost)))
        return np.array(out[:]), lost.value

    def emittance(self, stream=None):
        out = (C.c_double * 2)()
        _check(lib().gst_emittance(self._h, self._stream(stream), out))
        return np.array(out[:])

    def moments(self, stream=None):
        """The shard's additive record (gst_moments): sum it over the shards, then moments_finish()."""
        out = (C.c_double * MOMENTS_LEN)()
        _check(lib().gst_moments(self._h, self._stream(stream), out))
        return np.array(out[:])

    def lost(self, stream=None):
        out = np.zeros(max(self.n, 1), dtype=np.uint8)
        _check(lib().gst_bunch_lost(self._h, self._stream(stream), out.ctypes.data_as(C.POINTER(C.c_uint8))))
        return out[:self.n]

    def reference(self):
        g = C.c_double(0)
        t = C.c_int64(0)
        _check(lib().gst_bunch_reference(self._h, C.byref(g), C.byref(t)))
        return g.value, t.value

    def set_reference(self, beam, turn=0):
        b = gst_beam(float(beam["G"]), float(beam["mass_eV"]), float(beam["gamma0"]))
        _check(lib().gst_bunch_set_reference(self._h, C.byref(b), int(turn)))

    def close(self):
        if self._h:
            lib().gst_bunch_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def moments_finish(record):
    """gst_moments_finish: (polarization {Px, Py, Ps, |P|}, emittances {eps_x, eps_y}, particles counted) of a record
    of Bunch.moments() or of a component-wise sum of such records.  Host arithmetic in the library; needs no GPU."""
    rec = np.ascontiguousarray(record, dtype=np.float64)
    assert rec.shape == (MOMENTS_LEN,)
    pol, exy, alive = (C.c_double * 4)(), (C.c_double * 2)(), C.c_int64(0)
    _check(lib().gst_moments_finish(rec.ctypes.data_as(_dp), pol, exy, C.byref(alive)))
    return np.array(pol[:]), np.array(exy[:]), alive.value


def polarization_noalloc(sx, sy, ss, lost, out, stream=None):
    """gst_polarization_noalloc: sx, sy, ss float64 CUDA tensors of n elements, lost a uint8 CUDA tensor or None, out a
    float64 CUDA tensor of 5 elements that receives {Px, Py, Ps, |P|, counted}.  Asynchronous; allocates nothing."""
    import torch
    n = sx.numel()
    for t in (sx, sy, ss):
        assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and t.numel() == n
    assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() >= 5
    lp = None
    if lost is not None:
        assert lost.is_cuda and lost.dtype == torch.uint8 and lost.is_contiguous() and lost.numel() == n
        lp = C.c_void_p(lost.data_ptr())
    s = torch.cuda.current_stream() if stream is None else stream
    _check(lib().gst_polarization_noalloc(C.c_void_p(sx.data_ptr()), C.c_void_p(sy.data_ptr()), C.c_void_p(ss.data_ptr()),
                                          lp, n, C.c_void_p(out.data_ptr()), C.c_void_p(s.cuda_stream)))
