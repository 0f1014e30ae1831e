"""ctypes front end of the CPU oracle (TEST INFRASTRUCTURE -- see gst_oracle.hpp).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It takes the neutral lattice description produced by the seeded workload
generators (a numpy structured array with the fields of ELEM_DTYPE) and calls liboracle.so.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

DRIFT, SBEND, QUAD, MULTIPOLE, THINMULT, RFCAV, SNAKE, MARKER, FRINGE, SOLENOID, RBEND = range(11)
SPLIT_DRIFT_KICK, SPLIT_BEND_KICK, SPLIT_MATRIX_KICK = range(3)
PREC_DOUBLE, PREC_LONG_DOUBLE, PREC_QUAD = range(3)


class Element(C.Structure):
    _fields_ = [("type", C.c_int32), ("slice_mult", C.c_int32), ("L", C.c_double), ("h", C.c_double),
                ("k0", C.c_double), ("kn", C.c_double * 4), ("ks", C.c_double * 4),
                ("volt_eV", C.c_double), ("harmonic", C.c_double), ("phi_s", C.c_double), ("sign", C.c_double),
                ("snake_mu", C.c_double), ("snake_phi", C.c_double)]


class Beam(C.Structure):
    _fields_ = [("G", C.c_double), ("mass_eV", C.c_double), ("gamma0", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        dp = C.POINTER(C.c_double)
        _lib.orc_track.restype = C.c_int
        _lib.orc_track.argtypes = [C.POINTER(Element), C.c_size_t, C.POINTER(Beam)] + [dp] * 9 + [
            C.POINTER(C.c_uint8), C.c_size_t, C.c_int64, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, dp]
        _lib.orc_jacobian.restype = C.c_int
        _lib.orc_jacobian.argtypes = [C.POINTER(Element), C.c_size_t, C.POINTER(Beam), dp, C.c_int, C.c_int,
                                      C.c_double, dp, dp]
        _lib.orc_romberg.restype = C.c_int
        _lib.orc_romberg.argtypes = [dp, C.c_int, C.c_double, C.c_int, C.c_int, dp]
        _lib.orc_omega.restype = C.c_int
        _lib.orc_omega.argtypes = [C.POINTER(Element), C.POINTER(Beam), dp, dp]
        _lib.orc_polarization.restype = None
        _lib.orc_polarization.argtypes = [dp, dp, dp, C.POINTER(C.c_uint8), C.c_size_t, dp, C.POINTER(C.c_int64)]
        _lib.orc_emittance.restype = None
        _lib.orc_emittance.argtypes = [dp, dp, dp, dp, C.POINTER(C.c_uint8), C.c_size_t, dp]
    return _lib


def _elements(lattice):
    """numpy structured array (workload ELEM_DTYPE) -> ctypes array of the oracle's own struct."""
    arr = (Element * len(lattice))()
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


def _beam(beam):
    return Beam(float(beam["G"]), float(beam["mass_eV"]), float(beam["gamma0"]))


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def default_threads():
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def track(lattice, beam, state, n_turns, split, n_slices, depth, prec=PREC_LONG_DOUBLE, threads=None,
          lost=None, gamma0=None):
    """state: float64 array [9, n] (X,Px,Y,Py,T,Pt,Sx,Sy,Ss).  Returns (new_state, lost, gamma0_after)."""
    st = np.array(state, dtype=np.float64, order="C", copy=True)
    assert st.ndim == 2 and st.shape[0] == 9
    n = st.shape[1]
    lost = np.zeros(n, dtype=np.uint8) if lost is None else np.array(lost, dtype=np.uint8, copy=True)
    g0 = C.c_double(float(beam["gamma0"]) if gamma0 is None else float(gamma0))
    els = _elements(lattice)
    b = _beam(beam)
    rows = [np.ascontiguousarray(st[i]) for i in range(9)]
    rc = lib().orc_track(els, len(lattice), C.byref(b), *[_dp(r) for r in rows],
                         lost.ctypes.data_as(C.POINTER(C.c_uint8)), n, int(n_turns), int(split), int(n_slices),
                         int(depth), int(prec), int(threads or default_threads()), C.byref(g0))
    if rc != 0:
        raise ValueError("oracle: invalid arguments (rc=%d)" % rc)
    return np.stack(rows), lost, g0.value


def jacobian(lattice, beam, z0, split, n_slices, circumference=None):
    """One pass through `lattice` from z0: returns (J[6,6], z_f).  Dual numbers through the same code."""
    els = _elements(lattice)
    b = _beam(beam)
    z0 = np.ascontiguousarray(z0, dtype=np.float64)
    J = np.zeros(36)
    zf = np.zeros(6)
    Cc = float(sum(float(e["L"]) for e in lattice)) if circumference is None else float(circumference)
    rc = lib().orc_jacobian(els, len(lattice), C.byref(b), _dp(z0), int(split), int(n_slices), Cc, _dp(J), _dp(zf))
    if rc != 0:
        raise ValueError("oracle jacobian rc=%d" % rc)
    return J.reshape(6, 6), zf


def romberg(Om, ds, depth, prec=PREC_DOUBLE):
    Om = np.ascontiguousarray(Om, dtype=np.float64)
    N = Om.shape[0] - 1
    q = np.zeros(4)
    rc = lib().orc_romberg(_dp(Om), N, float(ds), int(depth), int(prec), _dp(q))
    if rc != 0:
        raise ValueError("oracle romberg rc=%d" % rc)
    return q


def omega(element, beam, z):
    els = _elements([element])
    b = _beam(beam)
    z = np.ascontiguousarray(z, dtype=np.float64)
    out = np.zeros(3)
    rc = lib().orc_omega(els, C.byref(b), _dp(z), _dp(out))
    if rc != 0:
        raise ValueError("oracle omega rc=%d" % rc)
    return out


def polarization(state, lost=None):
    st = np.ascontiguousarray(state, dtype=np.float64)
    n = st.shape[1]
    out = np.zeros(4)
    nl = C.c_int64(0)
    lp = None if lost is None else np.ascontiguousarray(lost, dtype=np.uint8).ctypes.data_as(C.POINTER(C.c_uint8))
    rows = [np.ascontiguousarray(st[i]) for i in (6, 7, 8)]
    lib().orc_polarization(*[_dp(r) for r in rows], lp, n, _dp(out), C.byref(nl))
    return out, nl.value


def emittance(state, lost=None):
    st = np.ascontiguousarray(state, dtype=np.float64)
    n = st.shape[1]
    out = np.zeros(2)
    lp = None if lost is None else np.ascontiguousarray(lost, dtype=np.uint8).ctypes.data_as(C.POINTER(C.c_uint8))
    rows = [np.ascontiguousarray(st[i]) for i in range(4)]
    lib().orc_emittance(*[_dp(r) for r in rows], lp, n, _dp(out))
    return out
