"""Pins for the thin-fringe spin kick (41) P:557-563 in the oracle (the multipole/dipole part).

(41) is the thin-fringe, lowest-order limit of the Thomas-BMT precession in the fringe's LONGITUDINAL field.
The pin integrates the lab-frame T-BMT equation (4) through a soft fringe of length ell whose field derives
from the scalar potential g(z) psi(x, y), psi = b_m Im (x+iy)^m / m + a_m Re (x+iy)^m / m  (so that inside,
g = 1, B_y + i B_x = (b_m + i a_m)(x+iy)^(m-1), the convention of (28)):  B_perp = g grad psi,  B_z = g' psi.
The transverse field turns the spin by an angle proportional to ell, so the result converges LINEARLY in ell to
the oracle's kick.  A wrong sign, a missing 1/m, sin and cos swapped, 1+G gamma in place of 1+G, or a wrong
entrance/exit sign all fail it.
"""
import math

import numpy as np
import pytest
from scipy.integrate import solve_ivp

from paper_1501_03450_b200 import workloads as W
from test_oracle_spin import BEAM200, GAMMA200, _tbmt_axis, run

G = BEAM200["G"]
S0 = np.array([2.0, 10.0, 1.0]) / math.sqrt(105.0)


def _psi_and_grad(x, y, k0, kn, ks):
    w = complex(x, y)
    psi = k0 * y
    gx, gy = 0.0, k0
    for m in range(2, 6):
        b, a = kn[m - 2], ks[m - 2]
        wm, wm1 = w ** m, w ** (m - 1)
        psi += (b * wm.imag + a * wm.real) / m
        # d/dx w^m = m w^(m-1),  d/dy w^m = i m w^(m-1)
        gx += b * wm1.imag + a * wm1.real
        gy += b * wm1.real - a * wm1.imag
    return psi, gx, gy


def _soft_fringe_spin(x, y, k0, kn, ks, ell, entering):
    """T-BMT along the straight line (x, y) = const, momentum along z, through a smooth-step fringe of length ell."""
    psi, gx, gy = _psi_and_grad(x, y, k0, kn, ks)
    u = np.array([0.0, 0.0, 1.0])

    def g(z):
        t = z / ell
        s = t * t * (3 - 2 * t)
        ds = 6 * t * (1 - t) / ell
        return (s, ds) if entering else (1 - s, -ds)

    def rhs(z, S):
        gz, dgz = g(z)
        b = np.array([gz * gx, gz * gy, dgz * psi])
        return np.cross(_tbmt_axis(u, b, G, GAMMA200, 1.0), S)
    return solve_ivp(rhs, (0, ell), S0, method="DOP853", rtol=1e-13, atol=1e-16).y[:, -1]


CASES = {
    "dipole": dict(k0=0.0115, kn=(0, 0, 0, 0), ks=(0, 0, 0, 0)),
    "quad": dict(k0=0.0, kn=(0.6, 0, 0, 0), ks=(0, 0, 0, 0)),
    "skew_quad": dict(k0=0.0, kn=(0, 0, 0, 0), ks=(0.5, 0, 0, 0)),
    "sextupole": dict(k0=0.0, kn=(0, 35.0, 0, 0), ks=(0, -20.0, 0, 0)),
    "mixed": dict(k0=0.02, kn=(0.3, 12.0, -300.0, 8000.0), ks=(0.1, -7.0, 200.0, -5000.0)),
}


@pytest.mark.parametrize("name", sorted(CASES))
@pytest.mark.parametrize("sign", [+1.0, -1.0])
def test_fringe_kick_is_the_thin_limit_of_tbmt_in_the_longitudinal_fringe_field(name, sign):
    c = CASES[name]
    x, y = 2.3e-2, -1.7e-2
    z = np.array([x, 0.0, y, 0.0, 0.0, 0.0])
    out = run([W.fringe(sign, c["k0"], c["kn"], c["ks"])], z, S0)
    assert np.array_equal(out[:6], z)                                        # orbit-transparent
    soft = [_soft_fringe_spin(x, y, c["k0"], c["kn"], c["ks"], ell, sign > 0) for ell in (1e-3, 1e-4, 1e-5)]
    d = [np.max(np.abs(sf - out[6:])) for sf in soft]
    assert 7 < d[0] / d[1] < 13 and 7 < d[1] / d[2] < 13, d                  # linear in the fringe length
    limit = (10 * soft[2] - soft[1]) / 9                                     # Richardson: the ell -> 0 limit
    kick = np.linalg.norm(out[6:] - S0)
    assert kick > 1e-4 and np.max(np.abs(limit - out[6:])) < 1e-4 * kick, (kick, limit - out[6:])


def test_entrance_and_exit_kicks_cancel_at_the_same_point_and_vanish_in_the_midplane_of_normal_magnets():
    z = np.array([2e-2, 0.0, -1e-2, 0.0, 0.0, 0.0])
    kn = (0.3, 12.0, -300.0, 8000.0)
    out = run([W.fringe(+1.0, 0.02, kn), W.fringe(-1.0, 0.02, kn)], z, S0)
    assert np.max(np.abs(out[6:] - S0)) < 1e-16
    mid = np.array([2e-2, 0.0, 0.0, 0.0, 0.0, 0.0])                          # Y = 0: sin(m phi) = 0 for every m
    out = run([W.fringe(+1.0, 0.02, kn)], mid, S0)
    assert np.max(np.abs(out[6:] - S0)) < 1e-18


def test_quadrupole_fringe_kick_value():
    # (41), m = 2: omega = -(1+G) k1 X Y about s-hat; a vertical spin is unchanged, a radial one turns towards y
    k1, X, Y = 0.6, 2e-2, -1e-2
    out = run([W.fringe(+1.0, 0.0, (k1, 0, 0, 0))], np.array([X, 0.0, Y, 0.0, 0.0, 0.0]), [1.0, 0.0, 0.0])
    om = -(1 + G) * k1 * X * Y
    assert np.max(np.abs(out[6:] - [math.cos(om), math.sin(om), 0.0])) < 1e-16
