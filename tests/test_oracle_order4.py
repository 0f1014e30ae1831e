"""Pins for the fourth-order composition of the slice maps in the CPU oracle.

The paper only points to the literature for "higher-order versions of (27)", so nothing here can be a
printed value.  What fixes the composition S4(ds) = S2(x1 ds) S2(x0 ds) S2(x1 ds) is mathematics:
  * it converges to the exact flow of the element's Hamiltonian (brute-force ODE integration of (3)+(20),
    the closed-form sector bend (10)) with error ratio 16 per halving of the slice length, where the
    second-order maps give 4;
  * it is symplectic (dual-number Jacobian) and time-reversible;
  * an exact slice map (sector bend under bend-kick / matrix-kick) is left alone.
A wrong coefficient, a dropped sub-step or a sub-step taken with the wrong length breaks the order-4
ratios (the scheme falls back to order 2 or does not converge to the flow at all).
"""
import math

import numpy as np
import pytest
from scipy.integrate import solve_ivp

from oracle import oracle as O
from paper_1501_03450_b200 import workloads as W
from test_oracle_orbit import B0, BEAM, S_SYMP, Z_TEST, _hamilton_rhs, run

ORDER4 = {W.SPLIT_DRIFT_KICK: W.SPLIT_DRIFT_KICK_4, W.SPLIT_BEND_KICK: W.SPLIT_BEND_KICK_4,
          W.SPLIT_MATRIX_KICK: W.SPLIT_MATRIX_KICK_4}
Z_BIG = np.array([8e-3, 6e-4, -6e-3, 4e-4, 0.0, 2e-3])      # large amplitudes: truncation errors well above round-off


@pytest.mark.parametrize("k1", [0.3, -0.3])
@pytest.mark.parametrize("split", [W.SPLIT_DRIFT_KICK, W.SPLIT_MATRIX_KICK])
def test_quadrupole_order4_converges_to_the_hamiltonian_flow_with_ratio_16(k1, split):
    L = 1.83
    ref = solve_ivp(_hamilton_rhs(0.0, 0.0, k1, B0), (0, L), Z_BIG, method="DOP853", rtol=3e-14, atol=1e-20).y[:, -1]
    scale = np.array([1e-3, 1e-4, 1e-3, 1e-4])
    e4 = [np.max(np.abs(run([W.quad(L, k1)], Z_BIG, split=ORDER4[split], n_slices=n)[:4] - ref[:4]) / scale) for n in (1, 2, 4)]
    e2 = [np.max(np.abs(run([W.quad(L, k1)], Z_BIG, split=split, n_slices=n)[:4] - ref[:4]) / scale) for n in (1, 2, 4)]
    if split == W.SPLIT_DRIFT_KICK:
        assert 12 < e4[0] / e4[1] < 20 and 13 < e4[1] / e4[2] < 19, (e4, e2)
        assert 3.5 < e2[1] / e2[2] < 4.5, e2
        assert e4[2] < 0.1 * e2[2]                 # the triple jump has a large error constant; its gain grows with n
    else:
        # matrix-kick: only the small nonlinear kick (25) is split off, so both errors are tiny and the
        # asymptotic ratios set in one halving later
        e4.append(np.max(np.abs(run([W.quad(L, k1)], Z_BIG, split=ORDER4[split], n_slices=8)[:4] - ref[:4]) / scale))
        e2.append(np.max(np.abs(run([W.quad(L, k1)], Z_BIG, split=split, n_slices=8)[:4] - ref[:4]) / scale))
        assert 10 < e4[1] / e4[2] < 20 and 13 < e4[2] / e4[3] < 19, (e4, e2)
        assert 3.0 < e2[2] / e2[3] < 4.5, e2
        assert all(a < b for a, b in zip(e4, e2))


def test_teapot_bend_order4_converges_to_the_exact_bend_with_ratio_16():
    e = W.sbend(9.45, math.radians(2.225), 1.002)
    exact = run([e], Z_BIG, split=W.SPLIT_BEND_KICK)[:6]
    scale = np.array([1e-3, 1e-4, 1e-3, 1e-4, 1e-6, 1.0])
    e4 = [np.max(np.abs(run([e], Z_BIG, split=W.SPLIT_DRIFT_KICK_4, n_slices=n)[:6] - exact) / scale) for n in (1, 2, 4, 8)]
    e2 = [np.max(np.abs(run([e], Z_BIG, split=W.SPLIT_DRIFT_KICK, n_slices=n)[:6] - exact) / scale) for n in (1, 2, 4, 8)]
    r4 = [e4[i] / e4[i + 1] for i in range(3)]
    assert all(13 < r < 19 for r in r4), (e4, r4)
    assert all(3.7 < e2[i] / e2[i + 1] < 4.3 for i in range(3)), e2


def test_sextupole_order4_against_ode():
    L = 0.75
    kn2, ks2 = 1.2, 0.3                                      # (28): By + i Bx = (b3 + i a3)(X + iY)^2

    def rhs(s, z):
        X, Px, Y, Py, T, Pt = z
        Ps = math.sqrt(1 + 2 * Pt / B0 + Pt * Pt - Px * Px - Py * Py)
        by = kn2 * (X * X - Y * Y) - ks2 * 2 * X * Y
        bx = kn2 * 2 * X * Y + ks2 * (X * X - Y * Y)
        return [Px / Ps, -by, Py / Ps, bx, 1 / B0 - (1 / B0 + Pt) / Ps, 0.0]
    ref = solve_ivp(rhs, (0, L), Z_BIG, method="DOP853", rtol=3e-14, atol=1e-20).y[:, -1]
    e = W.multipole(L, kn=(0.0, kn2, 0.0, 0.0), ks=(0.0, ks2, 0.0, 0.0))
    e4 = [np.max(np.abs(run([e], Z_BIG, split=W.SPLIT_BEND_KICK_4, n_slices=n)[:4] - ref[:4])) for n in (1, 2, 4)]
    e2 = [np.max(np.abs(run([e], Z_BIG, split=W.SPLIT_BEND_KICK, n_slices=n)[:4] - ref[:4])) for n in (1, 2, 4)]
    assert 12 < e4[0] / e4[1] < 20 and 12 < e4[1] / e4[2] < 20, (e4, e2)
    assert e4[2] < 0.1 * e2[2]


def test_exact_sector_bend_is_untouched_by_the_composition():
    e = W.sbend(9.45, math.radians(2.225), 1.002)
    for s2, s4 in ((W.SPLIT_BEND_KICK, W.SPLIT_BEND_KICK_4), (W.SPLIT_MATRIX_KICK, W.SPLIT_MATRIX_KICK_4)):
        a = run([e], Z_TEST, split=s2, n_slices=4, depth=3)
        b = run([e], Z_TEST, split=s4, n_slices=4, depth=3)
        assert np.array_equal(a, b)


ELEMENTS4 = {
    "sbend_teapot": (W.sbend(9.45, math.radians(2.225), 1.002), W.SPLIT_DRIFT_KICK_4),
    "quad_mk_f": (W.quad(1.83, 0.09), W.SPLIT_MATRIX_KICK_4),
    "quad_mk_d": (W.quad(1.83, -0.09), W.SPLIT_MATRIX_KICK_4),
    "quad_dk": (W.quad(1.83, 0.09), W.SPLIT_DRIFT_KICK_4),
    "sext_dk": (W.multipole(0.75, kn=(0.0, 1.2, 0.0, 0.0), ks=(0.0, 0.3, 0.0, 0.0)), W.SPLIT_MATRIX_KICK_4),
}


@pytest.mark.parametrize("name", sorted(ELEMENTS4))
def test_order4_maps_are_symplectic_and_reversible(name):
    e, split = ELEMENTS4[name]
    J, _ = O.jacobian(W.lattice([e]), BEAM, Z_TEST, split, 2)
    assert np.max(np.abs(J.T @ S_SYMP @ J - S_SYMP)) < 1e-12
    back = e.copy()
    back["L"] = -float(e["L"])
    S0 = np.array([2.0, 10.0, 1.0]) / math.sqrt(105.0)
    out = run([e, back], Z_TEST, split=split, n_slices=4, depth=3, S=S0)
    assert np.max(np.abs(out[:6] - Z_TEST)) < 1e-17
    assert np.max(np.abs(out[6:] - S0)) < 1e-15
