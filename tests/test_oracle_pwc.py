"""Pins for the mid-slice piece-wise-constant spin integrators of the oracle (section 4.1, (37) P:470-482; the
DKSKD / DKDSDKD orderings of P:742).

What fixes them (none of it a retyping of the oracle):
  * mid-plane orbit in a sector bend: all rotations are about y, so the scheme is the MIDPOINT rule for the
    scalar integral whose closed form is psi = -(1+G gamma)(hL + dasin) + hL; its error falls with ratio 4
    and is -1/2 of the trapezoid rule's (depth 1) at the same slicing -- the textbook relation;
  * uniform field on the design orbit: Omega is constant, so any slicing gives G gamma theta exactly;
  * a quadrupole: second-order convergence to brute-force integration of the lab-frame T-BMT equation along
    the Hamiltonian orbit, for both orderings;
  * the orbit does not know about the spin ordering: DKSKD, DKDSDKD and the trapezoid scheme leave the same
    orbit (half kicks add up, half maps compose).
"""
import math

import mpmath as mp
import numpy as np
import pytest
from scipy.integrate import solve_ivp

from paper_1501_03450_b200 import workloads as W
from test_oracle_spin import B200, BEAM200, GAMMA200, _tbmt_axis, fn5_particle, rhic_dipole, rhic_ir_quad, run

HALF, DKSKD = W.PWC_HALF_SLICE, W.PWC_DKSKD


def _midplane_case():
    e = rhic_dipole()
    L, h = float(e["L"]), float(e["h"])
    z, _ = fn5_particle()
    z = z.copy()
    z[3] = 0.0
    z[0], z[1] = 2e-2, 1.5e-3
    Pt = z[5]
    Pa = mp.sqrt(1 + 2 * mp.mpf(Pt) / B200 + mp.mpf(Pt) ** 2)
    exact_orbit = run([e], z, [0, 1, 0], split=W.SPLIT_BEND_KICK)
    dasin = mp.asin(mp.mpf(z[1]) / Pa) - mp.asin(mp.mpf(exact_orbit[1]) / Pa)
    psi = -(1 + mp.mpf(BEAM200["G"]) * mp.mpf(GAMMA200) * (1 + mp.mpf(B200) * mp.mpf(Pt))) * (mp.mpf(h) * L + dasin) \
        + mp.mpf(h) * L
    return e, z, psi


def _angle(out):
    """rotation angle about y that takes (1,0,0) to out[6:9]: S = (cos psi, 0, -sin psi)"""
    return mp.atan2(-mp.mpf(out[8]), mp.mpf(out[6]))


def test_midplane_bend_is_the_midpoint_rule_error_ratio_4_and_minus_half_of_trapezoid():
    e, z, psi = _midplane_case()
    wrap = lambda a: float((a + mp.pi) % (2 * mp.pi) - mp.pi)
    emid, etrap = {}, {}
    for n in (4, 8, 16, 32):
        emid[n] = wrap(_angle(run([e], z, [1.0, 0.0, 0.0], split=W.SPLIT_BEND_KICK, n_slices=n, depth=HALF)) - psi)
        etrap[n] = wrap(_angle(run([e], z, [1.0, 0.0, 0.0], split=W.SPLIT_BEND_KICK, n_slices=n, depth=1)) - psi)
    assert abs(emid[4]) > 1e-9
    for n in (4, 8, 16):
        assert 3.8 < emid[n] / emid[2 * n] < 4.2, emid
    for n in (8, 16, 32):
        assert -0.52 < emid[n] / etrap[n] < -0.48, (emid, etrap)


@pytest.mark.parametrize("kind", [HALF, DKSKD])
@pytest.mark.parametrize("split", [W.SPLIT_DRIFT_KICK, W.SPLIT_BEND_KICK])
def test_design_orbit_in_a_uniform_dipole_precesses_G_gamma_theta_for_any_slicing(kind, split):
    e = rhic_dipole()
    theta = float(e["h"]) * float(e["L"])
    psi = -BEAM200["G"] * GAMMA200 * theta
    errs = []
    for n in (1, 3, 8):
        out = run([e], np.zeros(6), [1.0, 0.0, 0.0], split=split, n_slices=n, depth=kind)
        errs.append(np.max(np.abs(out[6:] - [math.cos(psi), 0.0, -math.sin(psi)])))
        if split == W.SPLIT_BEND_KICK:                    # exact bend: the design orbit is kept, Omega is constant
            assert errs[-1] < 1e-13 and np.max(np.abs(out[:6])) < 1e-18
    # TEAPOT leaves the design orbit at second order in ds, and so does the spin
    assert split == W.SPLIT_BEND_KICK or (errs[0] < 1e-2 and errs[2] < errs[0] / 30), errs


@pytest.mark.parametrize("kind,split", [(HALF, W.SPLIT_MATRIX_KICK), (HALF, W.SPLIT_DRIFT_KICK), (DKSKD, W.SPLIT_DRIFT_KICK)])
def test_quadrupole_pwc_converges_to_tbmt_at_second_order(kind, split):
    e = rhic_ir_quad()
    L, k1 = float(e["L"]), float(e["kn"][0])
    z, S0 = fn5_particle()
    z = z.copy()
    z[0], z[2] = 8e-3, -6e-3
    G, b0 = BEAM200["G"], B200

    def rhs(s, y):
        X, Px, Y, Py, T, Pt = y[:6]
        S = y[6:9]
        P = math.sqrt(1 + 2 * Pt / b0 + Pt * Pt)
        Ps = math.sqrt(P * P - Px * Px - Py * Py)
        u = np.array([Px, Py, Ps]) / P
        gamma = GAMMA200 * (1 + b0 * Pt)
        b = np.array([k1 * Y, k1 * X, 0.0])
        dS = (P / Ps) * np.cross(_tbmt_axis(u, b, G, gamma, P), S)
        return [Px / Ps, -k1 * X, Py / Ps, k1 * Y, -(1 / b0 + Pt) / Ps + 1 / b0, 0.0, dS[0], dS[1], dS[2]]
    ref = solve_ivp(rhs, (0, L), np.concatenate([z, S0]), method="DOP853", rtol=1e-13, atol=1e-18).y[:, -1]
    err = [np.max(np.abs(run([e], z, S0, split=split, n_slices=n, depth=kind)[6:] - ref[6:])) for n in (4, 8, 16, 32)]
    assert err[0] > 1e-8
    assert all(3.6 < err[i] / err[i + 1] < 4.4 for i in range(3)), err


def test_the_orbit_does_not_depend_on_the_spin_ordering():
    e = rhic_ir_quad()
    d = rhic_dipole()
    z, S0 = fn5_particle()
    for split in (W.SPLIT_DRIFT_KICK, W.SPLIT_BEND_KICK, W.SPLIT_MATRIX_KICK):
        a = run([e, d], z, S0, split=split, n_slices=4, depth=1)[:6]
        for kind in (HALF, DKSKD):
            b = run([e, d], z, S0, split=split, n_slices=4, depth=kind)[:6]
            if kind == DKSKD and split != W.SPLIT_MATRIX_KICK:
                assert np.max(np.abs(a - b)) < 1e-16, (split, kind, a - b)      # half kicks add up, exact maps compose
            else:
                # two half maps of a split slice are not one slice map: second-order close (tiny for matrix-kick)
                assert np.max(np.abs(a[:4] - b[:4])) < (1e-9 if split == W.SPLIT_MATRIX_KICK else 1e-4)


def test_dkskd_and_half_slice_orderings_differ_at_second_order_only():
    e = rhic_ir_quad()
    z, S0 = fn5_particle()
    z = z.copy()
    z[0], z[2] = 8e-3, -6e-3
    diff = [np.max(np.abs(run([e], z, S0, split=W.SPLIT_DRIFT_KICK, n_slices=n, depth=HALF)[6:]
                          - run([e], z, S0, split=W.SPLIT_DRIFT_KICK, n_slices=n, depth=DKSKD)[6:])) for n in (4, 8, 16)]
    assert diff[0] > 1e-10 and 3.5 < diff[0] / diff[1] < 4.5 and 3.5 < diff[1] / diff[2] < 4.5, diff
