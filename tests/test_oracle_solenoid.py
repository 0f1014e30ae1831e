"""Pins for the solenoid of the oracle: body map (34), kinetic momentum in Omega (36), thin-pancake fringe spin
kick (40)  (section 3.7, section 4.4).

  * body orbit (34) against brute-force integration of Hamilton's equations of H_sol (33), typed from H;
  * symplectic (dual-number Jacobian), reversible;
  * the WHOLE element -- orbit, body spin precession with u-hat from the kinetic momentum, entrance and exit
    kicks (40) with their signs and magnitude (the factor 1/2 in FRONT of (40); the 1/2 inside its kinetic
    momentum changes the result by ~1e-9 here, below what this pin resolves) -- against the lab-frame Lorentz force + Thomas-BMT equation (4)
    through a Maxwellian soft-edge solenoid, B_z = b g(z), B_perp = -(b/2) g'(z) (x, y): converges linearly in
    the fringe length, and the Richardson limit is the oracle's result;
  * on the axis: no fringe kick, rotation about s-hat by -(1+G) b_0 L/((B rho)_o P).
The paper's solenoid (1.3 T, 2.1 m) and its 1.2 GeV proton are the test case.
"""
import math
import os

import numpy as np
import pytest
from scipy.integrate import solve_ivp

from oracle import oracle as O
from paper_1501_03450_b200 import workloads as W
from test_oracle_orbit import S_SYMP
from test_oracle_spin import _tbmt_axis

GLD = {}
for _line in open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "paper_solenoid_inputs.txt")):
    _f = _line.split("#")[0].split()
    if len(_f) == 2:
        GLD[_f[0]] = float(_f[1])
MASS = W.MASS_PROTON_EV
EKIN = GLD["proton_GeV"] * 1e9                      # P:729 "1.2 GeV proton" (kinetic energy reading, DESIGN R9)
GAMMA = 1.0 + EKIN / MASS
BETA = math.sqrt(1.0 - 1.0 / GAMMA ** 2)
BRHO = MASS * GAMMA * BETA / 299792458.0            # T m
KS = GLD["solenoid_B_T"] / BRHO                     # b_0/(B rho)_o for the 1.3 T solenoid
LSOL = GLD["solenoid_L_m"]
BEAM = W.beam(GAMMA)
G = BEAM["G"]
Z0 = np.array([1.2e-2, 2.0e-3, -0.9e-2, -1.5e-3, 0.0, 1.5e-3])
S0 = np.array([2.0, 10.0, 1.0]) / math.sqrt(105.0)


def run(elems, z, S=S0, n_slices=1, depth=1, prec=O.PREC_QUAD, split=W.SPLIT_MATRIX_KICK):
    st = np.zeros((9, 1))
    st[:6, 0] = z
    st[6:, 0] = S
    out, lost, _ = O.track(W.lattice(elems), BEAM, st, 1, split, n_slices, depth, prec=prec, threads=1)
    assert not lost[0]
    return out[:, 0]


def test_body_map_34_is_the_flow_of_H_sol_33():
    eta = KS / 2

    def rhs(s, y):
        X, Px, Y, Py, T, Pt = y
        kx, ky = Px + eta * Y, Py - eta * X                              # P - (e/p_o) A, A of (32)
        Ps = math.sqrt(1 + 2 * Pt / BETA + Pt * Pt - kx * kx - ky * ky)
        return [kx / Ps, eta * ky / Ps, ky / Ps, -eta * kx / Ps, -(1 / BETA + Pt) / Ps + 1 / BETA, 0.0]
    ref = solve_ivp(rhs, (0, LSOL), Z0, method="DOP853", rtol=1e-13, atol=1e-18).y[:, -1]
    for n in (1, 4):
        out = run([W.solenoid(LSOL, KS)], Z0, n_slices=n)
        assert np.max(np.abs(out[:4] - ref[:4])) < 2e-13, out[:4] - ref[:4]
        assert abs(out[4] - ref[4]) < 1e-13
    assert np.linalg.norm(ref[:4] - Z0[:4]) > 1e-3


def test_solenoid_map_is_symplectic_and_reversible():
    e = W.solenoid(LSOL, KS)
    J, _ = O.jacobian(W.lattice([e]), BEAM, Z0, W.SPLIT_MATRIX_KICK, 2)
    assert np.max(np.abs(J.T @ S_SYMP @ J - S_SYMP)) < 1e-12
    assert abs(J[0, 2]) > 1e-2                                           # the planes are coupled
    back = e.copy()
    back["L"] = -LSOL
    out = run([e, back], Z0, n_slices=4, depth=3)
    assert np.max(np.abs(out[:6] - Z0)) < 1e-16
    assert np.max(np.abs(out[6:] - S0)) < 1e-15


def _soft_solenoid(eps):
    """Lab-frame Lorentz force + T-BMT through B_z = b g(z), B_perp = -(b/2) g'(z)(x, y); g rises over
    [-eps/2, eps/2] and falls over [L - eps/2, L + eps/2] (smooth step).  Momenta in units of p_o."""
    b0 = KS
    Pt = Z0[5]
    P = math.sqrt(1 + 2 * Pt / BETA + Pt * Pt)
    gamma = GAMMA * (1 + BETA * Pt)

    def g(z):
        def step(t):
            t = min(max(t, 0.0), 1.0)
            return t * t * (3 - 2 * t), 6 * t * (1 - t) / eps
        a, da = step((z + eps / 2) / eps)
        c, dc = step((z - LSOL + eps / 2) / eps)
        return a - c, da - dc

    def rhs(z, y):
        x, yy = y[0], y[1]
        u = y[2:5]
        S = y[5:8]
        gz, dgz = g(z)
        b = np.array([-0.5 * b0 * dgz * x, -0.5 * b0 * dgz * yy, b0 * gz])
        dl = 1.0 / u[2]                                                  # path length per unit z
        du = dl * np.cross(u, b) / P
        dS = dl * np.cross(_tbmt_axis(u, b, G, gamma, P), S)
        return np.concatenate([[u[0] * dl, u[1] * dl], du, dS, [dl]])
    Ps = math.sqrt(P * P - Z0[1] ** 2 - Z0[3] ** 2)
    y0 = np.concatenate([[Z0[0], Z0[2]], [Z0[1] / P, Z0[3] / P, Ps / P], S0, [0.0]])
    pts = [-eps / 2, eps / 2, LSOL - eps / 2, LSOL + eps / 2]
    y = y0
    for a, c in zip(pts[:-1], pts[1:]):                                  # piecewise: the profile has kinks
        y = solve_ivp(rhs, (a, c), y, method="DOP853", rtol=1e-13, atol=1e-17).y[:, -1]
    orbit = np.array([y[0], P * y[2], y[1], P * y[3]])
    return orbit, y[5:8]


def test_whole_solenoid_is_the_hard_edge_limit_of_lorentz_force_plus_tbmt():
    out = run([W.solenoid(LSOL, KS)], Z0, n_slices=64, depth=4)
    soft = [_soft_solenoid(eps) for eps in (4e-3, 2e-3, 1e-3)]
    dS = [np.max(np.abs(s[1] - out[6:])) for s in soft]
    dO = [np.max(np.abs(s[0] - out[:4]) / np.array([1e-2, 1e-3, 1e-2, 1e-3])) for s in soft]
    assert 1.8 < dS[0] / dS[1] < 2.2 and 1.8 < dS[1] / dS[2] < 2.2, dS     # linear in the fringe length
    limS = 2 * soft[2][1] - soft[1][1]                                    # Richardson limit eps -> 0
    limO = 2 * soft[2][0] - soft[1][0]
    rot = np.linalg.norm(out[6:] - S0)
    assert rot > 0.3                                                      # a large rotation (about 40 degrees)
    assert np.max(np.abs(limS - out[6:])) < 2e-6, limS - out[6:]
    assert np.max(np.abs(limO - out[:4]) / np.array([1e-2, 1e-3, 1e-2, 1e-3])) < 1e-5, (limO - out[:4], dO)
    # sensitivity: the off-axis effects (fringe kicks of ~8 mrad each, transverse velocity) are three orders above
    # the tolerance -- the same particle on the axis ends up 1e-3 away
    on_axis = run([W.solenoid(LSOL, KS)], np.concatenate([[0, 0, 0, 0], Z0[4:]]), n_slices=64, depth=4)
    assert np.max(np.abs(on_axis[6:] - out[6:])) > 5e-4


def test_on_axis_particle_rotates_about_s_by_one_plus_G_times_the_field_integral():
    z = np.array([0.0, 0.0, 0.0, 0.0, 0.0, 1.5e-3])
    P = math.sqrt(1 + 2 * z[5] / BETA + z[5] ** 2)
    out = run([W.solenoid(LSOL, KS)], z, S=[1.0, 0.0, 0.0], n_slices=3, depth=1)
    ang = -(1 + G) * KS * LSOL / P
    assert np.max(np.abs(out[6:] - [math.cos(ang), math.sin(ang), 0.0])) < 1e-15
    assert np.max(np.abs(out[:4])) == 0.0


def test_romberg_orders_in_the_solenoid_body():
    ref = run([W.solenoid(LSOL, KS)], Z0, n_slices=256, depth=4)[6:]
    err = {(d, n): np.max(np.abs(run([W.solenoid(LSOL, KS)], Z0, n_slices=n, depth=d)[6:] - ref))
           for d in (1, 2) for n in (4, 8, 16)}
    assert 3.7 < err[1, 4] / err[1, 8] < 4.3 and 3.7 < err[1, 8] / err[1, 16] < 4.3, err
    assert err[2, 4] / err[2, 8] > 12 or err[2, 8] < 1e-13, err
