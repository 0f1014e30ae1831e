"""Pins for the SPIN part of the CPU oracle (no GPU, no CUDA path involved).

The strongest pins integrate the Thomas-BMT equation in its original lab-frame, time-domain form
(4) P:87 by brute force (DOP853) -- in Cartesian lab coordinates for the sector bend, so that
neither the (1+hX)/Ps factor nor the frame term h*y-hat of (6b) is assumed -- and compare with the
oracle's trapezoid/Romberg quaternion scheme at fine slicing.  The others are closed forms,
invariants and the convergence orders the paper reports.
"""
import math
import os

import mpmath as mp
import numpy as np
import pytest
from scipy.integrate import solve_ivp
from scipy.spatial.transform import Rotation

from oracle import oracle as O
from paper_1501_03450_b200 import workloads as W

mp.mp.dps = 40
GOLD = os.path.join(os.path.dirname(__file__), "golden", "paper_fig7_inputs.txt")


def golden():
    out = {}
    for line in open(GOLD):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = float(line[1])
    return out


GLD = golden()
MP_GEV = W.MASS_PROTON_EV / 1e9
GAMMA200 = GLD["energy_GeV"] / MP_GEV                      # "200 GeV protons" read as total energy
BEAM200 = W.beam(GAMMA200)
B200 = W.beta_of_gamma(GAMMA200)
BRHO200 = math.sqrt(GLD["energy_GeV"] ** 2 - MP_GEV ** 2) / 0.299792458   # T m


def fn5_particle():
    """Footnote 5."""
    z = np.array([GLD["X_m"], GLD["Px_rad"], GLD["Y_m"], GLD["Py_rad"], GLD["T_m"],
                  float(W.pt_of_delta(GLD["delta"], B200))])
    S = np.array([2.0, 10.0, 1.0]) / math.sqrt(105.0)
    return z, S


def rhic_dipole():
    return W.sbend(GLD["dipole_L_m"], math.radians(GLD["dipole_angle_deg"]))


def rhic_ir_quad():
    return W.quad(GLD["quad_L_m"], GLD["quad_gradient_T_per_m"] / BRHO200)


def run(elems, z, S, split=W.SPLIT_MATRIX_KICK, n_slices=1, depth=1, prec=O.PREC_QUAD, beam=BEAM200, turns=1):
    st = np.zeros((9, 1))
    st[:6, 0] = z
    st[6:, 0] = S
    out, lost, _ = O.track(W.lattice(elems), beam, st, turns, split, n_slices, depth, prec=prec, threads=1)
    assert not lost[0]
    return out[:, 0]


def test_golden_inputs_are_self_consistent():
    _, S = fn5_particle()
    assert np.max(np.abs(S - [GLD["Sx"], GLD["Sy"], GLD["Ss"]])) < 6e-5          # P:654 prints 4 digits
    B = BRHO200 * math.radians(GLD["dipole_angle_deg"]) / GLD["dipole_L_m"]
    assert abs(B - GLD["dipole_B_T"]) < 0.05                                       # "B ~ 2.75 T" P:664


# ---------------------------------------------------------------------------------------------
# brute force: lab-frame T-BMT (4) in a uniform vertical field vs the oracle's sector bend
# ---------------------------------------------------------------------------------------------
def _tbmt_axis(u, b, G, gamma, P):
    """-(1/P)[(1+G gamma) b - G(gamma-1)(u.b)u]: dS/dl = W x S, from (4) with dl = beta c dt, p = P p_o."""
    return -((1 + G * gamma) * b - G * (gamma - 1) * np.dot(u, b) * u) / P


def test_sector_bend_spin_equals_lab_frame_tbmt_integration():
    e = rhic_dipole()
    L, h, k0 = float(e["L"]), float(e["h"]), float(e["k0"])
    z, S0 = fn5_particle()
    G = BEAM200["G"]
    X, Px, Y, Py, T, Pt = z
    P = math.sqrt(1 + 2 * Pt / B200 + Pt * Pt)
    Ps = math.sqrt(P * P - Px * Px - Py * Py)
    gamma = GAMMA200 * (1 + B200 * Pt)
    # path length to the exit plane from the 40-digit circle geometry (horizontal radius Pa/k0)
    Pa = mp.sqrt(mp.mpf(P) ** 2 - mp.mpf(Py) ** 2)
    A = mp.sqrt(Pa ** 2 - mp.mpf(Px) ** 2)
    R = Pa / k0
    rho, th = 1 / mp.mpf(h), mp.mpf(h) * L
    # lab basis (e1,e2,e3) = (x-hat, y-hat, s-hat) at the entrance; centre of curvature at (-rho,0,0)
    cx, cz = float(X) - float(R * A / Pa), float(R * mp.mpf(Px) / Pa)          # gyro-centre (e1,e3)

    def exit_plane(a):    # gyration angle a: position relative to the centre of curvature, dotted with s-hat(theta)
        r1 = cx + R * (A / Pa * mp.cos(a) + mp.mpf(Px) / Pa * mp.sin(a)) + rho
        r3 = cz + R * (A / Pa * mp.sin(a) - mp.mpf(Px) / Pa * mp.cos(a))
        return -mp.sin(th) * r1 + mp.cos(th) * r3
    alpha = mp.findroot(exit_plane, th)
    path = float(R * alpha * mp.mpf(P) / Pa)
    b = np.array([0.0, k0, 0.0])

    def rhs(l, y):
        u, S = y[0:3], y[3:6]
        du = np.cross(u, b) / P                          # Lorentz force: d u/dl = u x b / P
        dS = np.cross(_tbmt_axis(u, b, G, gamma, P), S)
        return np.concatenate([du, dS])
    y0 = np.concatenate([[Px / P, Py / P, Ps / P], S0])
    sol = solve_ivp(rhs, (0, path), y0, method="DOP853", rtol=1e-13, atol=1e-16)
    u, S = sol.y[0:3, -1], sol.y[3:6, -1]
    t = float(th)
    xh = np.array([math.cos(t), 0, math.sin(t)])
    sh = np.array([-math.sin(t), 0, math.cos(t)])
    S_local = np.array([S @ xh, S[1], S @ sh])
    out = run([e], z, S0, split=W.SPLIT_BEND_KICK, n_slices=64, depth=4)
    assert abs(out[1] - P * (u @ xh)) < 1e-13            # the orbit agrees too (cf. test_oracle_orbit)
    assert np.max(np.abs(out[6:] - S_local)) < 2e-11, out[6:] - S_local
    # total precession is large (G gamma theta ~ 14.8 rad), so this fixes sign, frame term and convention
    assert np.linalg.norm(S_local - S0) > 0.1


@pytest.mark.parametrize("sign", [+1, -1])
def test_quadrupole_spin_equals_tbmt_integration_along_exact_orbit(sign):
    e = rhic_ir_quad()
    e["kn"][0] *= sign
    L, k1 = float(e["L"]), float(e["kn"][0])
    z, S0 = fn5_particle()
    z = z.copy()
    z[0], z[2] = 8e-3, -6e-3                              # larger offsets -> mrad-scale precession
    G = BEAM200["G"]
    b0 = B200

    def rhs(s, y):
        X, Px, Y, Py, T, Pt = y[:6]
        S = y[6:9]
        P = math.sqrt(1 + 2 * Pt / b0 + Pt * Pt)
        Ps = math.sqrt(P * P - Px * Px - Py * Py)
        u = np.array([Px, Py, Ps]) / P
        gamma = GAMMA200 * (1 + b0 * Pt)
        b = np.array([k1 * Y, k1 * X, 0.0])              # Maxwell: B_x = g y, B_y = g x
        dl = P / Ps                                       # path length per unit s in a straight element
        dS = dl * np.cross(_tbmt_axis(u, b, G, gamma, P), S)
        return [Px / Ps, -k1 * X, Py / Ps, k1 * Y, -(1 / b0 + Pt) / Ps + 1 / b0, 0.0, dS[0], dS[1], dS[2]]
    sol = solve_ivp(rhs, (0, L), np.concatenate([z, S0]), method="DOP853", rtol=1e-13, atol=1e-18)
    ref = sol.y[:, -1]
    out = run([e], z, S0, split=W.SPLIT_MATRIX_KICK, n_slices=64, depth=4)
    assert np.max(np.abs(out[:4] - ref[:4])) < 1e-9      # orbit: 2nd-order MK at 64 slices
    assert np.max(np.abs(out[6:] - ref[6:])) < 1e-9
    assert np.linalg.norm(ref[6:] - S0) > 1e-2


# ---------------------------------------------------------------------------------------------
# closed forms
# ---------------------------------------------------------------------------------------------
def test_omega_on_axis_in_a_bend_is_minus_G_gamma_h():
    e = rhic_dipole()
    Om = O.omega(e, BEAM200, np.zeros(6))
    assert Om[0] == 0 and Om[2] == 0
    assert abs(Om[1] + BEAM200["G"] * GAMMA200 * float(e["h"])) < 1e-15 * abs(Om[1])


def test_uniform_dipole_precesses_G_gamma_theta_relative_to_momentum():
    # on-axis, on-energy: local frame rotates with the momentum, so the local-frame rotation about
    # y-hat is -G gamma theta, for ANY slicing and depth (rotations about one axis commute).
    e = rhic_dipole()
    theta = float(e["h"] * e["L"])
    psi = -BEAM200["G"] * GAMMA200 * theta
    for n, d in ((1, 1), (4, 3), (8, 4)):
        out = run([e], np.zeros(6), [1.0, 0.0, 0.0], split=W.SPLIT_BEND_KICK, n_slices=n, depth=d)
        # right-handed rotation of x-hat about y-hat by psi: (cos psi, 0, -sin psi)
        assert np.max(np.abs(out[6:] - [math.cos(psi), 0.0, -math.sin(psi)])) < 1e-14


def test_planar_ring_spin_tune_is_G_gamma():
    c = W.config(1)
    Gg = c["beam"]["G"] * c["beam"]["gamma0"]
    out = run(list(c["lattice"]), np.zeros(6), [1.0, 0.0, 0.0], split=W.SPLIT_BEND_KICK, n_slices=4, depth=3,
              beam=c["beam"])
    psi = -2 * math.pi * Gg
    assert np.max(np.abs(out[6:] - [math.cos(psi), 0.0, -math.sin(psi)])) < 1e-12
    assert np.max(np.abs(out[:6])) < 1e-25               # the closed orbit is the origin


def test_midplane_bend_romberg_orders_against_closed_form():
    # Py = 0  =>  Omega || y-hat, rotations commute, the spin angle is the integral of Omega_y:
    # psi = -(1+G gamma)(hL + dasin) + hL, with dasin from the exact orbit (10c).  The scheme is then
    # Romberg quadrature of a scalar: errors fall as N^(-2(k+1)).
    e = rhic_dipole()
    L, h = float(e["L"]), float(e["h"])
    z, _ = fn5_particle()
    z = z.copy()
    z[3] = 0.0
    z[0], z[1] = 2e-2, 1.5e-3                             # large amplitude so that errors are above round-off
    Pt = z[5]
    gamma = GAMMA200 * (1 + B200 * Pt)
    Pa = mp.sqrt(1 + 2 * mp.mpf(Pt) / B200 + mp.mpf(Pt) ** 2)
    exact_orbit = run([e], z, [0, 1, 0], split=W.SPLIT_BEND_KICK)
    dasin = mp.asin(mp.mpf(z[1]) / Pa) - mp.asin(mp.mpf(exact_orbit[1]) / Pa)
    psi = -(1 + mp.mpf(BEAM200["G"]) * mp.mpf(GAMMA200) * (1 + mp.mpf(B200) * mp.mpf(Pt))) * (mp.mpf(h) * L + dasin) \
        + mp.mpf(h) * L
    expect = np.array([float(mp.cos(psi)), 0.0, float(-mp.sin(psi))])
    err = {}
    for d in (1, 2, 3):
        for n in (4, 8, 16, 32):
            out = run([e], z, [1.0, 0.0, 0.0], split=W.SPLIT_BEND_KICK, n_slices=n, depth=d)
            err[d, n] = np.linalg.norm(out[6:] - expect)
    assert err[1, 4] > 1e-9
    for n in (4, 8, 16):
        assert 3.7 < err[1, n] / err[1, 2 * n] < 4.3, ("PWC slope -2", err)
    assert 14 < err[2, 4] / err[2, 8] < 18 and 14 < err[2, 8] / err[2, 16] < 18, ("k=1 slope -4", err)
    assert err[3, 4] / err[3, 8] > 50 or err[3, 8] < 1e-14, ("k=2 slope -6", err)
    assert err[3, 8] < err[2, 8] < err[1, 8]


def test_fig7_replay_ir_quad_error_vs_slices():
    # errors against the 256-slice, k=3 result; PWC slope -2; 4 slices + 2 Romberg
    # iterations give "a four-decade reduction".
    e = rhic_ir_quad()
    z, S0 = fn5_particle()
    best = run([e], z, S0, n_slices=256, depth=4)[6:]
    err = {}
    for d in (1, 2, 3):
        for n in (4, 8, 16, 32):
            err[d, n] = np.linalg.norm(run([e], z, S0, n_slices=n, depth=d)[6:] - best)
    for n in (4, 8, 16):
        assert 3.6 < err[1, n] / err[1, 2 * n] < 4.4, err
    assert 12 < err[2, 4] / err[2, 8] < 20, err
    assert err[1, 4] / err[3, 4] > 10 ** (GLD["quad_4slices_k2_decades"] - 1), err


def test_vertical_spin_on_midplane_orbit_in_a_quad_does_not_precess():
    e = rhic_ir_quad()
    z = np.array([5e-3, 2e-4, 0.0, 0.0, 0.0, 3e-4])
    out = run([e], z, [0.0, 1.0, 0.0], n_slices=4, depth=3)
    assert np.max(np.abs(out[6:] - [0.0, 1.0, 0.0])) < 1e-30


def test_precession_magnitude_across_a_quad():
    e = rhic_ir_quad()
    A = 3e-3
    z = np.array([A, 0, 0, 0, 0, 0], dtype=float)
    out = run([e], z, [1.0, 0.0, 0.0], n_slices=16, depth=2)
    ang = math.acos(np.clip(out[6], -1, 1))
    est = (1 + BEAM200["G"] * GAMMA200) * A * float(e["kn"][0]) * float(e["L"])
    assert abs(ang / est - 1) < 0.1                       # "approximately": X shrinks ~6% inside this focusing quad


# ---------------------------------------------------------------------------------------------
# the scheme itself: half weights, product order, table, against an independent rotation library
# ---------------------------------------------------------------------------------------------
def _edge_product(Om, ds, stride):
    N = len(Om) - 1
    R = Rotation.identity()
    for i in range(0, N + 1, stride):
        w = 0.5 if i in (0, N) else 1.0
        R = Rotation.from_rotvec(w * stride * ds * Om[i]) * R         # later rotations on the left
    q = R.as_quat()                                                    # scipy: (x, y, z, w)
    q = np.array([q[3], q[0], q[1], q[2]])
    return q if q[0] > 0 else -q


def test_romberg_table_against_hand_built_table_with_scipy_rotations():
    rng = np.random.default_rng(5)
    N, ds = 8, 0.37
    Om = rng.normal(size=(N + 1, 3)) * 0.2
    for d in (1, 2, 3, 4):
        col = [_edge_product(Om, ds, 1 << (d - 1 - k)) for k in range(d)]
        tab = [col]
        for j in range(1, d):
            prev = tab[-1]
            tab.append([None] * j + [(4 ** j * prev[k] - prev[k - 1]) / (4 ** j - 1) for k in range(j, d)])
        q = tab[-1][-1]
        q = q / np.linalg.norm(q)
        got = O.romberg(Om, ds, d, prec=O.PREC_QUAD)
        assert np.max(np.abs(got - q)) < 5e-15, (d, got, q)
        assert abs(np.linalg.norm(got) - 1) < 1e-15


def test_spin_norm_is_preserved_over_many_elements():
    c = W.config(1)
    out, lost, _ = O.track(c["lattice"], c["beam"], c["state"], 10, c["split"], 4, 3, prec=O.PREC_LONG_DOUBLE)
    assert not lost.any()
    assert np.max(np.abs(np.linalg.norm(out[6:], axis=0) - 1)) < 1e-14


# ---------------------------------------------------------------------------------------------
# snakes (a12, A14): spin tune 1/2 at any energy
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("Gg", [45.5, 45.0, 41.37])
def test_two_orthogonal_snakes_give_spin_tune_one_half(Gg):
    g0 = W.gamma_for_Ggamma(Gg)
    bm = W.beam(g0)
    half = [W.sbend(2.0, math.pi / 8)] * 8
    ring = [W.snake(math.pi, math.radians(45))] + half + [W.snake(math.pi, math.radians(-45))] + half
    R = np.zeros((3, 3))
    for k in range(3):
        S = np.zeros(3)
        S[k] = 1.0
        R[:, k] = run(ring, np.zeros(6), S, split=W.SPLIT_BEND_KICK, n_slices=2, depth=2, beam=bm)[6:]
    assert abs(np.trace(R) + 1) < 1e-12                   # rotation angle pi  <=>  spin tune 1/2
    R2 = R @ R
    assert np.max(np.abs(R2 - np.eye(3))) < 1e-12
    # without snakes the same ring has spin tune G gamma
    R0 = np.zeros((3, 3))
    for k in range(3):
        S = np.zeros(3)
        S[k] = 1.0
        R0[:, k] = run(half + half, np.zeros(6), S, split=W.SPLIT_BEND_KICK, n_slices=2, depth=2, beam=bm)[6:]
    assert abs(np.trace(R0) - (1 + 2 * math.cos(2 * math.pi * Gg))) < 1e-11


def test_snake_is_a_rotation_by_mu_about_its_horizontal_axis():
    phi, mu = math.radians(30), 2.1
    S0 = np.array([0.3, -0.5, 0.8])
    S0 /= np.linalg.norm(S0)
    out = run([W.snake(mu, phi)], np.array([1e-3, 1e-4, 2e-3, -1e-4, 0.01, 1e-4]), S0)
    # component order (x, y, s); axis = (sin phi, 0, cos phi)
    expect = Rotation.from_rotvec(mu * np.array([math.sin(phi), 0.0, math.cos(phi)])).apply(S0)
    assert np.max(np.abs(out[6:] - expect)) < 1e-15
    assert np.all(out[:6] == [1e-3, 1e-4, 2e-3, -1e-4, 0.01, 1e-4])


def test_thin_multipole_spin_kick_matches_thick_limit():
    # A10: the thin lens is the L -> 0 limit of the thick multipole with k*L fixed
    z, S0 = fn5_particle()
    knl = (0.0, 0.35, 0.0, 0.0)
    thin = run([W.thin_multipole(knl)], z, S0)
    L = 1e-6
    thick = run([W.multipole(L, kn=tuple(k / L for k in knl))], z, S0, n_slices=1, depth=1)
    assert np.max(np.abs(thin[6:] - thick[6:])) < 1e-9
    assert np.max(np.abs(thin[:6] - thick[:6])) < 1e-9
