"""Pins for the RF cavity / ramp reading (A12, A13 -- formulas NOT in the paper) and for
the reductions (A18, A19) of the CPU oracle: the cavity's slope and the synchrotron tune at two energies against the
exact longitudinal map, the re-referencing element by element, adiabatic damping, and the crossing of an isolated
resonance against the Froissart-Stora formula to 3e-4 for the adiabatic invariant."""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_1501_03450_b200 import workloads as W


def _ring_with_cavity(sign, phi_s=0.0, volt=300e3):
    lat0 = W.fodo_ring(64)
    return W.fodo_ring(64, rf=W.cavity(volt, 360.0, phi_s, sign)), W.linear_optics(lat0)


def test_small_amplitude_synchrotron_tune_and_stable_sign():
    g0 = 25.0
    b0 = W.beta_of_gamma(g0)
    bm = W.beam(g0)
    lat, opt = _ring_with_cavity(+1.0)
    assert g0 > opt["gamma_t"]                                  # above transition (A12)
    J, _ = O.jacobian(lat, bm, np.zeros(6), W.SPLIT_MATRIX_KICK, 2)
    ev = np.linalg.eigvals(J)
    assert np.max(np.abs(np.abs(ev) - 1)) < 1e-9                # all three modes stable
    tunes = np.sort(np.abs(np.angle(ev)) / (2 * math.pi))
    eta_s = opt["alpha_c"] - 1 / g0 ** 2
    E0 = g0 * bm["mass_eV"]
    Qs = math.sqrt(360.0 * abs(eta_s) * 300e3 / (2 * math.pi * b0 ** 2 * E0))   # textbook, cos(phi_s) = 1
    assert abs(tunes[0] / Qs - 1) < 2e-3, (tunes[0], Qs)
    # the opposite sign is the unstable fixed point above transition
    lat_bad, _ = _ring_with_cavity(-1.0)
    Jb, _ = O.jacobian(lat_bad, bm, np.zeros(6), W.SPLIT_MATRIX_KICK, 2)
    assert np.max(np.abs(np.linalg.eigvals(Jb))) > 1 + 1e-3


def test_ramp_reference_energy_and_adiabatic_damping():
    g0 = 25.0
    bm = W.beam(g0)
    volt, phi_s = 3e6, math.asin(0.25)
    lat = W.fodo_ring(16, rf=W.cavity(volt, 12.0, phi_s, +1.0))
    n, turns = 64, 1500
    st = W.gaussian_bunch(11, n, g0, 1e-3, 1e-4, 1e-3, 1e-4, 0.0, 0.0)
    out, lost, g1 = O.track(lat, bm, st, turns, W.SPLIT_MATRIX_KICK, 2, 1, prec=O.PREC_DOUBLE)
    assert not lost.any()
    # A13: E0 grows by qV sin(phi_s) per turn
    assert abs(g1 - (g0 + turns * volt * 0.25 / bm["mass_eV"])) < 1e-9
    # G gamma_o(n) for the config-4 numbers quoted in SURVEY A13: 100 keV/turn -> 1.9108e-4 per turn
    assert abs(W.G_PROTON * 1e5 / W.MASS_PROTON_EV - 1.9108e-4) < 1e-8
    e0, e1 = O.emittance(st), O.emittance(out)
    bg0, bg1 = g0 * W.beta_of_gamma(g0), g1 * W.beta_of_gamma(g1)
    assert g1 / g0 > 1.015
    for k in range(2):                                          # normalised rms emittance is invariant
        assert abs(e1[k] * bg1 / (e0[k] * bg0) - 1) < 2e-3
        assert abs(e1[k] / e0[k] - 1) > 5e-3                    # while the geometric one shrinks
    # synchronous particle stays synchronous
    s0 = np.zeros((9, 1)); s0[7] = 1.0
    o2, _, _ = O.track(lat, bm, s0, 50, W.SPLIT_MATRIX_KICK, 2, 1, prec=O.PREC_QUAD)
    assert np.max(np.abs(o2[:6])) < 1e-25


def test_ramp_longitudinal_area_scales_with_the_reference_momentum():
    """A13 rescales Pt = (E - E0)/(p0 c) to the new p0 and leaves T alone: the (T, Pt) rms area of a short
    bunch (linear motion about phi_s) shrinks as p0/p0' = (beta gamma)_0/(beta gamma)_1, i.e. the normalised
    longitudinal emittance is the adiabatic invariant.  A missing or inverted Pt rescale leaves the ratio
    at 1 or at (p0'/p0)."""
    g0 = 25.0
    bm = W.beam(g0)
    volt, phi_s = 3e6, math.asin(0.25)
    lat = W.fodo_ring(16, rf=W.cavity(volt, 12.0, phi_s, +1.0))
    st = W.gaussian_bunch(12, 64, g0, 0.0, 0.0, 0.0, 0.0, 1e-4, 0.01)
    out, lost, g1 = O.track(lat, bm, st, 1500, W.SPLIT_MATRIX_KICK, 2, 1, prec=O.PREC_DOUBLE)
    assert not lost.any()

    def area(s):
        return math.sqrt(np.linalg.det(np.cov(s[4], s[5], bias=True)))

    shrink = g0 * W.beta_of_gamma(g0) / (g1 * W.beta_of_gamma(g1))
    assert shrink < 0.96
    assert abs(area(out) / area(st) / shrink - 1) < 3e-3


@pytest.mark.parametrize("dGg,eps", [(2.5e-4, 2e-3), (2.5e-4, 4.2e-3), (2.5e-4, 8e-3), (1e-3, 8.4e-3)])
def test_ramp_through_an_isolated_resonance_follows_froissart_stora(dGg, eps):
    """Polarization through the ramp (config 4's subject) against the textbook closed form: crossing an
    isolated resonance of strength eps at the rate alpha = d(G gamma)/d(theta) leaves
    Sy_f / Sy_i = 2 exp(-pi eps^2 / (2 alpha)) - 1 (Froissart and Stora, 1960).  The resonance is a thin
    partial snake (tune gap eps at integer G gamma) in a planar ring, the particle is on axis, so the only
    inputs are A13's gamma_o(n) in Omega (6b), the snake rotation (A14) and the bend precession.  The spin
    still nutates by eps/(distance to the resonance) = 2 eps at the end of the run: tolerance 0.02."""
    lat, bm, turns = W.resonance_crossing_ring(dGg, eps)
    st = np.zeros((9, 1))
    st[7] = 1.0
    out, lost, g1 = O.track(lat, bm, st, turns, W.SPLIT_BEND_KICK, 4, 3, prec=O.PREC_DOUBLE)
    assert not lost.any() and np.max(np.abs(out[:6])) == 0.0
    assert abs(W.G_PROTON * g1 - 45.5) < 1e-9
    alpha = dGg / (2 * math.pi)
    fs = 2 * math.exp(-math.pi * eps ** 2 / (2 * alpha)) - 1
    assert abs(out[7, 0] - fs) < 0.02, (out[7, 0], fs)
    assert abs(np.linalg.norm(out[6:9, 0]) - 1) < 1e-10


@pytest.mark.parametrize("g0", [3.0, 25.0])
def test_cavity_slope_and_synchrotron_tune_against_the_longitudinal_map(g0):
    """A12 at two energies, one below and one above transition (gamma_t = 6.13), so that every power of beta_o counts
    (beta_o = 0.943 at gamma_o = 3): (i) the cavity's linearised kick d(Pt')/dT = sign qV (2 pi h beta_o / C)/(p_o c) is the
    textbook omega_rf = h omega_rev; (ii) the one-turn Jacobian with the cavity is that thin kick times the Jacobian of
    the ring without it (nothing else in the turn knows about the cavity); (iii) the synchrotron tune equals the closed
    form of the 2x2 longitudinal map, cos mu = 1 - pi h eta_s qV cos(phi_s)/(beta_o^2 E_o), eta_s = alpha_c - 1/gamma_o^2
    from textbook optics, up to the synchro-betatron coupling of a cavity in a dispersive place (4e-4 / 4e-5 here): a wrong
    power of beta_o in k_rf changes the tune by 3 % at gamma_o = 3."""
    bm = W.beam(g0)
    b0 = W.beta_of_gamma(g0)
    E0 = g0 * bm["mass_eV"]
    ring = W.fodo_ring(64)
    opt = W.linear_optics(ring)
    C = float(np.sum(ring["L"]))
    volt, h = 300e3, 360.0
    sign = +1.0 if g0 > opt["gamma_t"] else -1.0               # the stable side
    a = sign * volt * (2 * math.pi * h * b0 / C) / (b0 * E0)   # (i)
    Jc, _ = O.jacobian(W.lattice([W.cavity(volt, h, 0.0, sign)]), bm, np.zeros(6), W.SPLIT_MATRIX_KICK, 2, circumference=C)
    K = np.eye(6)
    K[5, 4] = a
    assert np.max(np.abs(Jc - K)) < 1e-15 * max(1.0, abs(a)) + 1e-18, (Jc[5, 4], a)
    J0, _ = O.jacobian(ring, bm, np.zeros(6), W.SPLIT_MATRIX_KICK, 2)
    # fodo_ring puts the cavity in front of the ring
    lat = W.fodo_ring(64, rf=W.cavity(volt, h, 0.0, sign))
    assert int(lat[0]["type"]) == W.RFCAV
    J1, _ = O.jacobian(lat, bm, np.zeros(6), W.SPLIT_MATRIX_KICK, 2)
    assert np.max(np.abs(J1 - J0 @ K)) < 1e-12                  # (ii)
    ev = np.linalg.eigvals(J1)
    assert np.max(np.abs(np.abs(ev) - 1)) < 1e-9
    Qs = np.sort(np.abs(np.angle(ev)) / (2 * math.pi))[0]
    eta_s = opt["alpha_c"] - 1 / g0 ** 2
    # the slip factor the oracle's ring really has (dispersion included) is the textbook one
    D = np.linalg.solve(np.eye(4) - J0[:4, :4], J0[:4, 5])
    assert abs(-(J0[4, 5] + J0[4, :4] @ D) * b0 ** 2 / C / eta_s - 1) < 1e-9
    cos_mu = 1 - math.pi * h * eta_s * sign * volt / (b0 ** 2 * E0)
    Qs_closed = math.acos(cos_mu) / (2 * math.pi)
    assert abs(Qs / Qs_closed - 1) < (6e-4 if g0 < 10 else 6e-5), (Qs, Qs_closed)      # (iii)


def test_rereferencing_rescales_the_momenta_and_leaves_T_alone():
    """A13 element by element: through a ramping cavity T is unchanged to the last bit, Px and Py shrink by p_o/p_o',
    the particle's own energy gains qV sin(phi_s + sign k_rf T), and E_o gains qV sin(phi_s)."""
    g0 = 3.0                                            # low energy: p_o/p_o' is far from 1
    bm = W.beam(g0)
    m = bm["mass_eV"]
    volt, h, phi_s, C = 40e6, 7.0, math.asin(0.3), 100.0
    lat = W.lattice([W.drift(C), W.cavity(volt, h, phi_s, +1.0)])
    st = np.zeros((9, 3))
    st[1] = [1e-3, -2e-3, 0.0]
    st[3] = [5e-4, 0.0, 3e-3]
    st[4] = [0.02, -0.05, 0.0]
    st[5] = [1e-3, -2e-3, 0.0]
    st[7] = 1.0
    before, _, _ = O.track(W.lattice([W.drift(C)]), bm, st, 1, W.SPLIT_BEND_KICK, 1, 1, prec=O.PREC_QUAD)
    after, lost, g1 = O.track(lat, bm, st, 1, W.SPLIT_BEND_KICK, 1, 1, prec=O.PREC_QUAD)
    assert not lost.any()
    assert np.array_equal(after[4], before[4])                               # T untouched, bit for bit
    E0, E1 = g0 * m, g0 * m + volt * 0.3
    assert abs(g1 * m / E1 - 1) < 1e-15
    p0, p1 = math.sqrt(E0 ** 2 - m ** 2), math.sqrt(E1 ** 2 - m ** 2)
    assert np.max(np.abs(after[1][before[1] != 0] / before[1][before[1] != 0] - p0 / p1)) < 1e-15
    assert np.max(np.abs(after[3][before[3] != 0] / before[3][before[3] != 0] - p0 / p1)) < 1e-15
    b0 = p0 / E0
    E_part = E0 + p0 * before[5] + volt * np.sin(phi_s + (2 * math.pi * h * b0 / C) * before[4])
    assert np.max(np.abs(after[5] - (E_part - E1) / p1)) < 1e-15
    assert np.array_equal(after[6:9], before[6:9])                           # spin: identity (A12)


def _spin_axis_of_the_crossing_ring(Ggamma, eps, phi=0.0):
    """Invariant spin direction of the on-axis one-turn map R_snake(2 pi eps) R_y(-2 pi G gamma) of
    workloads.resonance_crossing_ring (the bends give Omega = -G gamma h y-hat; the partial snake ends the turn),
    from textbook quaternion composition; oriented along +y."""
    th, mu = -2 * math.pi * Ggamma, 2 * math.pi * eps
    w1, x1, y1, z1 = math.cos(mu / 2), math.sin(mu / 2) * math.sin(phi), 0.0, math.sin(mu / 2) * math.cos(phi)
    w2, x2, y2, z2 = math.cos(th / 2), 0.0, math.sin(th / 2), 0.0
    v = np.array([w1 * x2 + x1 * w2 + y1 * z2 - z1 * y2, w1 * y2 - x1 * z2 + y1 * w2 + z1 * x2,
                  w1 * z2 + x1 * y2 - y1 * x2 + z1 * w2])
    v /= np.linalg.norm(v)
    return v if v[1] > 0 else -v


@pytest.mark.parametrize("dGg,eps", [(2.5e-4, 2e-3), (2.5e-4, 4.2e-3), (2.5e-4, 8e-3), (1e-3, 8.4e-3), (1e-3, 2e-2)])
def test_froissart_stora_for_the_adiabatic_invariant(dGg, eps):
    """The sharp form of the crossing pin: half a unit of G gamma away from the resonance the stable spin direction n_0
    is tilted by 2 eps, and a spin that starts along y-hat nutates about it -- the 0.02 of the test above.  The adiabatic
    invariant is S.n_0: start ON the invariant direction of the starting energy, project on the invariant direction of
    the final energy, and the Froissart-Stora ratio 2 exp(-pi eps^2/(2 alpha)) - 1 comes out to 2e-4 (from a full flip,
    -0.96, through zero to +0.71), the remainder being the finite distance the ramp starts and ends at."""
    lat, bm, turns = W.resonance_crossing_ring(dGg, eps)
    Gg0 = W.G_PROTON * bm["gamma0"]
    st = np.zeros((9, 1))
    st[6:9, 0] = _spin_axis_of_the_crossing_ring(Gg0, eps)
    out, lost, g1 = O.track(lat, bm, st, turns, W.SPLIT_BEND_KICK, 4, 3, prec=O.PREC_DOUBLE)
    assert not lost.any() and abs(W.G_PROTON * g1 - (Gg0 + 1.0)) < 1e-9
    J = float(out[6:9, 0] @ _spin_axis_of_the_crossing_ring(W.G_PROTON * g1, eps))
    fs = 2 * math.exp(-math.pi * eps ** 2 / (2 * dGg / (2 * math.pi))) - 1
    assert abs(J - fs) < 3e-4, (J, fs)


def test_polarization_and_emittance_against_numpy():
    rng = np.random.default_rng(3)
    n = 1000
    st = rng.normal(size=(9, n))
    lost = (rng.uniform(size=n) < 0.1).astype(np.uint8)
    P, nl = O.polarization(st, lost)
    keep = lost == 0
    m = st[6:9, keep].mean(axis=1)
    assert nl == int(lost.sum())
    assert np.max(np.abs(P[:3] - m)) < 1e-15 and abs(P[3] - np.linalg.norm(m)) < 1e-15
    e = O.emittance(st, lost)
    for k in range(2):
        c = np.cov(st[2 * k, keep], st[2 * k + 1, keep], bias=True)
        assert abs(e[k] - math.sqrt(np.linalg.det(c))) < 1e-13
