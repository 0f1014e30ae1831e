"""Pins for the RF cavity / ramp reading (A12, A13 -- formulas NOT in the paper) and for
the reductions (A18, A19) of the CPU oracle.  Beyond these pins the cavity is "parity unpinned"."""
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
