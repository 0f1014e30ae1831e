"""Seeded synthetic workloads: the five BASELINE.json configurations (lattice + bunch + track args).

This module serves BOTH the CUDA path (via the binding) and the CPU oracle (via oracle/oracle.py)
and therefore holds NONE of the method's arithmetic: no symplectic map, no precession vector, no
quaternion.  What it does hold is lattice *design* arithmetic -- textbook linear transfer matrices
(drift, thick quadrupole, sector dipole) used to find the periodic Twiss functions, dispersion and
momentum compaction so that the RHIC-like bunches can be matched and the cavity sign chosen --
and the counter-based random number generator (numpy Philox) that draws the bunches.

The lattices are synthetic stand-ins for the RHIC SXF lattice of the paper, which is not
available; they take RHIC's shapes from P:577, P:664, P:699 and BASELINE.json.
states the recipe.
"""
import math

import numpy as np

DRIFT, SBEND, QUAD, MULTIPOLE, THINMULT, RFCAV, SNAKE, MARKER, FRINGE, SOLENOID, RBEND = range(11)
SPLIT_DRIFT_KICK, SPLIT_BEND_KICK, SPLIT_MATRIX_KICK = range(3)
# the same splits with the fourth-order composition of every non-exact slice map (gst.h)
SPLIT_DRIFT_KICK_4, SPLIT_BEND_KICK_4, SPLIT_MATRIX_KICK_4 = range(3, 6)
# spin ordering of the mid-slice piece-wise-constant comparison integrators ((37); gst_track_pwc)
PWC_HALF_SLICE, PWC_DKSKD = 0, -1
SPLIT_NAMES = {SPLIT_DRIFT_KICK: "drift_kick", SPLIT_BEND_KICK: "bend_kick", SPLIT_MATRIX_KICK: "matrix_kick",
               SPLIT_DRIFT_KICK_4: "drift_kick_4", SPLIT_BEND_KICK_4: "bend_kick_4", SPLIT_MATRIX_KICK_4: "matrix_kick_4"}

G_PROTON = 1.792847            # BASELINE.json
MASS_PROTON_EV = 938.27208816e6

ELEM_DTYPE = np.dtype([("type", "i4"), ("slice_mult", "i4"), ("L", "f8"), ("h", "f8"), ("k0", "f8"),
                       ("kn", "f8", (4,)), ("ks", "f8", (4,)),
                       ("volt_eV", "f8"), ("harmonic", "f8"), ("phi_s", "f8"), ("sign", "f8"),
                       ("snake_mu", "f8"), ("snake_phi", "f8")])


def _blank(t, L=0.0):
    e = np.zeros((), dtype=ELEM_DTYPE)
    e["type"] = t
    e["slice_mult"] = 1
    e["L"] = L
    return e


def drift(L):
    return _blank(DRIFT, L)


def sbend(L, angle, eta=1.0):
    e = _blank(SBEND, L)
    e["h"] = angle / L
    e["k0"] = eta * angle / L
    return e


def quad(L, k1, slice_mult=1):
    e = _blank(QUAD, L)
    e["kn"][0] = k1
    e["slice_mult"] = slice_mult
    return e


def multipole(L, kn=(0, 0, 0, 0), ks=(0, 0, 0, 0), slice_mult=1):
    e = _blank(MULTIPOLE, L)
    e["kn"] = kn
    e["ks"] = ks
    e["slice_mult"] = slice_mult
    return e


def thin_multipole(knl=(0, 0, 0, 0), ksl=(0, 0, 0, 0)):
    e = _blank(THINMULT)
    e["kn"] = knl
    e["ks"] = ksl
    return e


def thin_sextupole(k2l_mad):
    """MAD k2*L -> paper convention (28): b3 L/(B rho) = k2 L / 2 (A22)."""
    return thin_multipole(knl=(0.0, 0.5 * k2l_mad, 0.0, 0.0))


def cavity(volt_eV, harmonic, phi_s, sign):
    e = _blank(RFCAV)
    e["volt_eV"] = volt_eV
    e["harmonic"] = harmonic
    e["phi_s"] = phi_s
    e["sign"] = sign
    return e


def snake(mu, phi):
    e = _blank(SNAKE)
    e["snake_mu"] = mu
    e["snake_phi"] = phi
    return e


def marker():
    return _blank(MARKER)


def fringe(sign, k0=0.0, kn=(0, 0, 0, 0), ks=(0, 0, 0, 0)):
    """Thin-fringe spin kick (41) of a magnet with body strengths k0 (dipole), kn, ks (m = 2..5, per unit length,
    convention of (28)); sign = +1 at the entrance, -1 at the exit."""
    e = _blank(FRINGE)
    e["k0"] = k0
    e["kn"] = kn
    e["ks"] = ks
    e["sign"] = sign
    return e


def solenoid(L, ks, slice_mult=1):
    """Solenoid with thin-pancake fringes (section 3.7): ks = b_0/(B rho)_o [1/m] (eta of (35) is ks/2)."""
    e = _blank(SOLENOID)
    e["L"] = L
    e["k0"] = ks
    e["slice_mult"] = slice_mult
    return e


def rbend(L, angle, phi_entr=None, phi_exit=None, slice_mult=1):
    """Rectangular bend (section 3.2): magnet length L along its axis, total bend angle; the beam meets the
    entrance face at phi_entr and leaves at phi_exit (default symmetric: +-angle/2); sin(phi_entr) -
    sin(phi_exit) = L/rho_b fixes the field k0 = 1/rho_b (13b)."""
    if phi_entr is None:
        phi_entr, phi_exit = 0.5 * angle, -0.5 * angle
    assert abs((phi_entr - phi_exit) - angle) < 1e-15 * max(1.0, abs(angle))
    e = _blank(RBEND)
    e["L"] = L
    e["k0"] = (math.sin(phi_entr) - math.sin(phi_exit)) / L
    e["kn"] = (phi_entr, phi_exit, 0.0, 0.0)
    e["slice_mult"] = slice_mult
    return e


def with_fringes(magnet):
    """[entrance fringe, magnet, exit fringe] for a thick SBEND / QUAD / MULTIPOLE element."""
    k0 = float(magnet["k0"]) if int(magnet["type"]) == SBEND else 0.0
    kn, ks = tuple(magnet["kn"]), tuple(magnet["ks"])
    return [fringe(+1.0, k0, kn, ks), magnet, fringe(-1.0, k0, kn, ks)]


def lattice(elems):
    return np.array(list(elems), dtype=ELEM_DTYPE)


def beam(gamma0, G=G_PROTON, mass_eV=MASS_PROTON_EV):
    return {"G": float(G), "mass_eV": float(mass_eV), "gamma0": float(gamma0)}


def beta_of_gamma(g):
    return math.sqrt(1.0 - 1.0 / (g * g))


def steps_per_turn(lat, n_slices):
    """particle-element-steps per particle per turn."""
    thick = np.isin(lat["type"], (SBEND, QUAD, MULTIPOLE, SOLENOID, RBEND))
    return int(np.sum(np.where(thick, n_slices * lat["slice_mult"], 1)))


# ------------------------------------------------------------------------------------------------
# textbook linear optics (lattice design, not the tracking method)
# ------------------------------------------------------------------------------------------------
def _linear_maps(e):
    """(Mx 3x3 on (x, x', delta), My 2x2) of one element in the paraxial textbook approximation."""
    t, L = int(e["type"]), float(e["L"])
    Mx, My = np.eye(3), np.eye(2)
    if t == DRIFT or (t == MULTIPOLE and e["kn"][0] == 0):
        Mx[0, 1] = L
        My[0, 1] = L
    elif t == SBEND:
        h = float(e["h"])
        th = h * L
        c, s = math.cos(th), math.sin(th)
        Mx[:] = [[c, s / h, (1 - c) / h], [-h * s, c, s], [0, 0, 1]]
        My[0, 1] = L
    elif t in (QUAD, MULTIPOLE):
        k1 = float(e["kn"][0])
        w = math.sqrt(abs(k1))
        cf, sf = math.cos(w * L), math.sin(w * L)
        cd, sd = math.cosh(w * L), math.sinh(w * L)
        F = np.array([[cf, sf / w], [-w * sf, cf]])
        D = np.array([[cd, sd / w], [w * sd, cd]])
        Mx[:2, :2] = F if k1 > 0 else D
        My[:] = D if k1 > 0 else F
    elif t == THINMULT:
        k1l = float(e["kn"][0])
        Mx[1, 0] = -k1l
        My[1, 0] = k1l
    return Mx, My


def linear_optics(lat):
    """Periodic Twiss at the start of `lat` plus per-element entrance values.

    Returns dict(Qx, Qy, betx, alfx, bety, alfy, Dx, Dpx, alpha_c, gamma_t, C, and arrays
    betx_s, bety_s, Dx_s at every element entrance).
    """
    maps = [_linear_maps(e) for e in lat]
    Mx, My = np.eye(3), np.eye(2)
    for a, b in maps:
        Mx, My = a @ Mx, b @ My
    out = {}
    for name, M in (("x", Mx[:2, :2]), ("y", My)):
        cosmu = 0.5 * (M[0, 0] + M[1, 1])
        if abs(cosmu) >= 1:
            raise ValueError("unstable lattice in plane %s (cos mu = %g)" % (name, cosmu))
        sinmu = math.copysign(math.sqrt(1 - cosmu * cosmu), M[0, 1])
        out["bet" + name] = M[0, 1] / sinmu
        out["alf" + name] = (M[0, 0] - M[1, 1]) / (2 * sinmu)
    d = np.linalg.solve(np.eye(2) - Mx[:2, :2], Mx[:2, 2])
    out["Dx"], out["Dpx"] = float(d[0]), float(d[1])
    # propagate
    n = len(lat)
    bx, ax, by, ay = out["betx"], out["alfx"], out["bety"], out["alfy"]
    dv = np.array([out["Dx"], out["Dpx"], 1.0])
    betx_s, bety_s, Dx_s = np.zeros(n), np.zeros(n), np.zeros(n)
    mux = muy = 0.0
    I5 = 0.0  # integral of D*h ds
    for i, (a, b) in enumerate(maps):
        betx_s[i], bety_s[i], Dx_s[i] = bx, by, dv[0]
        e = lat[i]
        if int(e["type"]) == SBEND:
            h, L = float(e["h"]), float(e["L"])
            th = h * L
            I5 += dv[0] * math.sin(th) + dv[1] * (1 - math.cos(th)) / h + (th - math.sin(th)) / h
        for (M, bb, aa, which) in ((a[:2, :2], bx, ax, "x"), (b, by, ay, "y")):
            gg = (1 + aa * aa) / bb
            nb = M[0, 0] ** 2 * bb - 2 * M[0, 0] * M[0, 1] * aa + M[0, 1] ** 2 * gg
            na = -M[0, 0] * M[1, 0] * bb + (M[0, 0] * M[1, 1] + M[0, 1] * M[1, 0]) * aa - M[0, 1] * M[1, 1] * gg
            dmu = math.atan2(M[0, 1], M[0, 0] * bb - M[0, 1] * aa)
            if which == "x":
                bx, ax = nb, na
                mux += dmu
            else:
                by, ay = nb, na
                muy += dmu
        dv = a @ dv
    C = float(np.sum(lat["L"]))
    out.update(Qx=mux / (2 * math.pi), Qy=muy / (2 * math.pi), C=C, alpha_c=I5 / C,
               gamma_t=(1 / math.sqrt(I5 / C)) if I5 > 0 else float("inf"),
               betx_s=betx_s, bety_s=bety_s, Dx_s=Dx_s)
    return out


def natural_chromaticity(lat, opt):
    """Thin-quad estimate  xi = -(1/4 pi) sum k1 L beta  (entrance/exit average), per plane."""
    n = len(lat)
    xx = xy = 0.0
    for i, e in enumerate(lat):
        if int(e["type"]) == QUAD:
            j = (i + 1) % n
            k1l = float(e["kn"][0] * e["L"])
            xx -= k1l * 0.5 * (opt["betx_s"][i] + opt["betx_s"][j])
            xy += k1l * 0.5 * (opt["bety_s"][i] + opt["bety_s"][j])
    return xx / (4 * math.pi), xy / (4 * math.pi)


# ------------------------------------------------------------------------------------------------
# bunches
# ------------------------------------------------------------------------------------------------
def _rng(seed):
    return np.random.Generator(np.random.Philox(key=int(seed)))


def pt_of_delta(delta, beta0):
    """Invert (22): P = 1 + delta  ->  Pt  (A22)."""
    return np.sqrt(1.0 / beta0 ** 2 + 2.0 * delta + delta * delta) - 1.0 / beta0


def spins_vertical(n):
    S = np.zeros((3, n))
    S[1] = 1.0
    return S


def spins_sphere(rng, n):
    z = rng.uniform(-1.0, 1.0, n)
    ph = rng.uniform(0.0, 2 * math.pi, n)
    r = np.sqrt(1 - z * z)
    S = np.stack([r * np.cos(ph), z, r * np.sin(ph)])
    return S / np.sqrt(np.sum(S * S, axis=0))


def gaussian_bunch(seed, n, gamma0, sx, sxp, sy, syp, sdelta, sz, spins="vertical"):
    """Uncorrelated 6-D Gaussian (configs 1, 2): Px := x' sample, T := z/beta_o, Pt from delta (A22)."""
    rng = _rng(seed)
    b0 = beta_of_gamma(gamma0)
    g = rng.standard_normal((6, n))
    st = np.zeros((9, n))
    st[0], st[1], st[2], st[3] = sx * g[0], sxp * g[1], sy * g[2], syp * g[3]
    st[4] = sz * g[4] / b0
    st[5] = pt_of_delta(sdelta * g[5], b0)
    st[6:9] = spins_vertical(n) if spins == "vertical" else spins_sphere(rng, n)
    return st


def matched_bunch(seed, n, gamma0, opt, eps_n, sdelta, sz, spins="vertical"):
    """Matched Gaussian from the periodic Twiss at the lattice start + dispersion (A25)."""
    rng = _rng(seed)
    b0 = beta_of_gamma(gamma0)
    eps = eps_n / (b0 * gamma0)
    g = rng.standard_normal((6, n))
    delta = sdelta * g[5]
    st = np.zeros((9, n))
    st[0] = math.sqrt(eps * opt["betx"]) * g[0] + opt["Dx"] * delta
    st[1] = math.sqrt(eps / opt["betx"]) * (g[1] - opt["alfx"] * g[0]) + opt["Dpx"] * delta
    st[2] = math.sqrt(eps * opt["bety"]) * g[2]
    st[3] = math.sqrt(eps / opt["bety"]) * (g[3] - opt["alfy"] * g[2])
    st[4] = sz * g[4] / b0
    st[5] = pt_of_delta(delta, b0)
    st[6:9] = spins_vertical(n) if spins == "vertical" else spins_sphere(rng, n)
    return st


# ------------------------------------------------------------------------------------------------
# lattices
# ------------------------------------------------------------------------------------------------
def fodo_ring(n_cells, sextupole_k2l=None, rf=None):
    """BASELINE configs[0]/[1]: cells of [D 1, QF .5, D 1, SB 2, QD .5, D 1, SB 2], bends close the ring."""
    ang = 2 * math.pi / (2 * n_cells)
    cell = []
    cell.append(drift(1.0))
    cell.append(quad(0.5, +0.3))
    if sextupole_k2l:
        cell.append(thin_sextupole(+sextupole_k2l))
    cell.append(drift(1.0))
    cell.append(sbend(2.0, ang))
    cell.append(quad(0.5, -0.3))
    if sextupole_k2l:
        cell.append(thin_sextupole(-sextupole_k2l))
    cell.append(drift(1.0))
    cell.append(sbend(2.0, ang))
    els = []
    if rf is not None:
        els.append(rf)
    for _ in range(n_cells):
        els.extend(cell)
    return lattice(els)


RHIC_LIKE = dict(Lq=1.11, Lb=9.45, cell=29.622, n_arcs=6, cells_per_arc=11, k1=0.09,
                 straight=313.1247, straight_cells=10, drift_pieces=7, harmonic=360.0, volt_eV=300e3,
                 tunes=(33.57, 33.43))


def rhic_like_ring(gamma0, snakes=True, phi_s=0.0, chroma=(2.0, 2.0)):
    """BASELINE configs[2]: synthetic RHIC-like ring, C = 3833.8 m (SURVEY §8(d) recipe).

    6 arcs of 11 FODO cells [QF, sx, D, SB, D, QD, sx, D, SB, D] and 6 dipole-free straights of
    10 FODO cells whose long drifts are cut into 7 pieces; snakes (mu = pi, axes +-45 deg) at the
    centres of straights 1 and 4; one cavity at the start of straight 1.  Two thin-sextupole
    families set the linear chromaticity estimate to `chroma`.
    """
    p = RHIC_LIKE
    d = (p["cell"] - 2 * p["Lq"] - 2 * p["Lb"]) / 4
    ang = 2 * math.pi / (p["n_arcs"] * p["cells_per_arc"] * 2)
    scell_len = p["straight"] / p["straight_cells"]
    D = (scell_len - 2 * p["Lq"]) / 2
    piece = D / p["drift_pieces"]

    def build(k2f, k2d, cav_sign, ksf=p["k1"], ksd=-p["k1"]):
        arc_cell = [quad(p["Lq"], +p["k1"]), thin_sextupole(k2f), drift(d), sbend(p["Lb"], ang), drift(d),
                    quad(p["Lq"], -p["k1"]), thin_sextupole(k2d), drift(d), sbend(p["Lb"], ang), drift(d)]
        str_cell = [quad(p["Lq"], ksf)] + [drift(piece)] * p["drift_pieces"] + \
                   [quad(p["Lq"], ksd)] + [drift(piece)] * p["drift_pieces"]
        els = []
        for a in range(p["n_arcs"]):
            straight = []
            for c in range(p["straight_cells"]):
                straight.extend(str_cell)
            if a == 0:
                straight.insert(0, cavity(p["volt_eV"], p["harmonic"], phi_s, cav_sign))
            if snakes and a in (0, 3):
                mid = len(straight) // 2 + (1 if a == 0 else 0)
                straight.insert(mid, snake(math.pi, math.radians(45.0 if a == 0 else -45.0)))
            els.extend(straight)
            for c in range(p["cells_per_arc"]):
                els.extend(arc_cell)
        return lattice(els)

    # trim the straight-section quads (|k1| stays ~0.09) so that the linear tunes sit at p["tunes"]:
    # with all |k1| = 0.09 the ring lands on Qy = 33.495, i.e. on the half-integer stop band.
    ksf, ksd = p["k1"], -p["k1"]
    target = np.array(p["tunes"])
    for _ in range(8):
        def tunes(a, b):
            o = linear_optics(build(0.0, 0.0, 1.0, a, b))
            return np.array([o["Qx"], o["Qy"]])
        q0 = tunes(ksf, ksd)
        if np.max(np.abs(q0 - target)) < 1e-10:
            break
        eps = 1e-6
        Jt = np.stack([(tunes(ksf + eps, ksd) - q0) / eps, (tunes(ksf, ksd + eps) - q0) / eps], axis=1)
        dk = np.linalg.solve(Jt, target - q0)
        ksf, ksd = ksf + dk[0], ksd + dk[1]
    lat0 = build(0.0, 0.0, 1.0, ksf, ksd)
    opt = linear_optics(lat0)
    sign = 1.0 if gamma0 > opt["gamma_t"] else -1.0
    # two sextupole families: xi = xi_nat + (1/4pi) sum k2L D beta  ->  solve 2x2 for (k2f, k2d)
    xnat = natural_chromaticity(lat0, opt)
    idx = np.where(lat0["type"] == THINMULT)[0]
    fam_f, fam_d = idx[0::2], idx[1::2]
    A = np.zeros((2, 2))
    for col, fam in enumerate((fam_f, fam_d)):
        A[0, col] = np.sum(opt["Dx_s"][fam] * opt["betx_s"][fam]) / (4 * math.pi)
        A[1, col] = -np.sum(opt["Dx_s"][fam] * opt["bety_s"][fam]) / (4 * math.pi)
    k2f, k2d = np.linalg.solve(A, np.array(chroma) - np.array(xnat))
    lat = build(float(k2f), float(k2d), sign, ksf, ksd)
    info = dict(opt=opt, k2l=(float(k2f), float(k2d)), xi_nat=xnat, cav_sign=sign, k1_straight=(ksf, ksd))
    return lat, info


def resonance_crossing_ring(dGg_per_turn, eps, k=45, phi=0.0):
    """Isolated spin resonance with a known strength, crossed at a known rate (recipe for the
    Froissart-Stora pin of the ramp): the 16-cell FODO ring, a cavity that adds
    dGg_per_turn to G*gamma_o every turn (phi_s = asin(1/4), A13) and a thin partial snake of angle
    mu = 2 pi eps about a horizontal axis (A14).  For the on-axis particle the one-turn spin map is
    R_y(2 pi G gamma) R_n(mu), whose tune gap at integer G gamma is eps.  Starts at G gamma = k - 1/2;
    returns (lattice, beam, turns to reach k + 1/2)."""
    dE = dGg_per_turn * MASS_PROTON_EV / G_PROTON
    els = list(fodo_ring(16, rf=cavity(4.0 * dE, 12.0, math.asin(0.25), +1.0)))
    els.append(snake(2.0 * math.pi * eps, phi))
    return lattice(els), beam((k - 0.5) / G_PROTON), int(round(1.0 / dGg_per_turn))


# ------------------------------------------------------------------------------------------------
# the five BASELINE.json configurations (1-based)
# ------------------------------------------------------------------------------------------------
def gamma_for_Ggamma(Gg, G=G_PROTON):
    return Gg / G


def config(i, n_particles=None, n_turns=None):
    """Returns dict(name, lattice, beam, state[9,n], split, n_slices, depth, n_turns, info)."""
    if i == 1:
        n = n_particles or 64
        lat = fodo_ring(16)
        st = gaussian_bunch(0, n, 25.0, 1e-3, 1e-4, 1e-3, 1e-4, 1e-4, 0.0, "vertical")
        return dict(name="cfg1_tiny_fodo", lattice=lat, beam=beam(25.0), state=st, split=SPLIT_BEND_KICK,
                    n_slices=4, depth=3, n_turns=n_turns or 10, info={})
    if i == 2:
        n = n_particles or 4096
        lat0 = fodo_ring(64)
        opt = linear_optics(lat0)
        sign = 1.0 if 25.0 > opt["gamma_t"] else -1.0
        lat = fodo_ring(64, sextupole_k2l=0.2, rf=cavity(300e3, 360.0, 0.0, sign))   # A23
        st = gaussian_bunch(1, n, 25.0, 1e-3, 1e-4, 1e-3, 1e-4, 3e-4, 0.1, "sphere")
        return dict(name="cfg2_nonlinear_rf", lattice=lat, beam=beam(25.0), state=st, split=SPLIT_MATRIX_KICK,
                    n_slices=8, depth=4, n_turns=n_turns or 1000, info=dict(opt=opt))
    if i in (3, 4, 5):
        Gg = {3: 45.5, 4: 45.0, 5: 45.5}[i]
        g0 = gamma_for_Ggamma(Gg)
        phi_s = math.asin(1.0 / 3.0) if i == 4 else 0.0            # A13: 100 keV/turn at 300 kV
        lat, info = rhic_like_ring(g0, snakes=(i != 5), phi_s=phi_s)
        n = n_particles or {3: 65536, 4: 1 << 20, 5: 262144}[i]
        st = matched_bunch(i - 1, n, g0, info["opt"], 10e-6, 5e-4, 0.1, "vertical")
        nt = n_turns or {3: 1000, 4: 5000, 5: 100}[i]
        name = {3: "cfg3_rhic_like", 4: "cfg4_ramp", 5: "cfg5_sweep"}[i]
        return dict(name=name, lattice=lat, beam=beam(g0), state=st, split=SPLIT_BEND_KICK, n_slices=8, depth=4,
                    n_turns=nt, info=info)
    raise ValueError("config index must be 1..5")


def sweep_pairs():
    """Config 5: valid (n_slices, depth) pairs, 2^(depth-1) | n_slices (A4): 27 pairs."""
    return [(N, d) for N in (1, 2, 4, 8, 16, 32, 64) for d in range(1, 7) if N % (1 << (d - 1)) == 0]
