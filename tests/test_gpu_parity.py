"""GPU parity: the CUDA path, called through the C ABI (ctypes binding), against the CPU oracle on the
same seeded inputs, element by element.

Metrics (tests/parity_metrics.py): for an orbit coordinate c the bunch-scale error
max_j |gpu - oracle| / max_j |oracle_c| and, on the BASELINE configurations, the per-particle error
|gpu_j - oracle_j| / max(|oracle_cj|, rms_c); for spin components, absolute.  Tolerances from
BASELINE.json north_star: 1e-12 after one turn, 1e-9 after 100 turns; bunch polarization within 1e-6
for the near-resonance and ramp configs.  The oracle runs its literal formulas in long double (see
gst_oracle.hpp header).  The configurations' full lengths are in tests/test_gpu_parity_long.py.
"""
import math

import numpy as np
import pytest

from paper_1501_03450_b200 import workloads as W
from parity_metrics import orbit_err, orbit_err_per_particle, spin_err

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def gst():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1501_03450_b200 import gst as g
    g.lib()
    return g


@pytest.fixture(scope="module")
def O():
    from oracle import oracle
    oracle.lib()
    return oracle


def gpu_track(gst, lat, beam, state, n_turns, split, n_slices, depth, chunks=None, static=False, want_kernel=None,
              lean=False):
    """depth >= 1: gst_track; depth = W.PWC_HALF_SLICE / W.PWC_DKSKD (0 / -1): gst_track_pwc"""
    L = gst.Lattice(lat, beam)
    d = torch.tensor(state, dtype=torch.float64, device="cuda").contiguous()
    b = gst.Bunch(d)
    if static or lean:
        b.set_launch(gst.LAUNCH_LEAN if lean else gst.LAUNCH_STATIC)
    for nt in (chunks or [n_turns]):
        if depth >= 1:
            b.track(L, nt, split, n_slices, depth)
        else:
            b.track_pwc(L, nt, split, n_slices, depth)
    b.status()
    if want_kernel is not None:
        assert b.last_kernel() == want_kernel, b.last_kernel()
    pol, nlost = b.polarization()
    emit = b.emittance()
    lost = b.lost()
    g1, turn = b.reference()
    assert turn == n_turns
    out = d.cpu().numpy()
    b.close()
    L.close()
    return out, lost, pol, emit, g1


def mixed_lattice(ramp=True):
    """Every element type, both quad signs, a mis-powered bend, skew terms, slice multipliers."""
    ang = 2 * math.pi / 24
    els = [W.drift(0.7), W.quad(0.6, +0.35), W.thin_sextupole(0.4), W.drift(0.4),
           W.sbend(1.8, ang, eta=1.0), W.snake(math.pi, math.radians(45)),
           W.multipole(0.3, kn=(0.02, 0.9, -4.0, 30.0), ks=(0.01, -0.5, 3.0, -20.0), slice_mult=2),
           W.quad(0.6, -0.33, slice_mult=4), W.thin_multipole((0.001, -0.3, 2.0, 10.0), (0.002, 0.2, -1.0, 5.0)),
           W.marker(), W.drift(0.9), W.sbend(1.8, ang, eta=1.002),
           W.cavity(2e6, 8.0, math.asin(0.2) if ramp else 0.0, +1.0), W.drift(0.5),
           W.snake(2.0, math.radians(-30))]
    return W.lattice(els * 3)


# ---------------------------------------------------------------------------------------------
# config 1 (full) and config 2
# ---------------------------------------------------------------------------------------------
def test_config1_one_turn_and_ten_turns(gst, O):
    c = W.config(1)
    for turns, tol in ((1, 1e-12), (10, 1e-11)):
        ref, rlost, _ = O.track(c["lattice"], c["beam"], c["state"], turns, c["split"], c["n_slices"], c["depth"])
        got, lost, pol, emit, _ = gpu_track(gst, c["lattice"], c["beam"], c["state"], turns, c["split"], c["n_slices"], c["depth"])
        assert not rlost.any() and not lost.any()
        assert orbit_err(got, ref) < tol, (turns, orbit_err(got, ref))
        assert orbit_err_per_particle(got, ref) < tol, (turns, orbit_err_per_particle(got, ref))
        assert spin_err(got, ref) < tol, (turns, spin_err(got, ref))
        rp, _ = O.polarization(ref)
        assert np.max(np.abs(pol - rp)) < 1e-13
        assert np.max(np.abs(emit / O.emittance(ref) - 1)) < 1e-11


def test_config2_one_turn_full_bunch(gst, O):
    c = W.config(2)
    ref, rlost, _ = O.track(c["lattice"], c["beam"], c["state"], 1, c["split"], c["n_slices"], c["depth"])
    got, lost, pol, emit, _ = gpu_track(gst, c["lattice"], c["beam"], c["state"], 1, c["split"], c["n_slices"], c["depth"])
    assert not rlost.any() and not lost.any()
    assert orbit_err(got, ref) < 1e-12, orbit_err(got, ref)
    assert orbit_err_per_particle(got, ref) < 1e-12, orbit_err_per_particle(got, ref)
    assert spin_err(got, ref) < 1e-12, spin_err(got, ref)


def test_config2_hundred_turns(gst, O):
    c = W.config(2, n_particles=192)
    ref, rlost, _ = O.track(c["lattice"], c["beam"], c["state"], 100, c["split"], c["n_slices"], c["depth"])
    got, lost, pol, emit, _ = gpu_track(gst, c["lattice"], c["beam"], c["state"], 100, c["split"], c["n_slices"], c["depth"])
    assert not rlost.any() and not lost.any()
    assert orbit_err(got, ref) < 1e-9, orbit_err(got, ref)
    assert orbit_err_per_particle(got, ref) < 1e-9, orbit_err_per_particle(got, ref)
    assert spin_err(got, ref) < 1e-9, spin_err(got, ref)


# ---------------------------------------------------------------------------------------------
# every split x depth on a lattice with every element type; ragged particle count
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("split", [W.SPLIT_DRIFT_KICK, W.SPLIT_BEND_KICK, W.SPLIT_MATRIX_KICK,
                                   W.SPLIT_DRIFT_KICK_4, W.SPLIT_BEND_KICK_4, W.SPLIT_MATRIX_KICK_4])
@pytest.mark.parametrize("depth,n_slices", [(1, 1), (1, 3), (2, 2), (3, 4), (4, 8), (5, 16), (6, 32)])
def test_all_splits_depths_all_element_types(gst, O, split, depth, n_slices):
    lat = mixed_lattice()
    bm = W.beam(12.0)
    n = 200                                   # 3 full blocks of 64 and a ragged tail of 8
    st = W.gaussian_bunch(7, n, 12.0, 2e-3, 3e-4, 2e-3, 3e-4, 5e-4, 0.05, "sphere")
    ref, rlost, g_ref = O.track(lat, bm, st, 2, split, n_slices, depth)
    # 200 particles take a small-bunch kernel: orbit and spin in two warps for the second-order splits, else the fused
    # kernel with registers to spare; the fused variants (the one large bunches get included) must give the same
    auto = "track_split_kernel" if split < 3 else "track_kernel_fat"
    got, lost, pol, emit, g_gpu = gpu_track(gst, lat, bm, st, 2, split, n_slices, depth, want_kernel=auto)
    fat = gpu_track(gst, lat, bm, st, 2, split, n_slices, depth, static=True, want_kernel="track_kernel_fat")
    lean = gpu_track(gst, lat, bm, st, 2, split, n_slices, depth, lean=True, want_kernel="track_kernel")
    assert not rlost.any() and not lost.any()
    assert orbit_err(got, ref) < 2e-12, orbit_err(got, ref)
    assert spin_err(got, ref) < 2e-12, spin_err(got, ref)
    assert abs(g_gpu - g_ref) < 1e-12 * g_ref
    assert np.max(np.abs(np.linalg.norm(got[6:9], axis=0) - 1)) < 1e-12     # A9: |S| = 1 without renormalising
    for other in (fat, lean):
        assert orbit_err(other[0], ref) < 2e-12 and spin_err(other[0], ref) < 2e-12 and other[4] == g_gpu
        # the same source compiled again: the kernels differ by the compiler's choice of fused multiply-adds only
        assert orbit_err(other[0], got) < 1e-13 and spin_err(other[0], got) < 1e-13


@pytest.mark.parametrize("split", [W.SPLIT_DRIFT_KICK_4, W.SPLIT_BEND_KICK_4, W.SPLIT_MATRIX_KICK_4])
def test_order4_config3_ring_and_accuracy_gain(gst, O, split):
    """Fourth-order slice maps on the RHIC-like ring: parity with the oracle, and the orbit
    after 5 turns is closer to the 64-slice matrix-kick result than the second-order map's at equal slicing."""
    c = W.config(5, n_particles=96)
    ref, rlost, _ = O.track(c["lattice"], c["beam"], c["state"], 5, split, 4, 3)
    got, lost, pol, emit, _ = gpu_track(gst, c["lattice"], c["beam"], c["state"], 5, split, 4, 3)
    assert not rlost.any() and not lost.any()
    assert orbit_err(got, ref) < 1e-11 and spin_err(got, ref) < 1e-11, (orbit_err(got, ref), spin_err(got, ref))
    fine = gpu_track(gst, c["lattice"], c["beam"], c["state"], 5, W.SPLIT_MATRIX_KICK_4, 64, 3)[0]
    second = gpu_track(gst, c["lattice"], c["beam"], c["state"], 5, split - 3, 4, 3)[0]
    e4 = np.sqrt(np.mean((got[0] - fine[0]) ** 2))
    e2 = np.sqrt(np.mean((second[0] - fine[0]) ** 2))
    assert e4 < 0.2 * e2, (e4, e2)


@pytest.mark.parametrize("split", [W.SPLIT_DRIFT_KICK, W.SPLIT_BEND_KICK, W.SPLIT_MATRIX_KICK])
@pytest.mark.parametrize("order", [W.PWC_HALF_SLICE, W.PWC_DKSKD])
@pytest.mark.parametrize("n_slices", [1, 3, 8])
def test_pwc_mid_slice_integrators_all_element_types(gst, O, split, order, n_slices):
    """gst_track_pwc (section 4.1, (37)) against the oracle, every element type."""
    lat = mixed_lattice()
    bm = W.beam(12.0)
    st = W.gaussian_bunch(13, 200, 12.0, 2e-3, 3e-4, 2e-3, 3e-4, 5e-4, 0.05, "sphere")
    ref, rlost, g_ref = O.track(lat, bm, st, 2, split, n_slices, order)
    got, lost, pol, emit, g_gpu = gpu_track(gst, lat, bm, st, 2, split, n_slices, order)
    assert not rlost.any() and not lost.any()
    assert orbit_err(got, ref) < 2e-12, orbit_err(got, ref)
    assert spin_err(got, ref) < 2e-12, spin_err(got, ref)
    assert abs(g_gpu - g_ref) < 1e-12 * g_ref


def test_pwc_rejects_fourth_order_splits(gst):
    c = W.config(1)
    L = gst.Lattice(c["lattice"], c["beam"])
    b = gst.Bunch(torch.tensor(c["state"], dtype=torch.float64, device="cuda"))
    with pytest.raises(gst.GstError) as ei:
        b.track_pwc(L, 1, W.SPLIT_BEND_KICK_4, 4, W.PWC_HALF_SLICE)
    assert ei.value.status == gst.EINVAL
    b.close()
    L.close()


def test_thin_fringe_spin_kicks(gst, O):
    """GST_FRINGE (41) P:561 around every thick magnet of the mixed lattice."""
    els = []
    for e in mixed_lattice():
        els += W.with_fringes(e) if int(e["type"]) in (W.SBEND, W.QUAD, W.MULTIPOLE) else [e]
    lat = W.lattice(els)
    bm = W.beam(12.0)
    st = W.gaussian_bunch(17, 200, 12.0, 2e-3, 3e-4, 2e-3, 3e-4, 5e-4, 0.05, "sphere")
    ref, rlost, _ = O.track(lat, bm, st, 2, W.SPLIT_MATRIX_KICK, 4, 3)
    plain, _, _ = O.track(mixed_lattice(), bm, st, 2, W.SPLIT_MATRIX_KICK, 4, 3)
    got, lost, pol, emit, _ = gpu_track(gst, lat, bm, st, 2, W.SPLIT_MATRIX_KICK, 4, 3)
    assert not rlost.any() and not lost.any()
    assert orbit_err(got, ref) < 2e-12 and spin_err(got, ref) < 2e-12, (orbit_err(got, ref), spin_err(got, ref))
    assert spin_err(plain, ref) > 1e-6                       # the kicks are not a no-op on this bunch
    assert np.array_equal(plain[:6], ref[:6])                # and leave the orbit alone


@pytest.mark.parametrize("depth,n_slices", [(1, 3), (3, 4), (4, 8), (6, 32), (W.PWC_HALF_SLICE, 4), (W.PWC_DKSKD, 4)])
def test_solenoids_in_a_ring(gst, O, depth, n_slices):
    """GST_SOLENOID: body (34), kinetic momentum in Omega (36), fringe kicks (40)."""
    els = list(mixed_lattice())
    els.insert(3, W.solenoid(2.1, 0.2))                      # the paper's 1.3 T x 2.1 m magnet at a few GeV
    els.insert(20, W.solenoid(0.8, -0.35, slice_mult=2))
    lat = W.lattice(els)
    bm = W.beam(3.0)
    st = W.gaussian_bunch(19, 200, 3.0, 3e-3, 5e-4, 3e-3, 5e-4, 5e-4, 0.05, "sphere")
    ref, rlost, _ = O.track(lat, bm, st, 2, W.SPLIT_BEND_KICK, n_slices, depth)
    got, lost, pol, emit, _ = gpu_track(gst, lat, bm, st, 2, W.SPLIT_BEND_KICK, n_slices, depth)
    assert not rlost.any() and not lost.any()
    assert orbit_err(got, ref) < 2e-12 and spin_err(got, ref) < 2e-12, (orbit_err(got, ref), spin_err(got, ref))


@pytest.mark.parametrize("depth,n_slices", [(1, 3), (3, 4), (4, 8), (6, 32), (W.PWC_HALF_SLICE, 4), (W.PWC_DKSKD, 4)])
def test_rectangular_bends_in_a_ring(gst, O, depth, n_slices):
    """GST_RBEND: rotations (17), fringe map (15) and spin kick (42), body (13), offsets (18)(19)."""
    els = list(mixed_lattice())
    els.insert(2, W.rbend(2.4, 0.12))                         # symmetric
    els.insert(15, W.rbend(1.6, 0.09, 0.07, -0.02, slice_mult=2))   # asymmetric: offset (18)
    els.insert(30, W.rbend(2.0, -0.08))                       # bends the other way
    lat = W.lattice(els)
    bm = W.beam(12.0)
    st = W.gaussian_bunch(23, 200, 12.0, 2e-3, 3e-4, 2e-3, 3e-4, 5e-4, 0.05, "sphere")
    ref, rlost, g_ref = O.track(lat, bm, st, 2, W.SPLIT_BEND_KICK, n_slices, depth)
    got, lost, pol, emit, g_gpu = gpu_track(gst, lat, bm, st, 2, W.SPLIT_BEND_KICK, n_slices, depth)
    assert not rlost.any() and not lost.any()
    assert orbit_err(got, ref) < 2e-12 and spin_err(got, ref) < 2e-12, (orbit_err(got, ref), spin_err(got, ref))
    assert abs(g_gpu - g_ref) < 1e-12 * g_ref                 # the cavity sees the same circumference (arc lengths)


@pytest.mark.parametrize("split", [W.SPLIT_MATRIX_KICK, W.SPLIT_MATRIX_KICK_4])
def test_matrix_kick_at_large_transverse_momenta(gst, O, split):
    """The matrix-kick quadrupole takes 1/Ps from a series in pt^2/P^2 up to 2^-13 (angles of 11 mrad) and from the
    exact forms beyond (csrc/track_kernel.cuh: QuadMK): a bunch with angles from 0 to 47 mrad exercises both, in one
    warp, in the small-bunch and in the occupancy-oriented build of the kernel."""
    lat = W.lattice([W.drift(0.3), W.quad(0.5, +0.8), W.drift(0.2), W.quad(0.5, -0.8), W.drift(0.3)] * 2)
    bm = W.beam(5.0)
    st = W.gaussian_bunch(3, 200, 5.0, 2e-3, 2e-2, 2e-3, 2e-2, 1e-3, 0.01, "sphere")
    st[1, :40] *= 0.01                                   # some particles well inside the series' range
    st[3, :40] *= 0.01
    eps = (st[1] ** 2 + st[3] ** 2)
    assert (eps < 1e-5).sum() >= 30 and (eps > 2e-4).sum() >= 100
    ref, rlost, _ = O.track(lat, bm, st, 1, split, 8, 4)
    assert not rlost.any()
    for lean in (False, True):
        got, lost, *_ = gpu_track(gst, lat, bm, st, 1, split, 8, 4, lean=lean)
        assert not lost.any()
        assert orbit_err(got, ref) < 1e-12 and orbit_err_per_particle(got, ref) < 1e-12, (lean, orbit_err_per_particle(got, ref))
        assert spin_err(got, ref) < 1e-12, (lean, spin_err(got, ref))


def test_large_angle_per_slice_takes_the_sincos_branch(gst, O):
    # one slice through a strong bend at high G*gamma: rotation angle per edge > 1.4 rad
    lat = W.lattice([W.sbend(9.45, 0.2), W.drift(1.0)])
    bm = W.beam(W.gamma_for_Ggamma(45.5))
    st = W.gaussian_bunch(3, 70, bm["gamma0"], 1e-3, 1e-4, 1e-3, 1e-4, 1e-4, 0.0, "sphere")
    ref, _, _ = O.track(lat, bm, st, 1, W.SPLIT_BEND_KICK, 1, 1)
    got, lost, *_ = gpu_track(gst, lat, bm, st, 1, W.SPLIT_BEND_KICK, 1, 1)
    assert spin_err(got, ref) < 1e-12 and orbit_err(got, ref) < 1e-12


# ---------------------------------------------------------------------------------------------
# edge cases
# ---------------------------------------------------------------------------------------------
def test_empty_and_single_particle_bunches(gst, O):
    c = W.config(1)
    L = gst.Lattice(c["lattice"], c["beam"])
    d0 = torch.zeros((9, 0), dtype=torch.float64, device="cuda")
    b0 = gst.Bunch(d0)
    b0.track(L, 3, c["split"], 4, 3)
    pol, nl = b0.polarization()
    assert nl == 0 and np.all(pol == 0)
    b0.close()
    st = c["state"][:, :1].copy()
    ref, _, _ = O.track(c["lattice"], c["beam"], st, 3, c["split"], 4, 3)
    got, lost, *_ = gpu_track(gst, c["lattice"], c["beam"], st, 3, c["split"], 4, 3)
    assert orbit_err(got, ref) < 1e-12 and spin_err(got, ref) < 1e-12
    L.close()


def test_invalid_arguments_are_rejected(gst):
    c = W.config(1)
    L = gst.Lattice(c["lattice"], c["beam"])
    d = torch.tensor(c["state"], dtype=torch.float64, device="cuda")
    b = gst.Bunch(d)
    for args in ((1, 1, 4, 0), (1, 1, 4, 7), (1, 1, 0, 1), (1, 6, 4, 1), (1, 1, 4, 4), (-1, 1, 4, 1)):
        with pytest.raises(gst.GstError) as ei:
            b.track(L, *args)
        assert ei.value.status == gst.EINVAL
    bad = c["lattice"].copy()
    bad[1]["kn"][0] = 0.0
    with pytest.raises(gst.GstError):
        gst.Lattice(bad, c["beam"])
    bad = c["lattice"].copy()
    bad[3]["h"] = 0.0
    with pytest.raises(gst.GstError):
        gst.Lattice(bad, c["beam"])
    bad = c["lattice"].copy()
    bad[0]["type"] = 11
    with pytest.raises(gst.GstError):
        gst.Lattice(bad, c["beam"])
    b.close()
    L.close()


def test_lost_particles_are_flagged_identically_and_excluded_from_reductions(gst, O):
    c = W.config(1)
    st = c["state"].copy()
    st[1, 5] = 1.5          # |Px| > P: square root of a negative number in the first element (A15)
    st[3, 17] = -2.0
    ref, rlost, _ = O.track(c["lattice"], c["beam"], st, 2, c["split"], 4, 3)
    got, lost, pol, emit, _ = gpu_track(gst, c["lattice"], c["beam"], st, 2, c["split"], 4, 3)
    assert rlost[5] and rlost[17]
    assert np.array_equal(lost.astype(bool), rlost.astype(bool))
    keep = ~rlost.astype(bool)
    assert orbit_err(got[:, keep], ref[:, keep]) < 1e-12
    rp, nl = O.polarization(ref, rlost)
    assert np.max(np.abs(pol - rp)) < 1e-13
    assert np.max(np.abs(emit / O.emittance(ref, rlost) - 1)) < 1e-11


def test_shard_records_leave_lost_particles_out(gst, O):
    """gst_moments after tracking, two shards with one lost particle each: the summed record reports the bunch without
    them (A15, A18, A19), as the oracle's reductions over the whole tracked bunch do."""
    c = W.config(1)
    st = c["state"].copy()
    st[1, 5] = 1.5
    st[3, 40] = -2.0
    ref, rlost, _ = O.track(c["lattice"], c["beam"], st, 2, c["split"], 4, 3)
    assert rlost[5] and rlost[40] and rlost.sum() == 2
    L = gst.Lattice(c["lattice"], c["beam"])
    total = np.zeros(gst.MOMENTS_LEN)
    for lo, hi in ((0, 23), (23, st.shape[1])):
        d = torch.tensor(st[:, lo:hi], dtype=torch.float64, device="cuda").contiguous()
        b = gst.Bunch(d)
        b.track(L, 2, c["split"], 4, 3)
        rec = b.moments()
        assert rec[3] == hi - lo - 1
        total += rec
        b.close()
    L.close()
    pol, emit, alive = gst.moments_finish(total)
    rp, nl = O.polarization(ref, rlost)
    assert alive == st.shape[1] - 2 and nl == 2
    assert np.max(np.abs(pol - rp)) < 1e-13
    assert np.max(np.abs(emit / O.emittance(ref, rlost) - 1)) < 1e-11


def test_chain_rotation_is_bit_identical_to_the_static_launch(gst):
    """65 553 particles fill the sub-partitions unevenly, so the default launch rotates the warps of particles
    over the warp slots in chunks of turns (csrc/track_chain_kernel.cuh); state, lost flags and the ramping
    reference energy must come out exactly as from the static launch."""
    lat = mixed_lattice(ramp=True)
    bm = W.beam(12.0)
    n = 65536 + 17
    st = W.gaussian_bunch(29, n, 12.0, 2e-3, 3e-4, 2e-3, 3e-4, 5e-4, 0.05, "sphere")
    st[1, 5] = 1.5                                   # lost in the first chunk
    st[3, 40000] = -2.0
    rot = gpu_track(gst, lat, bm, st, 50, W.SPLIT_BEND_KICK, 4, 3, want_kernel="track_chain_kernel")
    sta = gpu_track(gst, lat, bm, st, 50, W.SPLIT_BEND_KICK, 4, 3, static=True, want_kernel="track_kernel")
    assert np.array_equal(rot[1], sta[1]) and rot[1][5] and rot[1][40000]
    keep = ~sta[1].astype(bool)
    assert np.array_equal(rot[0][:, keep], sta[0][:, keep])
    assert np.array_equal(rot[2], sta[2]) and rot[4] == sta[4]


@pytest.mark.parametrize("n,turns", [(37920, 16), (47360, 17), (75712, 33), (75744, 16), (65536, 40), (80000, 17),
                                     (262144 + 5, 16)])
def test_chain_rotation_edge_sizes(gst, n, turns):
    """Rotating launch at the edges of its plan: just over 2 warps per sub-partition, a shift of 2 slots, one chain short
    of a full chip, chunk counts that do not divide the turns, more chains than warp slots (1.06 and 3.46 waves)."""
    lat = mixed_lattice(ramp=True)
    bm = W.beam(12.0)
    st = W.gaussian_bunch(31, n, 12.0, 2e-3, 3e-4, 2e-3, 3e-4, 5e-4, 0.05, "sphere")
    rot = gpu_track(gst, lat, bm, st, turns, W.SPLIT_MATRIX_KICK, 2, 2)
    sta = gpu_track(gst, lat, bm, st, turns, W.SPLIT_MATRIX_KICK, 2, 2, static=True, want_kernel="track_kernel")
    assert not sta[1].any() and np.array_equal(rot[1], sta[1])
    assert np.array_equal(rot[0], sta[0]) and rot[4] == sta[4]


@pytest.mark.parametrize("split", [W.SPLIT_DRIFT_KICK, W.SPLIT_BEND_KICK, W.SPLIT_MATRIX_KICK])
@pytest.mark.parametrize("depth,n_slices", [(1, 1), (2, 2), (4, 8), (6, 32)])
def test_chain_rotation_every_split_and_low_depths(gst, split, depth, n_slices):
    """The rotating launch for instantiations whose register count (and hence occupancy) differs from the
    headline kernel's: the slot numbering must hold for any spread of the blocks over the SMs
    (csrc/track_chain_kernel.cuh), so state, lost flags and reference energy equal the static launch's."""
    lat = mixed_lattice(ramp=True)
    bm = W.beam(12.0)
    n = 65536 + 17
    st = W.gaussian_bunch(37, n, 12.0, 2e-3, 3e-4, 2e-3, 3e-4, 5e-4, 0.05, "sphere")
    st[1, 77] = 1.5
    turns = 16 if depth > 4 else 24
    rot = gpu_track(gst, lat, bm, st, turns, split, n_slices, depth, want_kernel="track_chain_kernel")
    sta = gpu_track(gst, lat, bm, st, turns, split, n_slices, depth, static=True, want_kernel="track_kernel")
    assert np.array_equal(rot[1], sta[1]) and rot[1][77]
    keep = ~sta[1].astype(bool)
    assert np.array_equal(rot[0][:, keep], sta[0][:, keep])
    assert np.array_equal(rot[2], sta[2]) and rot[4] == sta[4]


@pytest.mark.parametrize("split", [W.SPLIT_DRIFT_KICK, W.SPLIT_BEND_KICK, W.SPLIT_MATRIX_KICK])
@pytest.mark.parametrize("depth,n_slices", [(1, 1), (1, 3), (2, 2), (3, 4), (4, 8), (5, 16), (6, 32)])
def test_two_warp_kernel_agrees_with_the_fused_kernel(gst, O, split, depth, n_slices):
    """Small bunches take the kernel that gives a particle's orbit and its spin to two warps
    (csrc/track_split_kernel.cuh): the same functions as the fused kernel, compiled a second time, so the two agree to
    rounding; lost flags and the ramping reference energy exactly.  Every element type, a ragged last block, lost
    particles in the first and in the last block, enough turns for the ring of rotation vectors to wrap many times;
    and the two-warp kernel against the oracle."""
    ang = 2 * math.pi / 24
    fr = ((0.3, 2.0, 0.0, 0.0), (0.1, 0.0, 0.0, 0.0))
    lat = np.concatenate([mixed_lattice(ramp=True), W.lattice([
        W.solenoid(0.8, 0.12), W.drift(0.3), W.rbend(1.5, ang / 2), W.fringe(+1.0, 0.02, *fr), W.quad(0.5, 0.2),
        W.fringe(-1.0, 0.02, *fr), W.marker(), W.drift(0.2)])])
    bm = W.beam(12.0)
    n = 3 * 32 + 5
    st = W.gaussian_bunch(41, n, 12.0, 2e-3, 3e-4, 2e-3, 3e-4, 5e-4, 0.05, "sphere")
    st[1, 3] = 1.5
    st[3, n - 2] = -2.0
    turns = 3
    two = gpu_track(gst, lat, bm, st, turns, split, n_slices, depth, want_kernel="track_split_kernel")
    one = gpu_track(gst, lat, bm, st, turns, split, n_slices, depth, static=True, want_kernel="track_kernel_fat")
    assert np.array_equal(two[1], one[1]) and two[1][3] and two[1][n - 2] and two[1].sum() == 2
    keep = ~one[1].astype(bool)
    assert orbit_err(two[0][:, keep], one[0][:, keep]) < 1e-13
    assert spin_err(two[0][:, keep], one[0][:, keep]) < 1e-13
    assert np.array_equal(two[0][:, ~keep], st[:, ~keep])          # a lost particle's entries are left alone (gst.h)
    assert np.max(np.abs(two[2] - one[2])) < 1e-13 and two[4] == one[4]
    ref, rlost, g_ref = O.track(lat, bm, st, turns, split, n_slices, depth)
    assert np.array_equal(two[1].astype(bool), rlost.astype(bool))
    assert orbit_err(two[0][:, keep], ref[:, keep]) < 1e-11 and spin_err(two[0][:, keep], ref[:, keep]) < 1e-11


@pytest.mark.parametrize("n,turns,kernel", [(1, 1, "track_split_kernel"), (14208, 1, "track_split_kernel"), (14209, 1, "track_kernel_fat"),
                                            (37888, 16, "track_kernel_fat"), (37889, 1, "track_kernel"),
                                            (37920, 16, "track_chain_kernel"), (65536, 15, "track_kernel"),
                                            (65536, 16, "track_chain_kernel"), (148 * 8 * 64, 16, "track_kernel")])
def test_launch_planner_picks_the_kernel_by_bunch_size(gst, n, turns, kernel):
    """csrc/track_launch.cuh on a B200 (148 SMs): the two-warp kernel up to 3 warps of particles per SM, the small-bunch
    build of the fused kernel up to 2 warps per sub-partition, the rotating launch where one wave fills the
    sub-partitions unevenly and there are at least 16 turns, else one thread per particle with its slot for the whole
    call (a bunch that fills every warp slot exactly included)."""
    if torch.cuda.get_device_properties(0).multi_processor_count != 148:
        pytest.skip("the sizes are those of a 148-SM B200")
    lat = W.lattice([W.drift(1.0), W.quad(0.5, 0.3), W.drift(1.0), W.sbend(2.0, 0.1), W.quad(0.5, -0.3)])
    bm = W.beam(25.0)
    st = W.gaussian_bunch(3, n, 25.0, 1e-3, 1e-4, 1e-3, 1e-4, 1e-4, 0.05, "sphere")
    out, lost, pol, emit, g1 = gpu_track(gst, lat, bm, st, turns, W.SPLIT_BEND_KICK, 2, 2, want_kernel=kernel)
    assert not lost.any() and np.all(np.isfinite(out))


@pytest.mark.timeout(120)
@pytest.mark.parametrize("start,n", [(0, 1), (0, 15), (0, 16), (0, 17), (0, 32), (0, 1000), (2**32 - 32, 16), (2**32 - 32, 33),
                                     (2**32 - 64, 1000), (2**31 - 32, 100)])
def test_ring_of_the_two_warp_kernel_across_the_wrap_of_its_counter(gst, start, n):
    """The ring that carries rotation vectors from the orbit warp to the spin warp (csrc/track_split_kernel.cuh) counts
    its entries in 32 bits: 4.3e9 edges are under a million turns of a large ring in one gst_track.  Its protocol looks
    at the position within a half only, so the count may wrap; partial and exactly full last halves included."""
    from paper_1501_03450_b200 import gst_diag
    assert gst_diag.selftest_ring(start, n) == 0
    with pytest.raises(Exception):
        gst_diag.selftest_ring(start + 7, n)


def test_failed_rotating_launch_is_reported_by_every_synchronising_call(gst):
    """Fault injection (include/gst_diag.h): with a poll budget of one, the first warp that has to wait for a
    hand-off gives up as it would after a hang.  Every call that synchronises must then return GST_ECUDA once,
    launches enqueued behind the failure must do nothing, and the bunch must be usable again afterwards."""
    from paper_1501_03450_b200 import gst_diag
    lat = mixed_lattice(ramp=True)
    bm = W.beam(12.0)
    n = 65536
    st = W.gaussian_bunch(39, n, 12.0, 2e-3, 3e-4, 2e-3, 3e-4, 5e-4, 0.05, "sphere")
    want = gpu_track(gst, lat, bm, st, 32, W.SPLIT_BEND_KICK, 4, 3, want_kernel="track_chain_kernel")[0]
    L = gst.Lattice(lat, bm)
    calls = {"status": lambda b: b.status(), "polarization": lambda b: b.polarization(),
             "emittance": lambda b: b.emittance(), "lost": lambda b: b.lost()}
    for name, call in calls.items():
        d = torch.tensor(st, dtype=torch.float64, device="cuda").contiguous()
        b = gst.Bunch(d)
        gst_diag.chain_poll_limit(b, 1)
        b.track(L, 32, W.SPLIT_BEND_KICK, 4, 3)
        assert b.last_kernel() == "track_chain_kernel"
        b.track(L, 32, W.SPLIT_BEND_KICK, 4, 3)          # enqueued behind the failure: must not run
        with pytest.raises(gst.GstError) as ei:
            call(b)
        assert ei.value.status == gst.ECUDA and "track_chain_kernel" in str(ei.value), (name, str(ei.value))
        b.status()                                       # reported once, then clear
        # a checkpoint and a new reference make the bunch whole again (gst.h, "Errors")
        gst_diag.chain_poll_limit(b, 0)
        d.copy_(torch.tensor(st, dtype=torch.float64, device="cuda"))
        b.set_reference(bm, 0)
        b.track(L, 32, W.SPLIT_BEND_KICK, 4, 3)
        b.status()
        assert np.array_equal(d.cpu().numpy(), want), name
        b.close()
    L.close()


def test_bunch_and_lattice_handles_record_their_device(gst):
    """Entry points run on the device of their handle whatever the caller's current device is; with one GPU the
    check is that host memory is refused and that the guard leaves the current device alone."""
    c = W.config(1)
    L = gst.Lattice(c["lattice"], c["beam"])
    with pytest.raises(gst.GstError) as ei:
        import ctypes
        host = np.zeros((9, 8))
        h = ctypes.c_void_p()
        rows = [ctypes.c_void_p(host[i].ctypes.data) for i in range(9)]
        gst._check(gst.lib().gst_bunch_init(*rows, 8, ctypes.byref(h)))
    assert ei.value.status == gst.EINVAL
    before = torch.cuda.current_device()
    d = torch.tensor(c["state"], dtype=torch.float64, device="cuda").contiguous()
    b = gst.Bunch(d)
    b.track(L, 1, c["split"], 4, 3)
    b.status()
    assert torch.cuda.current_device() == before
    b.close()
    L.close()


def test_fig7_claims_through_the_c_abi(gst, capsys):
    """The paper's single-element study run on the GPU (studies.fig7): slope -2 without Romberg, slope -4
    with one iteration, and for the IR quadrupole "four slices plus two Romberg iterations yield a
    four-decade reduction"."""
    import argparse
    import json
    from paper_1501_03450_b200 import studies
    studies.fig7(argparse.Namespace(out=None))
    rows = [json.loads(l) for l in capsys.readouterr().out.splitlines() if l.startswith("{")]
    quad = {r["slices"]: r for r in rows if r["element"].startswith("IR quadrupole")}
    dip = {r["slices"]: r for r in rows if r["element"].startswith("arc dipole")}
    for tab in (quad, dip):
        for n in (4, 8, 16):
            assert 3.5 < tab[n]["pwc"] / tab[2 * n]["pwc"] < 4.5 and 3.5 < tab[n]["k0"] / tab[2 * n]["k0"] < 4.5
    for n in (8, 16, 32):
        assert 13 < quad[n]["k1"] / quad[2 * n]["k1"] < 19
    assert 14 < dip[16]["k1"] / dip[32]["k1"] < 19 and 14 < dip[32]["k1"] / dip[64]["k1"] < 19
    assert quad[4]["k2"] < 2e-4 * quad[4]["k0"]                     # four decades
    assert min(quad[128]["k3"], dip[128]["k3"]) < 1e-14            # round-off floor ~1e-15


@pytest.mark.parametrize("seed", range(8))
def test_random_lattices_of_every_element_type(gst, O, seed):
    """Seeded random lattices (every element type, random strengths, slice multipliers and order), a random split,
    slicing and spin scheme each: the CUDA path against the oracle."""
    rng = np.random.default_rng(1000 + seed)
    u = lambda a, b: float(rng.uniform(a, b))
    makers = [
        lambda: W.drift(u(0.1, 2.0)),
        lambda: W.quad(u(0.2, 0.8), u(0.03, 0.15) * rng.choice([-1, 1]), slice_mult=int(rng.integers(1, 3))),
        lambda: W.sbend(u(0.5, 3.0), u(0.01, 0.05) * rng.choice([-1, 1]), eta=u(0.998, 1.002)),
        lambda: W.rbend(u(0.5, 3.0), u(0.01, 0.05) * rng.choice([-1, 1])),
        lambda: W.multipole(u(0.1, 0.5), kn=(u(-0.05, 0.05), u(-2, 2), u(-30, 30), u(-300, 300)),
                            ks=(u(-0.05, 0.05), u(-2, 2), u(-30, 30), u(-300, 300))),
        lambda: W.thin_multipole((u(-0.01, 0.01), u(-1, 1), u(-10, 10), u(-100, 100)), (u(-0.01, 0.01), u(-1, 1), u(-10, 10), u(-100, 100))),
        lambda: W.solenoid(u(0.3, 1.5), u(0.05, 0.2) * rng.choice([-1, 1])),
        lambda: W.fringe(float(rng.choice([-1, 1])), u(-0.05, 0.05), (u(-0.5, 0.5), u(-5, 5), 0.0, 0.0), (u(-0.5, 0.5), 0.0, 0.0, 0.0)),
        lambda: W.snake(u(0.5, 3.1), u(-1.5, 1.5)),
        lambda: W.cavity(u(1e4, 2e5), float(rng.integers(1, 20)), u(-0.3, 0.3), float(rng.choice([-1, 1]))),
        lambda: W.marker(),
    ]
    els = [makers[int(rng.integers(len(makers)))]() for _ in range(44)]     # 44 unique records: over the shared-memory table
    lat = W.lattice(els)
    gam = u(3.0, 30.0)
    bm = W.beam(gam)
    st = W.gaussian_bunch(2000 + seed, 150, gam, 1e-3, 1e-4, 1e-3, 1e-4, 5e-4, 0.05, "sphere")
    split = int(rng.integers(0, 6))
    depth = int(rng.choice([-1, 0, 1, 2, 3, 4])) if split < 3 else int(rng.integers(1, 5))
    n_slices = (1 << max(depth - 1, 0)) * int(rng.integers(1, 4))
    ref, rlost, g_ref = O.track(lat, bm, st, 2, split, n_slices, depth)
    got, lost, pol, emit, g_gpu = gpu_track(gst, lat, bm, st, 2, split, n_slices, depth)
    assert np.array_equal(lost.astype(bool), rlost.astype(bool))
    keep = ~rlost.astype(bool)
    assert keep.sum() >= 140
    # a random lattice is not a stable ring: two turns amplify rounding differences more than the FODO-like lattices do
    assert orbit_err(got[:, keep], ref[:, keep]) < 2e-11, (split, depth, n_slices, orbit_err(got[:, keep], ref[:, keep]))
    assert spin_err(got[:, keep], ref[:, keep]) < 2e-11, (split, depth, n_slices, spin_err(got[:, keep], ref[:, keep]))
    assert abs(g_gpu - g_ref) < 1e-12 * g_ref


@pytest.mark.parametrize("case", ["only_drifts", "only_markers", "trailing_drifts", "drift_before_every_type", "leading_and_split_drifts"])
def test_lattice_compiler_edge_cases(gst, O, case):
    """gst_lattice_create merges runs of drifts into the element behind them and drops markers (csrc/gst_api.cu); the
    oracle goes through the user's lattice element by element.  The edges: rings of drifts or markers only, drifts left
    at the end of the ring (a hard boundary: no wrap-around into the first element), a drift space in front of EVERY
    element type, drifts cut into pieces with markers between them."""
    ang = 2 * math.pi / 40
    if case == "only_drifts":
        els = [W.drift(0.5), W.drift(1.25), W.marker(), W.drift(0.25)]
    elif case == "only_markers":
        els = [W.marker(), W.marker()]
    elif case == "trailing_drifts":
        els = [W.quad(0.4, 0.5), W.drift(0.3), W.sbend(1.0, ang), W.drift(0.7), W.marker(), W.drift(0.2)]
    elif case == "drift_before_every_type":
        els = []
        for e in (W.quad(0.4, 0.5), W.quad(0.4, -0.5), W.sbend(1.0, ang), W.multipole(0.3, kn=(0.02, 0.9, -4.0, 30.0)),
                  W.thin_sextupole(0.4), W.cavity(1e5, 3.0, 0.1, +1.0), W.snake(2.0, 0.3), W.fringe(+1.0, 0.02, (0.3, 0, 0, 0)),
                  W.solenoid(0.8, 0.2), W.rbend(1.2, 0.05), W.marker()):
            els += [W.drift(0.37), e]
    else:
        els = [W.drift(0.2), W.marker(), W.drift(0.3), W.drift(0.1), W.quad(0.4, 0.5), W.drift(0.6), W.marker(), W.drift(0.4),
               W.sbend(1.0, ang), W.marker(), W.thin_sextupole(-0.3), W.drift(0.5)]
    lat = W.lattice(els)
    bm = W.beam(8.0)
    st = W.gaussian_bunch(61, 100, 8.0, 2e-3, 3e-4, 2e-3, 3e-4, 5e-4, 0.05, "sphere")
    L = gst.Lattice(lat, bm)
    assert L.steps_per_turn(4) == W.steps_per_turn(lat, 4)          # the metric counts the USER lattice
    L.close()
    for split in (W.SPLIT_DRIFT_KICK, W.SPLIT_BEND_KICK, W.SPLIT_MATRIX_KICK):
        ref, rlost, g_ref = O.track(lat, bm, st, 3, split, 4, 3)
        got, lost, pol, emit, g_gpu = gpu_track(gst, lat, bm, st, 3, split, 4, 3)
        assert not rlost.any() and not lost.any()
        assert orbit_err(got, ref) < 2e-12 and spin_err(got, ref) < 2e-12, (split, orbit_err(got, ref), spin_err(got, ref))
        assert abs(g_gpu - g_ref) < 1e-12 * g_ref


def test_lattice_with_hundreds_of_unique_elements(gst, O):
    """A ring whose magnets all differ slightly (as a real machine's do): 448 unique records = 287 kB of element
    table, read from global memory instead of shared memory; the sequence alone still fits."""
    rng = np.random.default_rng(77)
    els = []
    for e in W.fodo_ring(64):
        e = e.copy()
        if int(e["type"]) == W.QUAD:
            e["kn"][0] *= 1.0 + 1e-3 * rng.standard_normal()
        elif int(e["type"]) == W.SBEND:
            e["k0"] *= 1.0 + 1e-4 * rng.standard_normal()
        else:
            e["L"] *= 1.0 + 1e-3 * rng.standard_normal()
        els.append(e)
    lat = W.lattice(els)
    assert len(np.unique(lat)) > 400
    bm = W.beam(25.0)
    st = W.gaussian_bunch(41, 96, 25.0, 1e-3, 1e-4, 1e-3, 1e-4, 3e-4, 0.05, "sphere")
    ref, rlost, _ = O.track(lat, bm, st, 3, W.SPLIT_MATRIX_KICK, 4, 3)
    got, lost, pol, emit, _ = gpu_track(gst, lat, bm, st, 3, W.SPLIT_MATRIX_KICK, 4, 3)
    assert not rlost.any() and not lost.any()
    assert orbit_err(got, ref) < 5e-12 and spin_err(got, ref) < 5e-12, (orbit_err(got, ref), spin_err(got, ref))


def test_long_lattice_whose_sequence_does_not_fit_shared_memory(gst, O):
    """10 500 elements: the 42 kB sequence stays in global memory (prefetched one element ahead), the table is staged."""
    lat = W.fodo_ring(1500)
    assert len(lat) > 10000
    bm = W.beam(25.0)
    st = W.gaussian_bunch(43, 70, 25.0, 1e-3, 1e-4, 1e-3, 1e-4, 3e-4, 0.05, "sphere")
    ref, rlost, _ = O.track(lat, bm, st, 1, W.SPLIT_BEND_KICK, 2, 2)
    got, lost, pol, emit, _ = gpu_track(gst, lat, bm, st, 1, W.SPLIT_BEND_KICK, 2, 2)
    assert not rlost.any() and not lost.any()
    assert orbit_err(got, ref) < 2e-11 and spin_err(got, ref) < 2e-11, (orbit_err(got, ref), spin_err(got, ref))


def test_two_bunches_on_two_streams(gst):
    """Two gst_track calls in flight on different streams (both take the cooperative sequence launch, which needs
    the whole chip): they serialise instead of dead-locking, and give the single-stream results."""
    lat = mixed_lattice(ramp=True)
    bm = W.beam(12.0)
    sts = [W.gaussian_bunch(50 + k, 65536, 12.0, 2e-3, 3e-4, 2e-3, 3e-4, 5e-4, 0.05, "sphere") for k in range(2)]
    want = [gpu_track(gst, lat, bm, st, 32, W.SPLIT_BEND_KICK, 4, 3)[0] for st in sts]
    L = gst.Lattice(lat, bm)
    devs = [torch.tensor(st, dtype=torch.float64, device="cuda").contiguous() for st in sts]
    bunches = [gst.Bunch(d) for d in devs]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    torch.cuda.synchronize()
    for b, s in zip(bunches, streams):
        b.track(L, 32, W.SPLIT_BEND_KICK, 4, 3, stream=s)
    torch.cuda.synchronize()
    for b, d, w in zip(bunches, devs, want):
        assert b.last_kernel() == "track_chain_kernel"
        assert np.array_equal(d.cpu().numpy(), w)
        b.close()
    L.close()


def test_chunked_tracking_is_bit_identical_to_one_call(gst):
    lat = mixed_lattice(ramp=True)
    bm = W.beam(12.0)
    st = W.gaussian_bunch(9, 130, 12.0, 1e-3, 1e-4, 1e-3, 1e-4, 3e-4, 0.05, "sphere")
    a, *_ , ga = gpu_track(gst, lat, bm, st, 12, W.SPLIT_MATRIX_KICK, 4, 3)
    b, *_ , gb = gpu_track(gst, lat, bm, st, 12, W.SPLIT_MATRIX_KICK, 4, 3, chunks=[5, 4, 3])
    assert np.array_equal(a, b) and ga == gb


def test_host_buffer_entry_point_matches_device_path(gst):
    c = W.config(1)
    dev, lost, pol, *_ = gpu_track(gst, c["lattice"], c["beam"], c["state"], 4, c["split"], 4, 3)
    L = gst.Lattice(c["lattice"], c["beam"])
    host = [np.ascontiguousarray(c["state"][i]) for i in range(9)]
    hpol, nl = L.track_host(host, 4, c["split"], 4, 3)
    assert np.array_equal(np.stack(host), dev) and np.array_equal(hpol, pol) and nl == 0
    L.close()


def test_reductions_match_oracle_on_a_large_bunch(gst, O):
    rng = np.random.default_rng(12)
    n = 300_001
    st = rng.normal(size=(9, n)) * np.array([1e-3, 1e-4, 2e-3, 3e-4, 0.1, 1e-3, 1, 1, 1])[:, None]
    st[0] += 5e-3           # offset beam: the mean-subtracted second pass must handle it
    d = torch.tensor(st, dtype=torch.float64, device="cuda").contiguous()
    b = gst.Bunch(d)
    pol, nl = b.polarization()
    emit = b.emittance()
    rp, _ = O.polarization(st)
    assert nl == 0 and np.max(np.abs(pol - rp)) < 1e-14
    assert np.max(np.abs(emit / O.emittance(st) - 1)) < 1e-12
    b.close()


def test_shard_records_add_up_to_the_whole_bunch(gst, O):
    """the records of gst_moments of disjoint shards add; gst_moments_finish of the sum is the report of
    the whole bunch (the all-reduce of distributed.global_report on one device: three uneven shards, offset beam, one
    shard displaced against the others so that the between-shard term matters)."""
    rng = np.random.default_rng(13)
    n = 100_003
    st = rng.normal(size=(9, n)) * np.array([1e-3, 1e-4, 2e-3, 3e-4, 0.1, 1e-3, 1, 1, 1])[:, None]
    st[0] += 5e-3
    cuts = [0, 17, 40_000, n]
    st[2, cuts[2]:] += 1e-3
    st[3, cuts[2]:] -= 2e-4
    total = np.zeros(gst.MOMENTS_LEN)
    for lo, hi in zip(cuts[:-1], cuts[1:]):
        d = torch.tensor(st[:, lo:hi], dtype=torch.float64, device="cuda").contiguous()
        b = gst.Bunch(d)
        rec = b.moments()
        pol1, emit1, alive1 = gst.moments_finish(rec)              # a single record = the bunch's own reports
        pol, _ = b.polarization()
        assert alive1 == hi - lo and np.array_equal(pol1, pol)
        assert np.max(np.abs(emit1 / b.emittance() - 1)) < 1e-13
        total += rec
        b.close()
    pol, emit, alive = gst.moments_finish(total)
    rp, _ = O.polarization(st)
    assert alive == n and np.max(np.abs(pol - rp)) < 1e-14
    assert np.max(np.abs(emit / O.emittance(st) - 1)) < 1e-12, emit / O.emittance(st) - 1
    d = torch.tensor(st, dtype=torch.float64, device="cuda").contiguous()
    b = gst.Bunch(d)
    assert np.max(np.abs(emit / b.emittance() - 1)) < 1e-12
    b.close()


# ---------------------------------------------------------------------------------------------
# RHIC-like ring (configs 3, 4, 5): reduced sizes in full, full size on sampled particles
# ---------------------------------------------------------------------------------------------
def test_config3_reduced_per_particle_and_polarization(gst, O):
    c = W.config(3, n_particles=512)
    ref, rlost, _ = O.track(c["lattice"], c["beam"], c["state"], 20, c["split"], c["n_slices"], c["depth"])
    got, lost, pol, emit, _ = gpu_track(gst, c["lattice"], c["beam"], c["state"], 20, c["split"], c["n_slices"], c["depth"])
    assert not rlost.any() and not lost.any()
    assert orbit_err(got, ref) < 1e-10 and spin_err(got, ref) < 1e-10, (orbit_err(got, ref), spin_err(got, ref))
    rp, _ = O.polarization(ref)
    assert np.max(np.abs(pol - rp)) < 1e-9


def test_config4_ramp_reduced(gst, O):
    c = W.config(4, n_particles=256)
    ref, rlost, g_ref = O.track(c["lattice"], c["beam"], c["state"], 40, c["split"], c["n_slices"], c["depth"])
    got, lost, pol, emit, g_gpu = gpu_track(gst, c["lattice"], c["beam"], c["state"], 40, c["split"], c["n_slices"],
                                            c["depth"], chunks=[10, 10, 10, 10])
    assert not rlost.any() and not lost.any()
    assert abs(g_gpu - g_ref) < 1e-13 * g_ref
    assert abs(W.G_PROTON * (g_gpu - c["beam"]["gamma0"]) - 40 * 1.9108e-4) < 1e-6      # A13
    assert orbit_err(got, ref) < 1e-10 and spin_err(got, ref) < 1e-10, (orbit_err(got, ref), spin_err(got, ref))
    rp, _ = O.polarization(ref)
    assert np.max(np.abs(pol - rp)) < 1e-6


def test_ramp_through_an_isolated_resonance(gst, O):
    """Froissart-Stora crossing (tests/test_oracle_rf_reductions.py) on the CUDA path: particle 0 is on axis
    and must land on the closed form; the rest of the bunch (betatron and momentum spread) must agree with the
    oracle through the partial flip, bunch polarization within the north star's 1e-6 for ramp configs."""
    dGg, eps = 2.5e-4, 4.2e-3
    lat, bm, turns = W.resonance_crossing_ring(dGg, eps)
    st = W.gaussian_bunch(21, 64, bm["gamma0"], 1e-3, 1e-4, 1e-3, 1e-4, 1e-4, 0.01)
    st[:6, 0] = 0.0
    ref, rlost, g_ref = O.track(lat, bm, st, turns, W.SPLIT_BEND_KICK, 4, 3)
    got, lost, pol, emit, g_gpu = gpu_track(gst, lat, bm, st, turns, W.SPLIT_BEND_KICK, 4, 3)
    assert not rlost.any() and not lost.any()
    # gamma_o(n): the CUDA path carries E_o as a compensated sum (ref_energy_add), so 4000 gains later it is still the
    # correctly rounded value; a plain fp64 sum is 1.8e-13 off here and shifts the spin phases by 7.6e-8
    assert abs(g_gpu - g_ref) < 4e-16 * g_ref and abs(W.G_PROTON * g_gpu - 45.5) < 1e-11
    fs = 2 * math.exp(-math.pi ** 2 * eps ** 2 / dGg) - 1
    assert abs(got[7, 0] - fs) < 0.02 and np.max(np.abs(got[:6, 0])) == 0.0, (got[7, 0], fs)
    assert orbit_err(got, ref) < 1e-8 and spin_err(got, ref) < 1e-8, (orbit_err(got, ref), spin_err(got, ref))
    rp, _ = O.polarization(ref)
    assert np.max(np.abs(pol - rp)) < 1e-6


@pytest.mark.parametrize("split", [W.SPLIT_DRIFT_KICK, W.SPLIT_BEND_KICK, W.SPLIT_MATRIX_KICK])
def test_config5_sweep_points_reduced(gst, O, split):
    c = W.config(5, n_particles=128)
    for n_slices, depth in ((1, 1), (4, 3), (16, 5)):
        ref, rlost, _ = O.track(c["lattice"], c["beam"], c["state"], 3, split, n_slices, depth)
        got, lost, pol, *_ = gpu_track(gst, c["lattice"], c["beam"], c["state"], 3, split, n_slices, depth)
        assert not rlost.any() and not lost.any()
        assert orbit_err(got, ref) < 1e-11 and spin_err(got, ref) < 1e-11, (n_slices, depth, orbit_err(got, ref), spin_err(got, ref))
        rp, _ = O.polarization(ref)
        assert np.max(np.abs(pol - rp)) < 1e-6


def test_config5_reference_run(gst, O):
    """The sweep's reference by refinement (matrix-kick, 128 slices, depth 6; studies.py) equals the oracle's."""
    c = W.config(5, n_particles=24)
    ref, rlost, _ = O.track(c["lattice"], c["beam"], c["state"], 3, W.SPLIT_MATRIX_KICK, 128, 6)
    got, lost, pol, emit, _ = gpu_track(gst, c["lattice"], c["beam"], c["state"], 3, W.SPLIT_MATRIX_KICK, 128, 6)
    assert not rlost.any() and not lost.any()
    assert orbit_err(got, ref) < 1e-10 and spin_err(got, ref) < 1e-10, (orbit_err(got, ref), spin_err(got, ref))


def test_branch_free_rcp_and_rsqrt_are_accurate_to_a_few_ulp(gst):
    from paper_1501_03450_b200 import gst_diag
    rcp, rsq = gst_diag.selftest_math()
    assert 0 < rcp < 4.0 and 0 < rsq < 4.0, (rcp, rsq)
