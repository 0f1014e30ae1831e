"""gst_polarization_noalloc (include/gst.h): the allocation-free variant of the polarization reduction, whose scratch is
a fixed device array inside the library, against the existing path (gst_bunch_init + gst_polarization), on two calls in a
row.  Collected last on purpose (the suite runs with pytest -x): the file name sorts behind every other test file.

The scratch keeps the last call's contents, so the second call is SMALLER than the first and has lost particles: stale
partial sums of the first call sit behind the records the second call writes, and a reduction that read them, or that
counted excluded particles, would fail the comparison.  Tolerance: 1e-14 absolute on the polarization components and
modulus, the bound of test_gpu_parity.py::test_reductions_match_oracle_on_a_large_bunch (the two paths add the same
numbers in the same order up to 303 104 particles, so they normally agree to the last bit).
"""
import ctypes as C

import numpy as np
import pytest

from paper_1501_03450_b200 import workloads as W

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

TOL = 1e-14


@pytest.fixture(scope="module")
def gst():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1501_03450_b200 import gst as g
    g.lib()
    return g


def existing_path(gst, dev_state):
    """{Px, Py, Ps, |P|}, lost count and lost flags from a bunch bound to the state (allocates: gst_bunch_init)."""
    b = gst.Bunch(dev_state)
    pol, nlost = b.polarization()
    b.close()
    return pol, nlost


def test_no_alloc_polarization_matches_the_existing_path_on_two_calls_in_a_row(gst):
    out = torch.full((5,), float("nan"), dtype=torch.float64, device="cuda")

    # ---- call 1: 300 001 particles (1172 blocks and a ragged tail), spins all over the sphere, nobody lost
    n1 = 300_001
    st1 = W.gaussian_bunch(71, n1, 25.0, 1e-3, 1e-4, 1e-3, 1e-4, 3e-4, 0.05, "sphere")
    d1 = torch.tensor(st1, dtype=torch.float64, device="cuda").contiguous()
    want1, nlost1 = existing_path(gst, d1)
    gst.polarization_noalloc(d1[6], d1[7], d1[8], None, out)
    got1 = out.cpu().numpy()                      # (the copy synchronises; the call itself does not)
    assert nlost1 == 0 and got1[4] == n1
    assert np.max(np.abs(got1[:4] - want1)) < TOL, (got1, want1)

    # ---- call 2, straight after: 200 particles of config 1 tracked for two turns, two of them lost on the way
    c = W.config(1, n_particles=200)
    st2 = c["state"].copy()
    st2[6:9] = W.gaussian_bunch(72, 200, 25.0, 0, 0, 0, 0, 0, 0, "sphere")[6:9]
    st2[1, 5] = 1.5                               # |Px| > P: lost in the first element (A15)
    st2[3, 170] = -2.0
    L = gst.Lattice(c["lattice"], c["beam"])
    d2 = torch.tensor(st2, dtype=torch.float64, device="cuda").contiguous()
    b = gst.Bunch(d2)
    b.track(L, 2, c["split"], c["n_slices"], c["depth"])
    want2, nlost2 = b.polarization()
    lost2 = b.lost()
    b.close()
    L.close()
    assert nlost2 == 2 and lost2[5] and lost2[170]
    lost_dev = torch.tensor(lost2, dtype=torch.uint8, device="cuda")
    gst.polarization_noalloc(d2[6], d2[7], d2[8], lost_dev, out)
    got2 = out.cpu().numpy()
    assert got2[4] == 200 - 2
    assert np.max(np.abs(got2[:4] - want2)) < TOL, (got2, want2)
    assert np.max(np.abs(got2[:4] - got1[:4])) > 1e-3          # a different bunch, not the first answer again

    # ---- and once more on the first bunch: the answer of call 1 to the last bit (same numbers, same order)
    gst.polarization_noalloc(d1[6], d1[7], d1[8], None, out)
    assert np.array_equal(out.cpu().numpy(), got1)


def test_no_alloc_polarization_limits_and_errors(gst):
    out = torch.zeros(5, dtype=torch.float64, device="cuda")
    # the maximum itself is accepted ...
    n = gst.NOALLOC_MAX_PARTICLES
    s = torch.zeros((3, n), dtype=torch.float64, device="cuda")
    s[1] = 1.0
    s[1, ::2] = -0.5
    gst.polarization_noalloc(s[0], s[1], s[2], None, out)
    got = out.cpu().numpy()
    assert got[4] == n and abs(got[1] - 0.25) < TOL and abs(got[3] - 0.25) < TOL and got[0] == 0.0 and got[2] == 0.0
    # ... one more is refused before anything is launched or read (the pointers are not even looked at), with a reason
    vp = C.c_void_p
    rc = gst.lib().gst_polarization_noalloc(vp(s.data_ptr()), vp(s.data_ptr()), vp(s.data_ptr()), None, n + 1,
                                            vp(out.data_ptr()), None)
    assert rc == gst.EINVAL and b"GST_NOALLOC_MAX_PARTICLES" in gst.lib().gst_last_error()
    assert np.array_equal(out.cpu().numpy(), got)               # the output was not touched
    # an empty bunch gives zeros; host memory for the output is refused
    gst.polarization_noalloc(s[0, :0], s[1, :0], s[2, :0], None, out)
    assert np.array_equal(out.cpu().numpy(), np.zeros(5))
    host = np.zeros(5)
    rc = gst.lib().gst_polarization_noalloc(vp(s.data_ptr()), vp(s.data_ptr()), vp(s.data_ptr()), None, 10,
                                            vp(host.ctypes.data), None)
    assert rc == gst.EINVAL
