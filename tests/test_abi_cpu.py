"""CPU-side checks of the boundary: the C-ABI library loads and exports every symbol include/gst.h and
include/gst_diag.h declare, and nothing else; the element struct layout matches; compute calls fail loudly
without a GPU."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_1501_03450_b200 import build as B
from paper_1501_03450_b200 import gst
from paper_1501_03450_b200 import gst_diag
from paper_1501_03450_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_builds_loads_and_exports_every_declared_symbol():
    B.build()
    L = gst.lib()
    declared = {}
    for header, exports in (("gst.h", gst.EXPORTS), ("gst_diag.h", gst_diag.EXPORTS)):
        hdr = open(os.path.join(ROOT, "include", header)).read()
        hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)            # prototypes only, not the prose
        declared[header] = set(re.findall(r"\b(gst_[a-z0-9_]+)\s*\(", hdr))
        assert declared[header] == set(exports), declared[header] ^ set(exports)
        for name in declared[header]:
            assert hasattr(L, name)
    # the product header holds the tracking ABI only: diagnostics and test hooks live behind gst_diag.h
    assert not any(n.startswith("gst_diag_") for n in declared["gst.h"])
    assert all(n.startswith("gst_diag_") for n in declared["gst_diag.h"])
    # ... and the library's dynamic symbol table exports exactly the two headers' functions
    import subprocess
    out = subprocess.run(["nm", "-D", "--defined-only", gst.LIB_PATH], capture_output=True, text=True).stdout
    exported = {l.split()[-1] for l in out.splitlines() if " T " in l and l.split()[-1].startswith("gst_")}
    assert exported == declared["gst.h"] | declared["gst_diag.h"], exported ^ (declared["gst.h"] | declared["gst_diag.h"])


def test_struct_layouts_match_the_header():
    assert C.sizeof(gst.gst_element) == 144 and C.sizeof(gst.gst_beam) == 24
    assert gst.gst_element.L.offset == 8 and gst.gst_element.kn.offset == 32 and gst.gst_element.snake_phi.offset == 136
    assert W.ELEM_DTYPE.itemsize == 144          # the neutral workload record has the same fields


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    c = W.config(1)
    with pytest.raises(gst.GstError) as ei:
        gst.Lattice(c["lattice"], c["beam"])
    assert ei.value.status == gst.ECUDA


def test_workload_recipes():
    c1, c2 = W.config(1), W.config(2, n_particles=16)
    assert len(c1["lattice"]) == 112 and W.steps_per_turn(c1["lattice"], 4) == 304
    assert len(c2["lattice"]) == 577 and W.steps_per_turn(c2["lattice"], 8) == 2369
    c3 = W.config(3, n_particles=16)
    lat = c3["lattice"]
    assert W.steps_per_turn(lat, 8) == 4311 and abs(float(np.sum(lat["L"])) - 3833.8) < 0.01
    assert int(np.sum(np.isin(lat["type"], (W.SBEND, W.QUAD, W.DRIFT)))) == 1488
    opt = c3["info"]["opt"]
    assert abs(opt["Qx"] - 33.57) < 1e-6 and abs(opt["Qy"] - 33.43) < 1e-6 and opt["gamma_t"] < c3["beam"]["gamma0"]
    assert abs(c3["beam"]["G"] * c3["beam"]["gamma0"] - 45.5) < 1e-12
    assert len(W.sweep_pairs()) == 27
    assert np.array_equal(W.config(3, n_particles=16)["state"], c3["state"])       # seeded, reproducible
