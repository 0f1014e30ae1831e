"""Error metrics shared by the GPU parity tests (no arithmetic of the method here).

Two metrics per orbit coordinate c ("Tolerance"):
  bunch-scale    max_j |gpu - oracle| / max_j |oracle_c|                    (SURVEY 8(c) "parity metric")
  per-particle   max_j |gpu_j - oracle_j| / max(|oracle_cj|, rms_j oracle_c)
The second is the north star's "per-particle ... relative" with an absolute floor: the rounding error of a map does not
shrink with a particle's own amplitude (the intermediate quantities 1 + hX, Ps, ... are O(1)), so below the bunch's rms
size of a coordinate the error is measured against that rms.  Spin components are compared absolutely (|S| = 1).
The oracle side is always its long-double instantiation (reading R1).
"""
import numpy as np


def orbit_err(got, ref):
    return max(np.max(np.abs(got[c] - ref[c])) / max(np.max(np.abs(ref[c])), 1e-300) for c in range(6))


def orbit_err_per_particle(got, ref):
    worst = 0.0
    for c in range(6):
        floor = max(float(np.sqrt(np.mean(ref[c] ** 2))), 1e-300)
        worst = max(worst, float(np.max(np.abs(got[c] - ref[c]) / np.maximum(np.abs(ref[c]), floor))))
    return worst


def spin_err(got, ref):
    return float(np.max(np.abs(got[6:9] - ref[6:9])))
