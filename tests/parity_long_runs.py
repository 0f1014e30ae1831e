"""Long parity runs that are too slow for the test suite (minutes of oracle time): the BASELINE configurations at
their full turn counts on reduced bunches, CUDA path against the oracle (long double), one markdown table.

    python tests/parity_long_runs.py --out profiles/rNN_parity_long.md        (on the GPU box)

Not collected by pytest (the name does not start with test_).  BASELINE's criteria: per-particle 1e-9 after 100 turns
for non-resonant configs; bunch polarization within 1e-6 for the near-resonance and ramp configs (3, 4, 5).
"""
import argparse
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=None)
    ap.add_argument("--particles", type=int, default=512)
    args = ap.parse_args()
    import torch
    from oracle import oracle as O
    from paper_1501_03450_b200 import gst
    from paper_1501_03450_b200 import workloads as W
    rows = []
    for cfg_i, turns in ((2, 1000), (3, 1000), (4, 5000), (5, 100)):
        c = W.config(cfg_i, n_particles=args.particles)
        st = c["state"]
        t0 = time.time()
        ref, rlost, g_ref = O.track(c["lattice"], c["beam"], st, turns, c["split"], c["n_slices"], c["depth"])
        t_or = time.time() - t0
        L = gst.Lattice(c["lattice"], c["beam"])
        d = torch.tensor(st, dtype=torch.float64, device="cuda").contiguous()
        b = gst.Bunch(d)
        done = 0
        while done < turns:                                   # chunks of 100 turns, as config 4 is meant to be run
            b.track(L, min(100, turns - done), c["split"], c["n_slices"], c["depth"])
            done += 100
        pol, nlost = b.polarization()
        got = d.cpu().numpy()
        g_gpu, _ = b.reference()
        b.close()
        L.close()
        orb = max(np.max(np.abs(got[k] - ref[k])) / max(np.max(np.abs(ref[k])), 1e-300) for k in range(6))
        spn = float(np.max(np.abs(got[6:9] - ref[6:9])))
        rp, _ = O.polarization(ref)
        rows.append((c["name"], args.particles, turns, W.SPLIT_NAMES[c["split"]], c["n_slices"], c["depth"], orb, spn,
                     float(np.max(np.abs(pol - rp))), float(pol[3]), int(nlost), int(rlost.sum()), abs(g_gpu - g_ref) / g_ref, t_or))
        print(rows[-1])
    if args.out:
        with open(args.out, "w") as f:
            f.write("# CUDA path against the oracle (long double) at the full turn counts, reduced bunches\n\n")
            f.write("Command: `python tests/parity_long_runs.py --particles %d --out %s`\n\n" % (args.particles, args.out))
            f.write("orbit: max over coordinates of max_j |gpu - oracle| / max_j |oracle|; spin: max absolute component difference;\n"
                    "dP: max difference of the bunch polarization components and modulus.\n\n")
            f.write("| config | particles | turns | split | slices | depth | orbit | spin | dP | |P| | lost gpu / oracle | d gamma0 | oracle s |\n")
            f.write("|---|---|---|---|---|---|---|---|---|---|---|---|---|\n")
            for r in rows:
                f.write("| %s | %d | %d | %s | %d | %d | %.2e | %.2e | %.2e | %.6f | %d / %d | %.1e | %.0f |\n" % r)


if __name__ == "__main__":
    main()
