"""The two BASELINE studies that are more than one timed launch, and the paper's single-element study, run through the
C ABI on one GPU.

    python -m paper_1501_03450_b200.studies ramp  [--particles N] [--turns T] [--chunk 100] [--out FILE.md]
    python -m paper_1501_03450_b200.studies sweep [--particles N] [--turns T] [--out FILE.md]
    python -m paper_1501_03450_b200.studies fig7  [--out FILE.md]

ramp  : BASELINE configs[3] (SURVEY config 4): the RHIC-like ring with its cavity ramping the energy by
        100 keV/turn from G*gamma = 45.0, 2^20 particles, 5000 turns; the bunch polarization, emittances
        and lost count are reported every `chunk` turns (gst_track in chunks + gst_polarization, the
        checkpoint pattern of P:776).
sweep : BASELINE configs[4] (SURVEY config 5): accuracy vs throughput on the ring without snakes,
        262 144 particles, 100 turns, for the three splits x the 27 valid (slices, depth) pairs (reading A4).
        Errors are the paper's (44) P:622 and (46) P:733 against a reference by refinement, as the paper
        does: matrix-kick, 128 slices, depth 6 -- computed by the same library; that this
        reference equals the CPU oracle's is what tests/test_gpu_parity.py::test_config5_reference_run checks.

fig7  : the paper's single-element study (Fig. 7): spin error of its test particle (footnote 5)
        across the RHIC IR quadrupole (1.83 m, 70 T/m), arc dipole (9.45 m, 2.225 deg) and the 1.3 T,
        2.1 m solenoid at 200 GeV and at 1.2 GeV, against the number of slices, for mid-slice PWC
        and for k = 0..3 Romberg iterations on the edge scheme; reference = 256 slices, k = 3.

Every number of the hot path comes from the CUDA kernels; torch is used for device memory, the error
norms of the report and nothing else.  One JSON line per report row on stdout; --out adds a markdown table.
"""
import argparse
import json
import sys
import time

import numpy as np

from . import workloads as W

G_PROTON = 1.792847


def _device_state(torch, state):
    return torch.tensor(state, dtype=torch.float64, device="cuda").contiguous()


def _timed_track(torch, bunch, lat, turns, split, n_slices, depth):
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    bunch.track(lat, turns, split, n_slices, depth)
    e1.record()
    e1.synchronize()
    return e0.elapsed_time(e1)


def ramp(args):
    import torch
    from . import gst
    cfg = W.config(4, n_particles=args.particles, n_turns=args.turns)
    n, turns = cfg["state"].shape[1], cfg["n_turns"]
    lat = gst.Lattice(cfg["lattice"], cfg["beam"])
    spt = lat.steps_per_turn(cfg["n_slices"])
    dev = _device_state(torch, cfg["state"])
    bunch = gst.Bunch(dev)
    rows, ms_total, done = [], 0.0, 0
    pol, lost = bunch.polarization()
    ex, ey = bunch.emittance()
    g0 = cfg["beam"]["gamma0"]
    bg0 = float(np.sqrt(g0 * g0 - 1.0))
    rows.append(dict(turn=0, G_gamma=G_PROTON * g0, P=[float(x) for x in pol], eps_n=[ex * bg0, ey * bg0], lost=int(lost)))
    print(json.dumps(rows[-1]))
    while done < turns:
        nt = min(args.chunk, turns - done)
        ms_total += _timed_track(torch, bunch, lat, nt, cfg["split"], cfg["n_slices"], cfg["depth"])
        done += nt
        pol, lost = bunch.polarization()
        ex, ey = bunch.emittance()
        g, turn = bunch.reference()
        bg = float(np.sqrt(g * g - 1.0))
        # normalised rms emittance beta*gamma*eps: constant under adiabatic damping (A13)
        rows.append(dict(turn=int(turn), G_gamma=G_PROTON * g, P=[float(x) for x in pol], eps_n=[ex * bg, ey * bg],
                         lost=int(lost)))
        print(json.dumps(rows[-1]))
        sys.stdout.flush()
    rate = float(n) * turns * spt / (ms_total * 1e-3)
    summary = dict(study="ramp", particles=n, turns=turns, chunk=args.chunk, steps_per_turn=spt,
                   track_ms=ms_total, steps_per_s=rate, split=W.SPLIT_NAMES[cfg["split"]],
                   n_slices=cfg["n_slices"], depth=cfg["depth"])
    print(json.dumps(summary))
    if args.out:
        with open(args.out, "w") as f:
            f.write("# Ramp through G*gamma = 45.0 -> %.3f (config 4), %d particles, %d turns\n\n" % (rows[-1]["G_gamma"], n, turns))
            f.write("Command: `python -m paper_1501_03450_b200.studies ramp --particles %d --turns %d --chunk %d`\n\n" % (n, turns, args.chunk))
            f.write("track kernel time %.1f s, %.4g particle-element-steps/s\n\n" % (ms_total * 1e-3, rate))
            f.write("| turn | G*gamma | Px | Py | Ps | |P| | eps_n,x [m] | eps_n,y [m] | lost |\n|---|---|---|---|---|---|---|---|---|\n")
            for r in rows:
                f.write("| %d | %.5f | %+.6f | %+.6f | %+.6f | %.6f | %.4e | %.4e | %d |\n"
                        % (r["turn"], r["G_gamma"], r["P"][0], r["P"][1], r["P"][2], r["P"][3], r["eps_n"][0], r["eps_n"][1], r["lost"]))
    bunch.close()
    lat.close()


def sweep(args):
    import torch
    from . import gst
    cfg = W.config(5, n_particles=args.particles, n_turns=args.turns)
    n, turns = cfg["state"].shape[1], cfg["n_turns"]
    lat = gst.Lattice(cfg["lattice"], cfg["beam"])
    init = _device_state(torch, cfg["state"])

    def run(split, n_slices, depth):
        dev = init.clone()
        b = gst.Bunch(dev)
        ms = _timed_track(torch, b, lat, turns, split, n_slices, depth)
        _, lost = b.polarization()
        b.close()
        return dev, ms, int(lost)

    ref_split = W.SPLIT_MATRIX_KICK_4 if args.order4 else W.SPLIT_MATRIX_KICK
    ref, ref_ms, ref_lost = run(ref_split, args.ref_slices, 6)
    print(json.dumps(dict(study="sweep", reference=dict(split=W.SPLIT_NAMES[ref_split], n_slices=args.ref_slices, depth=6, ms=ref_ms,
                                                        lost=ref_lost), particles=n, turns=turns)))
    rows = []
    splits = [W.SPLIT_DRIFT_KICK, W.SPLIT_BEND_KICK, W.SPLIT_MATRIX_KICK]
    if args.order4:
        splits += [W.SPLIT_DRIFT_KICK_4, W.SPLIT_BEND_KICK_4, W.SPLIT_MATRIX_KICK_4]
    for split in splits:
        for n_slices, depth in W.sweep_pairs():
            if n_slices > args.max_slices:
                continue
            dev, ms, lost = run(split, n_slices, depth)
            dS = torch.linalg.vector_norm(dev[6:9] - ref[6:9], dim=0).mean().item()          # (46) P:733
            dX = torch.sqrt(torch.mean((dev[0] - ref[0]) ** 2)).item()                          # (44) P:622
            spt = lat.steps_per_turn(n_slices)
            row = dict(split=W.SPLIT_NAMES[split], n_slices=n_slices, depth=depth, spin_err=dS, x_rms_err=dX,
                       ms=ms, steps_per_s=float(n) * turns * spt / (ms * 1e-3),
                       particle_turns_per_s=float(n) * turns / (ms * 1e-3), lost=lost)
            rows.append(row)
            print(json.dumps(row))
            sys.stdout.flush()
            del dev
    if args.out:
        with open(args.out, "w") as f:
            f.write("# Accuracy vs throughput (config 5): RHIC-like ring without snakes, %d particles, %d turns\n\n" % (n, turns))
            f.write("Command: `python -m paper_1501_03450_b200.studies sweep --particles %d --turns %d%s`\n\n"
                    % (n, turns, " --order4" if args.order4 else ""))
            f.write("Reference: %s, %d slices, depth 6 (%.1f s).  spin error = (46) P:733, X error = (44) P:622.\n\n"
                    % (W.SPLIT_NAMES[ref_split], args.ref_slices, ref_ms * 1e-3))
            f.write("| split | slices | depth | spin error | rms X error [m] | steps/s | particle-turns/s |\n|---|---|---|---|---|---|---|\n")
            for r in rows:
                f.write("| %s | %d | %d | %.3e | %.3e | %.4g | %.4g |\n" % (r["split"], r["n_slices"], r["depth"], r["spin_err"],
                                                                       r["x_rms_err"], r["steps_per_s"], r["particle_turns_per_s"]))
    lat.close()


def fig7(args):
    """Inputs are the ones the paper prints (cited above); the element maps are matrix-kick / exact."""
    import math
    import torch
    from . import gst
    mp_gev = W.MASS_PROTON_EV / 1e9

    def brho(gamma):
        return W.MASS_PROTON_EV * gamma * W.beta_of_gamma(gamma) / 299792458.0

    g200 = 200.0 / mp_gev                                    # "200 GeV protons": total energy (DESIGN R3)
    g12 = 1.0 + 1.2 / mp_gev                                 # "1.2 GeV proton": kinetic energy (DESIGN R9)
    cases = [("IR quadrupole 1.83 m, 70 T/m, 200 GeV", W.quad(1.83, 70.0 / brho(g200)), g200),
             ("arc dipole 9.45 m, 2.225 deg, 200 GeV", W.sbend(9.45, math.radians(2.225)), g200),
             ("solenoid 2.1 m, 1.3 T, 200 GeV", W.solenoid(2.1, 1.3 / brho(g200)), g200),
             ("solenoid 2.1 m, 1.3 T, 1.2 GeV", W.solenoid(2.1, 1.3 / brho(g12)), g12)]
    slices = [1, 2, 4, 8, 16, 32, 64, 128]
    lines = []
    for name, elem, gamma in cases:
        b0 = W.beta_of_gamma(gamma)
        delta = 1e-3
        pt = math.sqrt(1.0 / b0 ** 2 + 2 * delta + delta ** 2) - 1.0 / b0     # A22
        s0 = np.array([2.0, 10.0, 1.0]) / math.sqrt(105.0)                    # (0.1952, 0.9759, 0.0976)
        st = np.zeros((9, 32))
        st[:, :] = np.array([1.0e-3, 0.1e-3, 0.0, -0.2e-3, 0.0, pt, s0[0], s0[1], s0[2]])[:, None]
        lat = gst.Lattice(W.lattice([elem]), W.beam(gamma))

        def spin(n, depth):
            dev = _device_state(torch, st)
            b = gst.Bunch(dev)
            if depth >= 1:
                b.track(lat, 1, W.SPLIT_MATRIX_KICK, n, depth)
            else:
                b.track_pwc(lat, 1, W.SPLIT_MATRIX_KICK, n, W.PWC_HALF_SLICE)
            out = dev[6:9, 0].cpu().numpy()
            b.close()
            return out
        ref = spin(256, 4)
        rows = []
        for n in slices:
            errs = {"pwc": float(np.linalg.norm(spin(n, 0) - ref))}
            for d in (1, 2, 3, 4):
                errs["k%d" % (d - 1)] = float(np.linalg.norm(spin(n, d) - ref)) if n % (1 << (d - 1)) == 0 else None
            rows.append((n, errs))
            print(json.dumps(dict(element=name, slices=n, **errs)))
        lines.append((name, rows))
        lat.close()
    if args.out:
        with open(args.out, "w") as f:
            f.write("# Single-element spin errors against the number of slices (the paper's Fig. 7, P:648-660), computed on the GPU\n\n")
            f.write("Command: `python -m paper_1501_03450_b200.studies fig7`\n\n")
            f.write("|S - S_ref| for the test particle of footnote 5; S_ref = 256 slices, three Romberg iterations (P:652).  PWC = mid-slice\n"
                    "piece-wise constant (37); k = Romberg iterations on the slice-edge products (38)(39), k = 0 is the trapezoid product.\n\n")
            for name, rows in lines:
                f.write("## %s\n\n| slices | PWC | k = 0 | k = 1 | k = 2 | k = 3 |\n|---|---|---|---|---|---|\n" % name)
                for n, e in rows:
                    f.write("| %d | %s |\n" % (n, " | ".join("%.2e" % e[k] if e[k] is not None else "" for k in ("pwc", "k0", "k1", "k2", "k3"))))
                f.write("\n")


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    sub = ap.add_subparsers(dest="study", required=True)
    r = sub.add_parser("ramp")
    r.add_argument("--particles", type=int, default=None)
    r.add_argument("--turns", type=int, default=None)
    r.add_argument("--chunk", type=int, default=100)
    r.add_argument("--out", default=None)
    s = sub.add_parser("sweep")
    s.add_argument("--particles", type=int, default=None)
    s.add_argument("--turns", type=int, default=None)
    s.add_argument("--ref-slices", type=int, default=128)
    s.add_argument("--max-slices", type=int, default=64)
    s.add_argument("--order4", action="store_true",
                   help="add the fourth-order compositions (SURVEY 8(f) f1); the reference becomes matrix_kick_4")
    s.add_argument("--out", default=None)
    g = sub.add_parser("fig7")
    g.add_argument("--out", default=None)
    args = ap.parse_args(argv)
    t0 = time.time()
    {"ramp": ramp, "sweep": sweep, "fig7": fig7}[args.study](args)
    print(json.dumps(dict(wall_s=time.time() - t0)))


if __name__ == "__main__":
    main()
