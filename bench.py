#!/usr/bin/env python
"""bench.py -- headline benchmark: particle-element-steps/s (fp64 spin+orbit) on the RHIC-like ring.

A "step" is one pass of the whole hot path over one bunch: gst_track for the configuration's full
number of turns (a0-a12, a14) followed by gst_polarization (a13).  Workload at N=1: BASELINE.json
configs[2] (SURVEY "config 3"): 65 536 particles x 1000 turns of the synthetic RHIC-like ring,
bend-kick split, 8 slices, Romberg depth 4 -- the configuration the metric is quoted on.  With N>1
GPUs every rank tracks its own 65 536-particle shard (weak scaling; particles are independent, no
data-path collective; one 5-double all-reduce per polarization report).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

Prints ONE JSON line (rank 0).  `--impl reference` times the CPU oracle (test infrastructure, as it
stands) on the host cores on a bounded sample of the same workload.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_1501_03450_b200 import workloads as W  # noqa: E402

METRIC = "particle-element-steps/sec (fp64 spin+orbit) on 1 B200; % of FP64 peak"
UNIT = "particle-element-steps/s"
NOMINAL_FP64_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12     # SMs x FP64 FMA lanes x 2 flop x max SM clock = 37.2


def load_flop_model():
    """Executed fp64 flops (2*DFMA + DADD + DMUL, thread level) per particle-turn, from the committed ncu
    capture (profiles/, written by paper_1501_03450_b200/flop_model.py)."""
    p = os.path.join(ROOT, "paper_1501_03450_b200", "flop_model.json")
    if os.path.exists(p):
        return json.load(open(p))
    return {}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE config (1-based as in SURVEY 8(d))")
    ap.add_argument("--turns", type=int, default=None, help="override turns per step (default: the config's)")
    ap.add_argument("--particles", type=int, default=None)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[1])); mx.append(float(r[2])); pw.append(float(r[3]))
                for k, nm in enumerate(names):
                    if r[5 + k].lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def cpu_baseline(cfg, budget_s=15.0):
    """The oracle as it stands (fp64 instantiation, literal formulas), all host cores, bounded sample."""
    from oracle import oracle as O
    cores = O.default_threads()
    lat, beam = cfg["lattice"], cfg["beam"]
    spt = W.steps_per_turn(lat, cfg["n_slices"])
    n = min(cfg["state"].shape[1], cores * 16)
    st = cfg["state"][:, :n]
    O.track(lat, beam, st, 1, cfg["split"], cfg["n_slices"], cfg["depth"], prec=O.PREC_DOUBLE, threads=cores)   # warm: library load, threads
    t0 = time.perf_counter()
    O.track(lat, beam, st, 8, cfg["split"], cfg["n_slices"], cfg["depth"], prec=O.PREC_DOUBLE, threads=cores)
    t1 = (time.perf_counter() - t0) / 8
    turns = int(max(2, min(20000, budget_s / max(t1, 1e-4))))
    t0 = time.perf_counter()
    O.track(lat, beam, st, turns, cfg["split"], cfg["n_slices"], cfg["depth"], prec=O.PREC_DOUBLE, threads=cores)
    dt = time.perf_counter() - t0
    return {"value": n * turns * spt / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "%d particles x %d turns of %s (%d steps/turn), oracle in double, %d threads, %.1f s"
                      % (n, turns, cfg["name"], spt, cores, dt),
            "particle_turns_per_s": n * turns / dt}


def run_reference(args, cfg):
    """--impl reference: the oracle on the host cores; a step = a bounded sample of the workload."""
    from oracle import oracle as O
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cores = O.default_threads()
    lat, beam = cfg["lattice"], cfg["beam"]
    spt = W.steps_per_turn(lat, cfg["n_slices"])
    n = min(cfg["state"].shape[1], cores * 16)
    turns = 4
    st = cfg["state"][:, :n]
    for _ in range(args.warmup):
        O.track(lat, beam, st, 1, cfg["split"], cfg["n_slices"], cfg["depth"], prec=O.PREC_DOUBLE, threads=cores)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        O.track(lat, beam, st, turns, cfg["split"], cfg["n_slices"], cfg["depth"], prec=O.PREC_DOUBLE, threads=cores)
    dt = time.perf_counter() - t0
    value = args.steps * n * turns * spt / dt
    sample = "each step = %d particles x %d turns of %s, oracle in double on %d threads" % (n, turns, cfg["name"], cores)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(cfg, n, turns, args.gpus),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def workload_config(cfg, n, turns, gpus):
    return {"workload": "BASELINE configs[2] RHIC-like synthetic ring (SURVEY config 3)" if cfg["name"] == "cfg3_rhic_like"
            else cfg["name"],
            "particles_per_gpu": int(n), "turns_per_step": int(turns), "elements": int(len(cfg["lattice"])),
            "steps_per_particle_turn": int(W.steps_per_turn(cfg["lattice"], cfg["n_slices"])),
            "split": W.SPLIT_NAMES[cfg["split"]], "n_slices": cfg["n_slices"], "romberg_depth": cfg["depth"],
            "parallelism": "particle shards x%d, lattice replicated" % gpus,
            "l2": "state (72 B/particle) is register-resident for the whole step; a 256 MiB buffer is written between "
                  "timed steps to flush L2"}


def main():
    args = parse_args()
    cfg = W.config(args.config, n_particles=args.particles, n_turns=args.turns)
    if args.impl == "reference":
        run_reference(args, cfg)
        return

    import torch
    import torch.distributed as dist
    from paper_1501_03450_b200 import distributed as D
    from paper_1501_03450_b200 import gst
    from paper_1501_03450_b200 import gst_diag

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    gst.lib()

    if rank > 0:      # weak scaling: every rank gets its own bunch of the same size, drawn with its own seed
        n = cfg["state"].shape[1]
        cfg["state"] = W.matched_bunch(1000 + rank, n, cfg["beam"]["gamma0"], cfg["info"]["opt"], 10e-6, 5e-4, 0.1) \
            if "opt" in cfg["info"] and args.config >= 3 else cfg["state"]
    n = cfg["state"].shape[1]
    turns = cfg["n_turns"]
    split, n_slices, depth = cfg["split"], cfg["n_slices"], cfg["depth"]
    lat = gst.Lattice(cfg["lattice"], cfg["beam"])
    spt = lat.steps_per_turn(n_slices)
    assert spt == W.steps_per_turn(cfg["lattice"], n_slices)
    host = torch.tensor(cfg["state"], dtype=torch.float64).pin_memory()
    dev = host.to("cuda", non_blocking=True).contiguous()
    bunch = gst.Bunch(dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step():
        bunch.track(lat, turns, split, n_slices, depth, stream)
        pol, nlost = bunch.polarization(stream)
        return D.global_polarization(pol, n - nlost, device="cuda") if world > 1 else (pol, n - nlost)

    for _ in range(args.warmup):
        step()
        flush.fill_(1)
    # ---- device-resident timing: K steps, CUDA events on the launching stream, max over ranks
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
          for _ in range(args.steps)]
    t_wall0 = time.perf_counter()
    for k in range(args.steps):
        ev[k][0].record(stream)
        bunch.track(lat, turns, split, n_slices, depth, stream)
        ev[k][1].record(stream)
        pol, nlost = bunch.polarization(stream)
        if world > 1:
            pol, _ = D.global_polarization(pol, n - nlost, device="cuda")
        ev[k][2].record(stream)
        flush.fill_(k)
    barrier()
    wall = time.perf_counter() - t_wall0
    clocks = sampler.stop()
    step_ms = [e[0].elapsed_time(e[2]) for e in ev]
    track_ms = [e[0].elapsed_time(e[1]) for e in ev]
    total_ms = torch.tensor([sum(step_ms)], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(total_ms, op=dist.ReduceOp.MAX)
    total_ms = float(total_ms.item())
    units_per_step = float(n) * turns * spt * world
    value = units_per_step * args.steps / (total_ms * 1e-3)

    # ---- end to end through the host-buffer C-ABI call: H2D + track + reduce + D2H every step
    e2e = None
    if not args.no_e2e:
        hrows = [host[i] for i in range(9)]
        lat.track_host(hrows, turns, split, n_slices, depth)          # warm-up
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            hrows = [host[i] for i in range(9)]
            lat.track_host(hrows, turns, split, n_slices, depth)
        barrier()
        dt = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(dt, op=dist.ReduceOp.MAX)
        e2e = {"value": units_per_step * args.steps / float(dt.item()), "unit": UNIT,
               "h2d_bytes_per_step": 9 * 8 * n, "d2h_bytes_per_step": 9 * 8 * n + 4 * 8 + 8,
               "api": "gst_track_host (pinned host buffers; H2D, gst_track, gst_polarization, D2H inside the timed region)"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (track_kernel): FP64 CUDA-core ALU bound
    fm = load_flop_model()
    key = "%s_%s_n%d_d%d" % (cfg["name"], W.SPLIT_NAMES[split], n_slices, depth)
    flop_pt = fm.get(key, {}).get("flop_per_particle_turn")
    peak_meas, peak_ms = gst_diag.fp64_peak()
    peak_rrr, _ = gst_diag.fp64_peak_rrr()
    k_ms = float(np.mean(track_ms))
    roof = {"bound": "alu", "unit": "TFLOP/s", "kernel": "gst::%s<%d,%d,2>" % (bunch.last_kernel(), split, depth),
            "kernel_ms": k_ms, "peak": peak_meas, "peak_kind": "measured DFMA chains (gst_diag_fp64_peak), this run",
            "peak_nominal": NOMINAL_FP64_TFLOPS,
            "peak_three_register_dfma": peak_rrr,   # context: DFMA R,R,R takes 3 cycles on B200
            "traffic": fm.get(key, {}).get("dram_bytes_per_launch"),
            "algorithmic_hbm_bytes_per_launch": 144 * n, "hbm_gbs": 144 * n / (k_ms * 1e-3) / 1e9}
    if flop_pt:
        ach = flop_pt * n * turns / (k_ms * 1e-3) / 1e12
        roof.update(achieved=ach, frac=ach / peak_meas, frac_of_nominal=ach / NOMINAL_FP64_TFLOPS,
                    flop_per_particle_turn=flop_pt, flop_per_step=flop_pt / spt,
                    flop_source=fm[key].get("source"))
    else:
        roof.update(achieved=None, frac=None, note="no flop model for this configuration (run flop_model.py on an ncu capture)")

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic", "config": workload_config(cfg, n, turns, world),
           "particle_turns_per_s": float(n) * turns * world * args.steps / (total_ms * 1e-3),
           "polarization": [float(x) for x in pol], "wall_s": wall, "clocks": clocks, "e2e": e2e,
           "gpu_launches": args.steps * 3,
           "launches_per_step": "%s + moments_kernel + finalize_kernel" % bunch.last_kernel(),
           "roofline": roof}
    if not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(cfg)
    print(json.dumps(out))
    bunch.close()
    lat.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
