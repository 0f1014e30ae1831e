#!/usr/bin/env python
"""bench.py -- headline benchmark: particle-element-steps/s (fp64 spin+orbit) on the RHIC-like ring.

A "step" is one pass of the whole hot path over one bunch: gst_track for the configuration's full
number of turns (a0-a12, a14) followed by gst_polarization (a13).  Workload at N=1: BASELINE.json
configs[2] (SURVEY "config 3"): 65 536 particles x 1000 turns of the synthetic RHIC-like ring,
bend-kick split, 8 slices, Romberg depth 4 -- the configuration the metric is quoted on.  With N>1
GPUs every rank tracks its own 65 536-particle shard (weak scaling; particles are independent, no
data-path collective; one 5-double all-reduce per polarization report).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--config C] [--split NAME] [--slices N] [--depth D] [--turns T] [--particles P]

Prints ONE JSON line (rank 0).  `--impl reference` times the CPU oracle (test infrastructure, as it
stands) on the host cores on a bounded sample of the same workload.

The roofline fraction needs the number of fp64 flops the kernel EXECUTES per particle-turn, which only ncu can count:
flop_model.json (written by flop_model.py from committed ncu captures under profiles/) holds it per instantiation,
together with the registers and stack frame of the kernel that was captured and the fingerprint of the kernel sources
it was compiled from.  `frac` is printed only when the loaded library's kernel has the same; otherwise it is null and the
line says why (re-capture: see flop_model.py).
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
SPLIT_BY_NAME = {v: k for k, v in W.SPLIT_NAMES.items()}
FLOP_MODEL = os.path.join(ROOT, "flop_model.json")


def load_flop_model():
    """Executed fp64 flops (2*DFMA + DADD + DMUL, thread level) per particle-turn, from the committed ncu
    captures (profiles/, parsed by flop_model.py)."""
    if os.path.exists(FLOP_MODEL):
        return json.load(open(FLOP_MODEL))
    return {}


def model_key(cfg, split, n_slices, depth):
    return "%s_%s_n%d_d%d" % (cfg["name"], W.SPLIT_NAMES[split], n_slices, depth)


def parse_args(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE config (1-based as in SURVEY 8(d))")
    ap.add_argument("--turns", type=int, default=None, help="override turns per step (default: the config's)")
    ap.add_argument("--particles", type=int, default=None)
    ap.add_argument("--split", default=None, choices=sorted(SPLIT_BY_NAME), help="override the config's split")
    ap.add_argument("--slices", type=int, default=None)
    ap.add_argument("--depth", type=int, default=None)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args(argv)


def configure(args):
    cfg = W.config(args.config, n_particles=args.particles, n_turns=args.turns)
    if args.split is not None:
        cfg["split"] = SPLIT_BY_NAME[args.split]
    if args.slices is not None:
        cfg["n_slices"] = args.slices
    if args.depth is not None:
        cfg["depth"] = args.depth
    return cfg


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
        return None
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
    return {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(cfg, n, turns, args.gpus),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}


def workload_config(cfg, n, turns, gpus):
    return {"workload": "BASELINE configs[2] RHIC-like synthetic ring (SURVEY config 3)" if cfg["name"] == "cfg3_rhic_like"
            else cfg["name"],
            "name": cfg["name"], "particles_per_gpu": int(n), "turns_per_step": int(turns), "elements": int(len(cfg["lattice"])),
            "steps_per_particle_turn": int(W.steps_per_turn(cfg["lattice"], cfg["n_slices"])),
            "split": W.SPLIT_NAMES[cfg["split"]], "n_slices": cfg["n_slices"], "romberg_depth": cfg["depth"],
            "parallelism": "particle shards x%d, lattice replicated" % gpus,
            "l2": "state (72 B/particle) is register-resident for the whole step; a 256 MiB buffer is written between "
                  "timed steps to flush L2"}


class CudaMachine:
    """Everything the measured loop needs from the machine: the tracker behind the C ABI, device timers, the L2 flush
    and the collective backend.  (tests/test_distributed_cpu.py runs the same loop, run_ours(), on two gloo ranks with a
    stand-in for this class -- the tracking call is injected there, never here.)"""
    dist_backend = "nccl"

    def __init__(self, local_rank):
        import torch
        if not torch.cuda.is_available():
            raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
        from paper_1501_03450_b200 import gst, gst_diag
        self.torch, self.gst, self.diag, self.local = torch, gst, gst_diag, local_rank
        torch.cuda.set_device(local_rank)
        gst.lib()
        self.device = torch.device("cuda", local_rank)
        self.flush_buf = None

    def open(self, cfg):
        torch = self.torch
        self.lat = self.gst.Lattice(cfg["lattice"], cfg["beam"])
        self.host = torch.tensor(cfg["state"], dtype=torch.float64).pin_memory()
        self.dev = self.host.to("cuda", non_blocking=True).contiguous()
        self.bunch = self.gst.Bunch(self.dev)
        self.flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
        self.stream = torch.cuda.current_stream()
        return self.lat.steps_per_turn(cfg["n_slices"])

    def track(self, turns, split, n_slices, depth):
        self.bunch.track(self.lat, turns, split, n_slices, depth, self.stream)

    def polarization(self):
        return self.bunch.polarization(self.stream)

    def track_host(self, turns, split, n_slices, depth):
        rows = [self.host[i] for i in range(9)]
        return self.lat.track_host(rows, turns, split, n_slices, depth)

    def last_kernel(self):
        return self.bunch.last_kernel()

    def flush(self, k):
        self.flush_buf.fill_(k % 251)

    def sync(self):
        self.torch.cuda.synchronize()

    def mark(self):
        ev = self.torch.cuda.Event(enable_timing=True)
        ev.record(self.stream)
        return ev

    @staticmethod
    def ms_between(a, b):
        return a.elapsed_time(b)

    def clock_sampler(self):
        return ClockSampler(self.local)

    def roofline(self, cfg, n, turns, spt, kernel_ms):
        """FP64 CUDA-core ALU roofline of the tracking kernel."""
        split, n_slices, depth = cfg["split"], cfg["n_slices"], cfg["depth"]
        fm = load_flop_model().get(model_key(cfg, split, n_slices, depth), {})
        peak_meas, _ = self.diag.fp64_peak()
        peak_rrr, _ = self.diag.fp64_peak_rrr()
        kname = self.last_kernel()
        info = dict(self.diag.kernel_info(split, depth, kname), source_hash=self.diag.kernel_source_hash())
        roof = {"bound": "alu", "unit": "TFLOP/s",
                "kernel": "gst::%s<%d,%d,%d>" % (kname, split % 3, depth, 4 if split >= 3 else 2),
                "kernel_ms": kernel_ms, "kernel_info": info, "peak": peak_meas,
                "peak_kind": "measured DFMA chains (gst_diag_fp64_peak), this run", "peak_nominal": NOMINAL_FP64_TFLOPS,
                "peak_three_register_dfma": peak_rrr,   # context: DFMA R,R,R takes 3 cycles on B200
                "traffic": fm.get("dram_bytes_per_launch"),
                "algorithmic_hbm_bytes_per_launch": 144 * n, "hbm_gbs": 144 * n / (kernel_ms * 1e-3) / 1e9}
        flop_pt = fm.get("flop_per_particle_turn")
        cap = fm.get("capture", {})
        why = None
        if not flop_pt:
            why = "no flop model for %s (capture it with ncu and run flop_model.py)" % model_key(cfg, split, n_slices, depth)
        elif cap.get("kernel") != kname or cap.get("kernel_info") != info:
            why = ("the flop model was captured on %s %s, the loaded library has %s %s: re-capture (flop_model.py)"
                   % (cap.get("kernel"), cap.get("kernel_info"), kname, info))
        if why:
            roof.update(achieved=None, frac=None, note=why)
        else:
            ach = flop_pt * n * turns / (kernel_ms * 1e-3) / 1e12
            roof.update(achieved=ach, frac=ach / peak_meas, frac_of_nominal=ach / NOMINAL_FP64_TFLOPS,
                        flop_per_particle_turn=flop_pt, flop_per_step=flop_pt / spt,
                        fp64_inst_per_particle_turn=fm.get("fp64_inst_per_particle_turn"),
                        fp64_pipe_active_pct_in_capture=cap.get("fp64_pipe_pct_of_peak"),
                        flop_source=fm.get("source"))
        return roof

    def close(self):
        self.bunch.close()
        self.lat.close()


def run_ours(args, cfg, machine, config_index):
    """The measured loop: W warm-up steps, K timed steps between barriers, device timers, max over ranks.
    Returns the JSON line (a dict) on rank 0, None elsewhere."""
    import torch
    import torch.distributed as dist
    from paper_1501_03450_b200 import distributed as D

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world > 1 and not dist.is_initialized():
        kw = {"device_id": machine.device} if machine.dist_backend == "nccl" else {}
        dist.init_process_group(machine.dist_backend, **kw)

    if rank > 0 and "opt" in cfg["info"] and config_index >= 3:
        # weak scaling: every rank gets its own bunch of the same size, drawn with its own seed
        n = cfg["state"].shape[1]
        cfg["state"] = W.matched_bunch(1000 + rank, n, cfg["beam"]["gamma0"], cfg["info"]["opt"], 10e-6, 5e-4, 0.1)
    n = cfg["state"].shape[1]
    turns = cfg["n_turns"]
    split, n_slices, depth = cfg["split"], cfg["n_slices"], cfg["depth"]
    spt = machine.open(cfg)
    assert spt == W.steps_per_turn(cfg["lattice"], n_slices)

    def reduce_max(x):
        t = torch.tensor([x], dtype=torch.float64, device=machine.device)
        if world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    def barrier():
        if world > 1:
            dist.barrier()
        machine.sync()

    def report(pol, nlost):
        """bunch-wide polarization: one all-reduce of five doubles"""
        return D.global_polarization(pol, n - nlost, device=machine.device) if world > 1 else (pol, n - nlost)

    for k in range(args.warmup):
        machine.track(turns, split, n_slices, depth)
        report(*machine.polarization())
        machine.flush(k)
    # ---- device-resident timing: K steps, device timers on the launching stream, max over ranks
    sampler = machine.clock_sampler()
    barrier()
    sampler.start()
    marks = []
    t_wall0 = time.perf_counter()
    alive = n
    for k in range(args.steps):
        m0 = machine.mark()
        machine.track(turns, split, n_slices, depth)
        m1 = machine.mark()
        pol, nlost = machine.polarization()
        pol, alive = report(pol, nlost)
        m2 = machine.mark()
        marks.append((m0, m1, m2))
        machine.flush(k)
    barrier()
    wall = time.perf_counter() - t_wall0
    clocks = sampler.stop()
    step_ms = [machine.ms_between(m[0], m[2]) for m in marks]
    track_ms = [machine.ms_between(m[0], m[1]) for m in marks]
    total_ms = reduce_max(sum(step_ms))
    units_per_step = float(n) * turns * spt * world
    value = units_per_step * args.steps / (total_ms * 1e-3)
    lost_total = n * world - int(alive)

    # ---- end to end through the host-buffer C-ABI call: H2D + track + reduce + D2H every step
    e2e = None
    if not args.no_e2e:
        machine.track_host(turns, split, n_slices, depth)          # warm-up
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            machine.track_host(turns, split, n_slices, depth)
        barrier()
        dt = reduce_max(time.perf_counter() - t0)
        e2e = {"value": units_per_step * args.steps / dt, "unit": UNIT,
               "h2d_bytes_per_step": 9 * 8 * n, "d2h_bytes_per_step": 9 * 8 * n + 4 * 8 + 8,
               "api": "gst_track_host (pinned host buffers; H2D, gst_track, gst_polarization, D2H inside the timed region)"}

    out = None
    if rank == 0:
        out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
               "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
               "dtype": "f64", "data": "synthetic", "config": workload_config(cfg, n, turns, world),
               "particle_turns_per_s": float(n) * turns * world * args.steps / (total_ms * 1e-3),
               "polarization": [float(x) for x in pol], "lost": lost_total, "wall_s": wall, "clocks": clocks, "e2e": e2e,
               "gpu_launches": args.steps * 3,
               "launches_per_step": "%s + moments_kernel + finalize_kernel" % machine.last_kernel(),
               "roofline": machine.roofline(cfg, n, turns, spt, float(np.mean(track_ms)))}
        if not args.no_cpu_baseline:
            out["cpu_baseline"] = cpu_baseline(cfg)
    machine.close()
    return out


def main(argv=None):
    args = parse_args(argv)
    cfg = configure(args)
    if args.impl == "reference":
        line = run_reference(args, cfg)
        if line is not None:
            print(json.dumps(line))
        return 0
    import torch.distributed as dist
    line = run_ours(args, cfg, CudaMachine(int(os.environ.get("LOCAL_RANK", "0"))), args.config)
    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()
    if line is None:
        return 0
    print(json.dumps(line))
    if line["lost"] != 0:         # the BASELINE bunches lose nobody: a loss means the run is not the workload
        sys.stderr.write("bench.py: %d particles were lost\n" % line["lost"])
        return 1
    return 0


if __name__ == "__main__":
    sys.exit(main())
