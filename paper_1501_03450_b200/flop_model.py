"""Turn an `ncu --page raw --csv` dump of one track_kernel launch into the flop model bench.py uses.

    ncu -i gpurun_out/prof.ncu-rep --page raw --csv > profiles/rNN_track_raw.csv
    python -m paper_1501_03450_b200.flop_model profiles/rNN_track_raw.csv \
        --key cfg3_rhic_like_bend_kick_n8_d4 --particles 65536 --turns 2

Counts EXECUTED fp64 flops at thread level (predicated-off lanes excluded):
    flop = 2 * dfma + dadd + dmul      (smsp__sass_thread_inst_executed_op_d{fma,add,mul}_pred_on.sum)
as BASELINE.json's north_star asks, divides by particles x turns of the captured launch and stores the
result in paper_1501_03450_b200/flop_model.json.  The per-particle-turn count does not depend on the
number of turns or particles (every particle runs the same element loop), so a short capture serves the
full-size bench launch.
"""
import argparse
import csv
import json
import os

HERE = os.path.dirname(os.path.abspath(__file__))
OUT = os.path.join(HERE, "flop_model.json")

WANT = {
    "dfma": "smsp__sass_thread_inst_executed_op_dfma_pred_on.sum",
    "dadd": "smsp__sass_thread_inst_executed_op_dadd_pred_on.sum",
    "dmul": "smsp__sass_thread_inst_executed_op_dmul_pred_on.sum",
    "dram_read": "dram__bytes_read.sum",
    "dram_write": "dram__bytes_write.sum",
    "duration_ns": "gpu__time_duration.sum",
    "regs": "launch__registers_per_thread",
    "fp64_pipe_pct": "sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active",
    "warps_active_pct": "sm__warps_active.avg.pct_of_peak_sustained_active",
    "inst_executed": "smsp__inst_executed.sum",
    "sm_cycles_active_avg": "sm__cycles_active.avg",
}


def read_raw(path):
    """Accepts both ncu CSV layouts: `--page raw --csv` (wide: one column per metric) and
    `--csv --metrics ...` (long: one row per metric).  Lines before the header (==PROF== ...) are skipped."""
    rows = [r for r in csv.reader(open(path)) if r]
    hdr = next(i for i, r in enumerate(rows) if r[0] == "ID")
    names = rows[hdr]
    out = {}
    if "Metric Name" in names:
        kn, ku, kv = names.index("Metric Name"), names.index("Metric Unit"), names.index("Metric Value")
        first = rows[hdr + 1][0]
        for r in rows[hdr + 1:]:
            if r[0] == first and len(r) > kv:
                out[r[kn]] = (r[kv], r[ku])
    else:
        units, vals = rows[hdr + 1], rows[hdr + 2]
        for n, u, v in zip(names, units, vals):
            out[n] = (v, u)
    return out


def to_float(v, u):
    x = float(v.replace(",", ""))
    scale = {"Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "byte": 1, "inst": 1, "usecond": 1e3, "msecond": 1e6, "nsecond": 1,
             "second": 1e9, "us": 1e3, "ms": 1e6, "ns": 1, "s": 1e9}
    return x * scale.get(u, 1)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("raw_csv")
    ap.add_argument("--key", required=True)
    ap.add_argument("--particles", type=int, required=True)
    ap.add_argument("--turns", type=int, required=True)
    a = ap.parse_args()
    raw = read_raw(a.raw_csv)
    got = {}
    for k, name in WANT.items():
        if name in raw:
            got[k] = to_float(*raw[name])
    flop = 2 * got["dfma"] + got["dadd"] + got["dmul"]
    pt = a.particles * a.turns
    entry = {
        "flop_per_particle_turn": flop / pt,
        "dfma_per_particle_turn": got["dfma"] / pt, "dadd_per_particle_turn": got["dadd"] / pt,
        "dmul_per_particle_turn": got["dmul"] / pt,
        "fp64_inst_per_particle_turn": (got["dfma"] + got["dadd"] + got["dmul"]) / pt,
        "dram_bytes_per_launch": got.get("dram_read", 0) + got.get("dram_write", 0),
        "capture": {"particles": a.particles, "turns": a.turns, "duration_ms": got.get("duration_ns", 0) / 1e6,
                    "registers_per_thread": got.get("regs"), "fp64_pipe_pct_of_peak": got.get("fp64_pipe_pct"),
                    "warps_active_pct": got.get("warps_active_pct")},
        "source": os.path.relpath(a.raw_csv, os.path.dirname(HERE)),
    }
    model = json.load(open(OUT)) if os.path.exists(OUT) else {}
    model[a.key] = entry
    json.dump(model, open(OUT, "w"), indent=1, sort_keys=True)
    print(json.dumps(entry, indent=1))


if __name__ == "__main__":
    main()
