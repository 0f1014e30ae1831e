"""Turn ncu counter captures of the tracking kernel into flop_model.json, the flop counts bench.py's roofline uses.

One capture = two files made by the SAME bench.py command on the GPU box, first plain, then under ncu:

    python bench.py ARGS --steps 1 --warmup 0 --turns 16 --no-e2e --no-cpu-baseline > gpurun_out/fm_TAG.json &&
    ncu --clock-control none -k regex:track_ -c 1 --csv --metrics METRICS --log-file gpurun_out/fm_TAG.csv \
        python bench.py ARGS --steps 1 --warmup 0 --turns 16 --no-e2e --no-cpu-baseline

(METRICS below.)  Then, here:   python flop_model.py [--source-hash H] profiles/r02_fm_TAG.csv [more .csv ...]
Each .csv needs its .json beside it: the JSON line names the workload, the kernel that ran and its registers and
stack frame (gst_diag_kernel_info), which bench.py later compares with the loaded library before it prints a fraction.

Counts EXECUTED fp64 flops at thread level (predicated-off lanes excluded):
    flop = 2 * dfma + dadd + dmul      (smsp__sass_thread_inst_executed_op_d{fma,add,mul}_pred_on.sum)
as BASELINE.json's north_star asks, divided by particles x turns of the captured launch.  The per-particle-turn count
does not depend on the number of turns or particles (every particle runs the same element loop), so a short capture
serves the full-size bench launch.
"""
import csv
import json
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
OUT = os.path.join(HERE, "flop_model.json")

METRICS = ("smsp__sass_thread_inst_executed_op_dfma_pred_on.sum,smsp__sass_thread_inst_executed_op_dadd_pred_on.sum,"
           "smsp__sass_thread_inst_executed_op_dmul_pred_on.sum,smsp__inst_executed.sum,sm__inst_executed_pipe_fp64.sum,"
           "sm__inst_executed_pipe_xu.sum,gpu__time_duration.sum,dram__bytes_read.sum,dram__bytes_write.sum,"
           "launch__registers_per_thread,sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active,"
           "sm__warps_active.avg.pct_of_peak_sustained_active,smsp__inst_executed_op_branch.sum,"
           "smsp__issue_active.avg.pct_of_peak_sustained_active,sass__inst_executed_register_spilling")

WANT = {
    "dfma": "smsp__sass_thread_inst_executed_op_dfma_pred_on.sum",
    "dadd": "smsp__sass_thread_inst_executed_op_dadd_pred_on.sum",
    "dmul": "smsp__sass_thread_inst_executed_op_dmul_pred_on.sum",
    "dram_read": "dram__bytes_read.sum",
    "dram_write": "dram__bytes_write.sum",
    "duration_ns": "gpu__time_duration.sum",
    "regs": "launch__registers_per_thread",
    "fp64_pipe_pct": "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active",
    "issue_pct": "smsp__issue_active.avg.pct_of_peak_sustained_active",
    "warps_active_pct": "sm__warps_active.avg.pct_of_peak_sustained_active",
    "inst_executed": "smsp__inst_executed.sum",
    "inst_fp64_pipe": "sm__inst_executed_pipe_fp64.sum",
    "branches": "smsp__inst_executed_op_branch.sum",
    "spill_inst": "sass__inst_executed_register_spilling",
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


def entry_from(csv_path, source_hash=None):
    line = None
    for ln in open(os.path.splitext(csv_path)[0] + ".json"):
        if ln.startswith("{"):
            line = json.loads(ln)
    cfg, roof = line["config"], line["roofline"]
    key = "%s_%s_n%d_d%d" % (cfg["name"], cfg["split"], cfg["n_slices"], cfg["romberg_depth"])
    particles, turns = cfg["particles_per_gpu"], cfg["turns_per_step"]
    raw = read_raw(csv_path)
    got = {k: to_float(*raw[name]) for k, name in WANT.items() if name in raw and raw[name][0] not in ("n/a", "")}
    flop = 2 * got["dfma"] + got["dadd"] + got["dmul"]
    pt = particles * turns
    kname = roof["kernel"].split("::")[1].split("<")[0]
    info = dict(roof["kernel_info"])
    if "source_hash" not in info:      # a line printed before bench.py carried the fingerprint: name it on the command line
        if not source_hash:
            raise SystemExit("%s: no kernel source fingerprint in the bench line; pass --source-hash" % csv_path)
        info["source_hash"] = source_hash
    return key, {
        "flop_per_particle_turn": flop / pt,
        "dfma_per_particle_turn": got["dfma"] / pt, "dadd_per_particle_turn": got["dadd"] / pt,
        "dmul_per_particle_turn": got["dmul"] / pt,
        "fp64_inst_per_particle_turn": (got["dfma"] + got["dadd"] + got["dmul"]) / pt,
        "warp_inst_per_warp_turn": got.get("inst_executed", 0) / (pt / 32.0),
        "dram_bytes_per_launch": got.get("dram_read", 0) + got.get("dram_write", 0),
        "capture": {"particles": particles, "turns": turns, "duration_ms": got.get("duration_ns", 0) / 1e6,
                    "kernel": kname, "kernel_info": info,
                    "registers_per_thread": got.get("regs"), "fp64_pipe_pct_of_peak": got.get("fp64_pipe_pct"),
                    "issue_active_pct": got.get("issue_pct"), "warps_active_pct": got.get("warps_active_pct"),
                    "spill_instructions": got.get("spill_inst"), "branch_instructions": got.get("branches")},
        "source": os.path.relpath(csv_path, HERE),
    }


def main():
    model = json.load(open(OUT)) if os.path.exists(OUT) else {}
    args = sys.argv[1:]
    source_hash = None
    if "--source-hash" in args:
        k = args.index("--source-hash")
        source_hash = args[k + 1]
        del args[k:k + 2]
    for path in args:
        key, entry = entry_from(path, source_hash)
        model[key] = entry
        print(key, "%.0f flop/particle-turn, %.0f fp64 instructions, kernel %s %s"
              % (entry["flop_per_particle_turn"], entry["fp64_inst_per_particle_turn"], entry["capture"]["kernel"],
                 entry["capture"]["kernel_info"]))
    json.dump(model, open(OUT, "w"), indent=1, sort_keys=True)


if __name__ == "__main__":
    main()
