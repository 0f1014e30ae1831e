"""bench.py as the driver launches it, on a shortened step (16 turns): the one JSON line carries every key of the
measurement contract, the CUDA path ran (its kernel is named, launches are counted, nothing was lost), the end-to-end
leg copied what it says, and the roofline fraction comes from a flop count captured on the loaded kernels.  The same
under torchrun with one rank (the N > 1 launch: NCCL rendezvous on 127.0.0.1, barrier, max over ranks, all-reduce),
and the reference arm (the oracle on the host cores)."""
import json
import os
import socket
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SHORT = ["--steps", "2", "--warmup", "3", "--turns", "16"]


def run_bench(cmd, timeout=600):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    p = subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=timeout)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [l for l in p.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, p.stdout[-2000:]
    return json.loads(lines[0])


def check_line(d, n_gpus):
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline"):
        assert k in d, k
    assert d["n_gpus"] == n_gpus and d["steps"] == 2 and d["warmup"] == 3 and d["higher_is_better"] is True
    assert d["scaling"] == "weak" and d["dtype"] == "f64" and d["data"] == "synthetic" and d["vs_baseline"] is None
    assert "workload" in d["config"] and d["config"]["particles_per_gpu"] == 65536 and d["config"]["turns_per_step"] == 16
    assert d["lost"] == 0 and d["gpu_launches"] >= 3 * d["steps"]
    steps = d["config"]["steps_per_particle_turn"] * 65536 * 16 * n_gpus
    assert abs(d["value"] - steps / (d["ms_per_step"] * 1e-3)) < 1e-6 * d["value"]
    assert 5e10 < d["value"] < 1e12                      # a B200 does 2e11; a CPU fallback would do 2e8
    e = d["e2e"]
    assert e["h2d_bytes_per_step"] == 72 * 65536 and e["d2h_bytes_per_step"] >= 72 * 65536 and 0 < e["value"] <= 1.05 * d["value"]
    r = d["roofline"]
    assert r["bound"] == "alu" and r["kernel"].startswith("gst::track_chain_kernel") and r["kernel_ms"] <= d["ms_per_step"]
    # the committed flop model was captured on exactly these kernels (registers, stack frame, source fingerprint)
    assert r["frac"] is not None and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9 and 0.3 < r["frac"] < 1.0
    assert d["clocks"]["sm_mhz"] is None or d["clocks"]["sm_mhz"] > 0


def test_bench_line_of_the_default_launch():
    d = run_bench([sys.executable, "bench.py"] + SHORT + ["--no-cpu-baseline"])
    check_line(d, 1)


def test_bench_line_under_torchrun_with_one_rank():
    with socket.socket() as sk:                          # a port that is free right now
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    d = run_bench([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "1", "--master-addr",
                   "127.0.0.1", "--master-port", str(port), "bench.py", "--gpus", "1"] + SHORT + ["--no-cpu-baseline"])
    check_line(d, 1)
    assert "particle shards x1" in d["config"]["parallelism"]


def test_reference_arm_runs_the_oracle_on_the_host():
    d = run_bench([sys.executable, "bench.py", "--impl", "reference", "--steps", "1", "--warmup", "1"])
    assert d["impl"] == "reference" and d["gpu_launches"] == 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["value"] == d["value"] and d["e2e"]["h2d_bytes_per_step"] == 0 and 1e6 < d["value"] < 5e9
