"""world_size-2 gloo test of the N>1 path's host logic: sharding + the polarization all-reduce."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1501_03450_b200 import distributed as D


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, S, alive_mask, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    lo, hi = D.shard_bounds(S.shape[1], rank, world)
    m = alive_mask[lo:hi]
    loc = S[:, lo:hi][:, m]
    pol = loc.mean(axis=1) if loc.shape[1] else np.zeros(3)
    g, alive = D.global_polarization(np.append(pol, np.linalg.norm(pol)), int(m.sum()))
    if rank == 0:
        out.put((g, alive))
    dist.destroy_process_group()


def test_sharded_polarization_equals_whole_bunch():
    rng = np.random.default_rng(0)
    n = 1001
    S = rng.normal(size=(3, n))
    S /= np.linalg.norm(S, axis=0)
    mask = rng.uniform(size=n) > 0.05
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, S, mask, out)) for r in range(2)]
    for p in procs:
        p.start()
    g, alive = out.get(timeout=120)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    ref = S[:, mask].mean(axis=1)
    assert alive == int(mask.sum())
    assert np.max(np.abs(g[:3] - ref)) < 1e-15 and abs(g[3] - np.linalg.norm(ref)) < 1e-15


def _record(X, Px, Y, Py, S, alive):
    """The record of include/gst.h gst_moments, from its definition (numpy)."""
    S, X, Px, Y, Py = S[:, alive], X[alive], Px[alive], Y[alive], Py[alive]
    n = float(alive.sum())
    rec = np.zeros(20)
    rec[0:3] = S.sum(axis=1)
    rec[3] = n
    rec[4:8] = [X.sum(), Px.sum(), Y.sum(), Py.sum()]
    if n > 0:
        for k, (u, p) in enumerate(((X, Px), (Y, Py))):
            du, dp = u - u.mean(), p - p.mean()
            rec[8 + 3 * k: 11 + 3 * k] = [(du * du).sum(), (dp * dp).sum(), (du * dp).sum()]
            rec[14 + 3 * k: 17 + 3 * k] = [n * u.mean() ** 2, n * p.mean() ** 2, n * u.mean() * p.mean()]
    return rec


def _bunch(n, seed):
    rng = np.random.default_rng(seed)
    X, Px, Y, Py = (rng.normal(size=n) * s for s in (1e-3, 1e-4, 2e-3, 3e-4))
    Px += 0.3 * X                                                  # correlated planes: the cross term counts
    X += 5e-3                                                      # offset beam
    S = rng.normal(size=(3, n))
    S /= np.linalg.norm(S, axis=0)
    return X, Px, Y, Py, S, rng.uniform(size=n) > 0.05


def _emittance(u, p):
    return np.sqrt(np.var(u) * np.var(p) - np.mean((u - u.mean()) * (p - p.mean())) ** 2)


def test_records_of_shards_add_up_to_the_whole_bunch():
    """gst_moments_finish (host arithmetic of the library) on a sum of shard records against numpy on the whole
    bunch: uneven shards, an empty one, one shifted against the others."""
    from paper_1501_03450_b200 import gst
    X, Px, Y, Py, S, alive = _bunch(5000, 1)
    Y[3000:] += 4e-3
    total = np.zeros(20)
    for lo, hi in ((0, 1), (1, 1), (1, 3000), (3000, 5000)):
        total += _record(X[lo:hi], Px[lo:hi], Y[lo:hi], Py[lo:hi], S[:, lo:hi], alive[lo:hi])
    pol, exy, n_alive = gst.moments_finish(total)
    assert n_alive == int(alive.sum())
    assert np.max(np.abs(pol[:3] - S[:, alive].mean(axis=1))) < 1e-15
    ref = np.array([_emittance(X[alive], Px[alive]), _emittance(Y[alive], Py[alive])])
    assert np.max(np.abs(exy / ref - 1)) < 1e-12
    pol1, exy1, _ = gst.moments_finish(_record(X, Px, Y, Py, S, alive))     # one record: the between-shard term is zero
    assert np.max(np.abs(exy1 / ref - 1)) < 1e-12 and np.max(np.abs(pol1 - pol)) < 1e-15
    pol0, exy0, n0 = gst.moments_finish(np.zeros(20))                       # nobody left
    assert n0 == 0 and not pol0.any() and not exy0.any()
    with pytest.raises(gst.GstError):
        gst.moments_finish(np.full(20, np.nan))


def _report_worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    X, Px, Y, Py, S, alive = _bunch(4001, 2)
    lo, hi = D.shard_bounds(4001, rank, world)
    rep = D.global_report(_record(X[lo:hi], Px[lo:hi], Y[lo:hi], Py[lo:hi], S[:, lo:hi], alive[lo:hi]))
    out.put((rank, rep))
    dist.destroy_process_group()


def test_global_report_is_one_allreduce_of_the_records():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_report_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    reps = dict(out.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    X, Px, Y, Py, S, alive = _bunch(4001, 2)
    ref = np.array([_emittance(X[alive], Px[alive]), _emittance(Y[alive], Py[alive])])
    for rank in (0, 1):                                                      # every rank holds the whole-bunch report
        pol, exy, n_alive = reps[rank]
        assert n_alive == int(alive.sum())
        assert np.max(np.abs(pol[:3] - S[:, alive].mean(axis=1))) < 1e-15
        assert np.max(np.abs(exy / ref - 1)) < 1e-12
    assert np.array_equal(reps[0][1], reps[1][1])


def test_shard_bounds_cover_everything_once():
    for n in (0, 1, 7, 65536, 65537):
        for w in (1, 2, 3, 8):
            b = [D.shard_bounds(n, r, w) for r in range(w)]
            assert b[0][0] == 0 and b[-1][1] == n
            assert all(b[i][1] == b[i + 1][0] for i in range(w - 1))


# ---------------------------------------------------------------------------------------------
# bench.py's own N>1 code path (rank-local bunches, barriers, max-over-ranks timing, the 5-double all-reduce) on two
# gloo ranks.  The tracking call is injected HERE: a stand-in for bench.CudaMachine that "tracks" by sleeping.
# ---------------------------------------------------------------------------------------------
class _StubSampler:
    def start(self):
        pass

    def stop(self):
        return {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}


class _StubMachine:
    dist_backend = "gloo"
    device = torch.device("cpu")

    def __init__(self, rank):
        self.rank = rank

    def open(self, cfg):
        from paper_1501_03450_b200 import workloads as W
        self.state = np.array(cfg["state"])
        self.state[6:9] = 0.0
        self.state[7] = 1.0 if self.rank == 0 else 0.5          # the ranks report different polarizations
        self.state[8] = 0.0 if self.rank == 0 else 0.25
        return W.steps_per_turn(cfg["lattice"], cfg["n_slices"])

    def track(self, turns, split, n_slices, depth):
        import time
        time.sleep(0.02 * (self.rank + 1))                      # rank 1 is the slow one

    def polarization(self):
        p = self.state[6:9].mean(axis=1)
        return np.append(p, np.linalg.norm(p)), 0

    def track_host(self, turns, split, n_slices, depth):
        self.track(turns, split, n_slices, depth)

    def last_kernel(self):
        return "stub"

    def flush(self, k):
        pass

    def sync(self):
        pass

    def mark(self):
        import time
        return time.perf_counter()

    @staticmethod
    def ms_between(a, b):
        return 1e3 * (b - a)

    def clock_sampler(self):
        return _StubSampler()

    def roofline(self, cfg, n, turns, spt, kernel_ms):
        return {"kernel_ms": kernel_ms}

    def close(self):
        pass


def _bench_worker(rank, world, port, out):
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    sys.path.insert(0, root)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    import bench
    args = bench.parse_args(["--gpus", "2", "--steps", "3", "--warmup", "1", "--config", "3", "--particles", "64",
                             "--turns", "2", "--no-cpu-baseline"])
    cfg = bench.configure(args)
    seed0 = cfg["state"].copy()
    line = bench.run_ours(args, cfg, _StubMachine(rank), args.config)
    out.put((rank, line, bool(np.array_equal(seed0, cfg["state"]))))
    dist.destroy_process_group()


def test_bench_rank_shard_and_allreduce_path_on_two_gloo_ranks():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_bench_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = dict((r, (line, same)) for r, line, same in (out.get(timeout=300) for _ in range(2)))
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    line, same0 = got[0]
    assert got[1][0] is None and line is not None                # rank 0 alone reports
    assert same0 and not got[1][1]                               # weak scaling: rank 1 drew its own bunch
    assert line["n_gpus"] == 2 and line["scaling"] == "weak" and line["lost"] == 0
    spt = line["config"]["steps_per_particle_turn"]
    units = 2 * 64 * 2 * spt                                     # BOTH ranks' particles x turns x steps per turn
    # the time is the slow rank's (max over ranks): 3 steps of >= 40 ms
    assert line["ms_per_step"] >= 40.0 and line["ms_per_step"] < 400.0
    assert abs(line["value"] - units / (line["ms_per_step"] * 1e-3)) < 1e-6 * line["value"]
    assert abs(line["e2e"]["value"] / line["value"] - 1) < 0.5
    # bunch-wide polarization = mean over both ranks' particles
    assert np.allclose(line["polarization"][:3], [0.0, 0.75, 0.125], atol=1e-15)
    assert abs(line["polarization"][3] - np.hypot(0.75, 0.125)) < 1e-15
