"""world_size-2 gloo test of the N>1 path's host logic: sharding + the polarization all-reduce."""
import os
import socket

import numpy as np
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


def test_shard_bounds_cover_everything_once():
    for n in (0, 1, 7, 65536, 65537):
        for w in (1, 2, 3, 8):
            b = [D.shard_bounds(n, r, w) for r in range(w)]
            assert b[0][0] == 0 and b[-1][1] == n
            assert all(b[i][1] == b[i + 1][0] for i in range(w - 1))
