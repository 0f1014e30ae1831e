"""Particle-sharded multi-GPU helpers: particles are independent, so each
rank tracks its own contiguous shard with the lattice replicated and NO exchange during tracking.
The only collective on the path is the sum behind a bunch-wide report: one all-reduce of five doubles for the
polarization alone (global_polarization), of gst.MOMENTS_LEN = 20 doubles for polarization and emittances together
(global_report).  Works with any torch.distributed backend (nccl on GPUs, gloo in the CPU tests).
"""
import numpy as np


def shard_bounds(n, rank, world):
    """Contiguous particle range [lo, hi) of `rank`."""
    return n * rank // world, n * (rank + 1) // world


def global_polarization(local_pol, local_alive, device="cpu"):
    """Combine per-rank {Px,Py,Ps,|P|} and alive counts into the whole-bunch polarization (A18)."""
    import torch
    import torch.distributed as dist
    v = torch.zeros(5, dtype=torch.float64, device=device)
    v[:3] = torch.as_tensor(np.asarray(local_pol[:3]) * float(local_alive), dtype=torch.float64)
    v[3] = float(local_alive)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(v, op=dist.ReduceOp.SUM)
    v = v.cpu().numpy()
    alive = v[3]
    p = v[:3] / alive if alive > 0 else np.zeros(3)
    return np.array([p[0], p[1], p[2], float(np.linalg.norm(p))]), int(alive)


def global_report(local_record, device="cpu"):
    """Whole-bunch polarization {Px,Py,Ps,|P|}, rms emittances {eps_x, eps_y} and alive count from each rank's
    Bunch.moments() record (include/gst.h: gst_moments): the records add, so ONE all-reduce of 20 doubles, then
    gst_moments_finish on every rank."""
    import torch
    import torch.distributed as dist
    from . import gst
    v = torch.as_tensor(np.asarray(local_record, dtype=np.float64), dtype=torch.float64).to(device)
    assert v.numel() == gst.MOMENTS_LEN
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(v, op=dist.ReduceOp.SUM)
    return gst.moments_finish(v.cpu().numpy())
