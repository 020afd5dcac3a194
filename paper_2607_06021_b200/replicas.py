"""Multi-GPU plumbing for bench.py: the path does not shard (replicas only), so N ranks
run N independent solves (one process per GPU, different seeds) with no collective on the data path.  The only
communication is the timing protocol: barrier, max-over-ranks of the device time, sum of the units processed.
A batch of independent problems (lrp_cross_deim_solve_batch / _host) is split over the ranks by `shard`; `gather_ints`
collects the per-problem scalars (rank, sweeps, converged) for the report.  Works with any torch.distributed backend
(nccl on GPUs; gloo in the CPU tests)."""
from __future__ import annotations

import os


def env_world():
    """(rank, local_rank, world_size) from the torchrun environment (1-process defaults)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str, device=None):
    """Initialise torch.distributed from MASTER_ADDR/MASTER_PORT if WORLD_SIZE > 1; returns the module or None."""
    rank, _, world = env_world()
    if world <= 1:
        return None
    import torch.distributed as dist
    if not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        kw = {}
        if device is not None and backend == "nccl":
            kw["device_id"] = device
        dist.init_process_group(backend=backend, rank=rank, world_size=world, **kw)
    return dist


def barrier(dist):
    if dist is not None:
        dist.barrier()


def aggregate(dist, local_ms: float, local_units: float, device="cpu"):
    """Whole-job numbers: (max over ranks of the elapsed ms, sum over ranks of the units processed)."""
    if dist is None:
        return float(local_ms), float(local_units)
    import torch
    t = torch.tensor([float(local_ms)], dtype=torch.float64, device=device)
    u = torch.tensor([float(local_units)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def throughput(dist, local_ms: float, local_units: float, device="cpu") -> dict:
    ms, units = aggregate(dist, local_ms, local_units, device)
    return dict(ms=ms, units=units, per_s=units / (ms * 1e-3) if ms > 0 else 0.0)


def shard(nprob: int, rank: int, world: int) -> tuple[int, int]:
    """[lo, hi): the problems of a batch of `nprob` independent problems that `rank` of `world` solves -- contiguous blocks
    whose sizes differ by at most one; nothing is exchanged on the data path."""
    if nprob < 0 or world < 1 or not 0 <= rank < world:
        raise ValueError("shard: need nprob >= 0 and 0 <= rank < world")
    base, rem = divmod(nprob, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def gather_ints(dist, local: list[int], nprob: int, device="cpu") -> list[int]:
    """Per-problem integers of the whole batch, in problem order, on every rank: `local` holds this rank's block
    (the `shard` of nprob).  One all_reduce(SUM) of a zero-padded vector; no process group -> the list itself."""
    if dist is None:
        return list(local)
    import torch
    rank, world = dist.get_rank(), dist.get_world_size()
    lo, hi = shard(nprob, rank, world)
    if len(local) != hi - lo:
        raise ValueError("gather_ints: local list does not match this rank's shard")
    v = torch.zeros(nprob, dtype=torch.int64, device=device)
    if hi > lo:
        v[lo:hi] = torch.tensor(list(local), dtype=torch.int64, device=device)
    dist.all_reduce(v, op=dist.ReduceOp.SUM)
    return [int(x) for x in v.tolist()]
