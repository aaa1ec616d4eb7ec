"""Multi-GPU plumbing of the benchmark: the transform shards over independent batch
channels / whole transforms, so N ranks are N replicas with NO data-path collective.  What is shared between
ranks is only bookkeeping: which seeded inputs a rank generates, and the reduction of the device timings
(max over ranks) and of the units processed (sum over ranks).  Works on any torch.distributed backend
(`nccl` on the GPU box, `gloo` in the CPU tests).
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def world():
    """(rank, world_size) of the default process group, (0, 1) when torch.distributed is not initialised."""
    if dist.is_available() and dist.is_initialized():
        return dist.get_rank(), dist.get_world_size()
    return 0, 1


def rank_seed(seed: int, rank: int) -> int:
    """Seed of rank `rank`'s replica: every rank transforms different data of the same workload."""
    return int(seed) + 1000 * int(rank)


def spawn_ranks(nproc: int, argv, env=None) -> int:
    """Launch `nproc` ranks of the script `argv` (one per GPU of this node) the way the driver does -- torchrun with a
    loop-back rendezvous on a free port -- and return its exit code.  bench.py calls this when it is started plainly
    with --gpus N > 1 (no WORLD_SIZE in the environment), so that `python bench.py --gpus N` really runs N ranks."""
    import os
    import socket
    import subprocess
    import sys

    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={int(nproc)}",
           "--master-addr", "127.0.0.1", "--master-port", str(port)] + list(argv)
    return subprocess.run(cmd, env=dict(os.environ if env is None else env)).returncode


def reduce_timing(ms: float, units: float, device=None):
    """(max over ranks of `ms`, sum over ranks of `units`): whole-job time and whole-job work."""
    _, n = world()
    if n == 1:
        return float(ms), float(units)
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def whole_job_rate(ms: float, units: float, device=None) -> float:
    """units / s of the whole job: all ranks' units over the slowest rank's time."""
    tmax, usum = reduce_timing(ms, units, device)
    return usum / (tmax * 1e-3)
