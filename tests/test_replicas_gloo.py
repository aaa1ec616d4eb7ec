"""N > 1 path on CPU: two gloo ranks run the bookkeeping bench.py uses under torchrun (DESIGN.md "Multi-GPU":
replicas, no data-path collective; whole-job value = sum of units / max of device time)."""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

from paper_2510_01785_b200 import replicas, synth  # noqa: E402


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world_size, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world_size))
    dist.init_process_group("gloo", rank=rank, world_size=world_size)
    try:
        assert replicas.world() == (rank, world_size)
        # each rank times its own replica: rank 1 is the slow one
        ms, units = (10.0, 4.0) if rank == 0 else (25.0, 4.0)
        tmax, usum = replicas.reduce_timing(ms, units)
        rate = replicas.whole_job_rate(ms, units)
        # replicas see different seeded data of the same shape
        a = synth.powerlaw_alm(replicas.rank_seed(101, rank), 8, 8, 1)
        gathered = [None] * world_size
        dist.all_gather_object(gathered, float(np.abs(a).sum()))
        lo, hi = replicas.channel_shard(7, rank, world_size)
        np.save(os.path.join(out_dir, f"r{rank}.npy"), np.array([tmax, usum, rate, gathered[0], gathered[1], lo, hi]))
    finally:
        dist.destroy_process_group()


def test_two_rank_replicas_gloo(tmp_path):
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r0 = np.load(tmp_path / "r0.npy")
    r1 = np.load(tmp_path / "r1.npy")
    for r in (r0, r1):
        assert r[0] == 25.0 and r[1] == 8.0  # max of times, sum of units
        assert r[2] == pytest.approx(8.0 / 25e-3)
        assert r[3] != r[4]  # different data per replica
    # the channel shards tile [0, 7) without overlap
    assert (r0[5], r0[6], r1[5], r1[6]) == (0, 4, 4, 7)


def test_single_process_defaults():
    assert replicas.world() == (0, 1)
    assert replicas.reduce_timing(3.0, 2.0) == (3.0, 2.0)
    assert replicas.whole_job_rate(4.0, 2.0) == pytest.approx(500.0)
    covered = []
    for r in range(5):
        lo, hi = replicas.channel_shard(3, r, 5)
        covered += list(range(lo, hi))
    assert covered == [0, 1, 2]
