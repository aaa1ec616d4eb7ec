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
        np.save(os.path.join(out_dir, f"r{rank}.npy"), np.array([tmax, usum, rate, gathered[0], gathered[1]]))
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


def test_single_process_defaults():
    assert replicas.world() == (0, 1)
    assert replicas.reduce_timing(3.0, 2.0) == (3.0, 2.0)
    assert replicas.whole_job_rate(4.0, 2.0) == pytest.approx(500.0)


_RANK_SCRIPT = """
import os, sys
import torch.distributed as dist
sys.path.insert(0, {root!r})
from paper_2510_01785_b200 import replicas
dist.init_process_group("gloo")
r, n = replicas.world()
t, u = replicas.reduce_timing(10.0 * (r + 1), 4.0)
open(os.path.join({out!r}, "rank%d.txt" % r), "w").write("%d %d %g %g %s" % (r, n, t, u, " ".join(sys.argv[1:])))
dist.destroy_process_group()
"""


def test_spawn_ranks_runs_n_ranks_of_the_same_command(tmp_path):
    """What `python bench.py --gpus 2` does when it is started without torchrun: replicas.spawn_ranks launches the
    ranks (torchrun, loop-back rendezvous) and every rank sees WORLD_SIZE = 2 and the original arguments."""
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    script = tmp_path / "rank_script.py"
    script.write_text(_RANK_SCRIPT.format(root=root, out=str(tmp_path)))
    rc = replicas.spawn_ranks(2, [str(script), "--gpus", "2", "--steps", "5"])
    assert rc == 0
    got = sorted((tmp_path / f"rank{r}.txt").read_text() for r in range(2))
    assert got == ["0 2 20 8 --gpus 2 --steps 5", "1 2 20 8 --gpus 2 --steps 5"]


def test_bench_self_spawn_branch_is_wired():
    """bench.py hands a plain `--gpus N` launch to replicas.spawn_ranks before it touches CUDA."""
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    src = open(os.path.join(root, "bench.py")).read()
    i = src.index('if args.gpus > 1 and "WORLD_SIZE" not in os.environ:')
    assert "replicas.spawn_ranks(args.gpus" in src[i:i + 400] and i < src.index("import torch.distributed as dist")
