"""-m "not gpu": the N > 1 plumbing of bench.py on CPU (gloo, world_size 2).

The path does not shard (replicas only), so the only multi-rank logic is: every rank runs
its own replica, the per-rank device timings are reduced with MAX, value = N x pairs / max time, and only rank 0
prints.  This test runs that logic in two gloo processes.
"""
import os
import socket
import sys

import pytest

torch = pytest.importorskip("torch")
import torch.multiprocessing as mp  # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r "measured" 10 + r ms for the device leg and 20 + 2r ms for the host leg
    got = bench.max_over_ranks([10.0 + rank, 20.0 + 2 * rank], dist, torch.device("cpu"))
    value = bench.whole_job_rate(1_000_000_000, 5, world, got[0])
    with open(os.path.join(out_dir, f"rank{rank}.txt"), "w") as f:
        f.write(f"{got[0]} {got[1]} {value}\n")
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_rate_world2(tmp_path):
    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    for rank in range(world):
        a, b, v = map(float, open(tmp_path / f"rank{rank}.txt").read().split())
        assert (a, b) == (11.0, 22.0)                       # MAX over ranks, identical on every rank
        assert v == pytest.approx(2 * 1e9 * 5 / 11e-3 / 1e9)  # whole-job pairs / slowest rank


def test_single_process_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([3.5, 7.0], None, None) == [3.5, 7.0]
    assert bench.whole_job_rate(4_512_452_500, 10, 1, 45.0) == pytest.approx(1002.767, rel=1e-5)


def test_sample_problem_is_pure_slicing():
    sys.path.insert(0, ROOT)
    import bench
    from paper_1808_01478_b200 import inputs
    p = inputs.reduced_config(4)
    s = bench.sample_problem(p, 0.25, 2)
    assert s.n_frames == 2 and s.species_counts() == [275, 1075] and s.n_bins == p.n_bins and s.r_max == p.r_max
    assert (s.coords[1, 275] == p.coords[1, 1100]).all()      # first particle of species 1
