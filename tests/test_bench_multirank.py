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


def test_gpus_flag_starts_the_ranks_itself():
    """`python bench.py --gpus 2` without torchrun must start two ranks (here: gloo on the CPU, no GPU work)."""
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    env["CUDA_VISIBLE_DEVICES"] = ""
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--rank-check"], env=env,
                       capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(s) for s in r.stdout.splitlines() if s.startswith("{")]
    assert len(lines) == 1                                    # only rank 0 prints
    assert lines[0]["n_gpus"] == 2 and lines[0]["max_ms"] == 11.0
    assert lines[0]["value"] == pytest.approx(2 * 1e9 / 11e-3 / 1e9)


def test_both_arms_print_the_same_config_object():
    sys.path.insert(0, ROOT)
    import bench
    from paper_1808_01478_b200 import inputs
    p = inputs.config1()
    a = bench.config_block(p, bench.WORKLOADS[1], 1, (2, 3, 4, 5))
    b = bench.config_block(p, bench.WORKLOADS[1], 1, bench.GATING_CONFIGS)
    assert a == b and a["headline_config"] == 5 and a["configs_timed"] == [2, 3, 4, 5]


def test_expected_wavefronts_of_uniform_bins():
    sys.path.insert(0, ROOT)
    import numpy as np
    import bench
    # 32 uniform draws over many bins: the expected maximum load of 32 balls in 32 bins, about 3.5
    assert 3.4 < bench.expected_wavefronts(np.ones(50000), 1.0) < 3.65
    # one bin only: every lane hits the same address, which the hardware merges into one wavefront
    assert bench.expected_wavefronts(np.array([0.0, 5.0, 0.0]), 1.0) == 1.0
