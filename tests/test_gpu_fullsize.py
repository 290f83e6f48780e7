"""-m gpu: the five BASELINE.json configs at FULL size, in the launch configuration bench.py times.

Config 1 and 2: the whole result against the fp32 oracle.  Configs 3-5 are too large for the oracle to finish in
seconds, so the full-size result is tied to it through exact decompositions of the integer histogram:
  * a species split (extra offsets) turns one row into three rows that must add up to it, and the oracle computes
    the (A, A) block outright;
  * the sum over frames equals the sum of the per-chunk results, and the oracle computes one chunk outright;
  * the remaining rows are compared with the plain cross-validation kernel (CDH_FLAG_SIMPLE_KERNEL, library
    sqrtf / rintf / floorf, no pruning), itself pinned to the oracle on the oracle-sized blocks;
  * closed forms: total = N(N-1)/2 when r_max covers every pair, kept fraction = sphere / cell volume.
"""
import math

import numpy as np
import pytest

import paper_1808_01478_b200 as cdh
from paper_1808_01478_b200 import inputs
from oracle import oracle as cdh_oracle

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def run(ctx, p):
    out = cdh.histograms_device(ctx, p)
    torch.cuda.synchronize()
    return out.cpu().numpy().view(np.uint64)


def same(got, want, what):
    assert got.shape == want.shape, what
    if not np.array_equal(got, want):
        d = got.astype(np.int64) - want.astype(np.int64)
        raise AssertionError(f"{what}: {np.count_nonzero(d)} bins differ, L1 = {int(np.abs(d).sum())}")


@pytest.fixture(scope="module")
def ctx():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    with cdh.Context(0) as c:
        yield c


@pytest.fixture(scope="module")
def ctx_simple():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    with cdh.Context(0, cdh.FLAG_SIMPLE_KERNEL) as c:
        yield c


def with_offsets(p, offsets, name):
    return inputs.Problem(name, p.coords, np.asarray(offsets, dtype=np.int32), p.box_type, p.box, p.r_max, p.n_bins)


def test_config2_full_bit_exact(ctx):
    p = inputs.config2()
    got = run(ctx, p)
    same(got, cdh_oracle.problem_histograms(p, "f32"), "config 2, all six histograms")
    assert got.sum() / p.evaluated_pairs == pytest.approx(math.pi / 6, rel=2e-3)      # sphere r = L/2 in the cube


def test_config3_full(ctx, ctx_simple):
    p = inputs.config3()
    got = run(ctx, p)
    info = ctx.last_call_info()
    assert info["fast"] and info["sweeps"] == 1
    # (0,0) block outright against the oracle
    a = inputs.Problem("cfg3_A", p.coords[:, :40000], np.array([0, 40000], dtype=np.int32), p.box_type, p.box, p.r_max, p.n_bins)
    same(got[0:1], cdh_oracle.problem_histograms(a, "f32"), "config 3 row (0,0) vs oracle")
    # all rows against the cross-validation kernel (27 shifts for every pair)
    same(got, run(ctx_simple, p), "config 3 vs plain kernel")
    assert got.sum() / p.evaluated_pairs == pytest.approx(math.pi / 12, rel=2e-3)     # V = d^3 sqrt(2)/2, r = d sqrt(2)/4


def test_config4_full(ctx):
    p = inputs.config4()
    got = run(ctx, p)
    parts = np.zeros_like(got)
    for f0 in range(0, 64, 8):
        chunk = inputs.Problem(f"cfg4_{f0}", np.ascontiguousarray(p.coords[f0:f0 + 8]), p.species_offsets, p.box_type, p.box,
                               p.r_max, p.n_bins)
        h = run(ctx, chunk)
        if f0 == 24:
            same(h, cdh_oracle.problem_histograms(chunk, "f32"), "config 4 frames 24..31 vs oracle")
        parts += h
    same(got, parts, "config 4: 64 frames in one call vs the sum of 8-frame calls (Eq. 2)")
    assert got.sum() / p.evaluated_pairs == pytest.approx(math.pi / 6, rel=2e-3)


def test_config5_full(ctx):
    p = inputs.config5()
    got = run(ctx, p)
    info = ctx.last_call_info()
    assert info["sweeps"] == 1 and info["fast"]
    assert int(got.sum()) == 499_999_500_000                     # P1: every pair is binned
    n_a = 50_000
    split = run(ctx, with_offsets(p, [0, n_a, p.n_total], "cfg5_split"))
    same(split.sum(axis=0, keepdims=True), got, "config 5: (A,A) + (A,B) + (B,B) vs the one-species call")
    a = inputs.Problem("cfg5_A", p.coords[:, :n_a], np.array([0, n_a], dtype=np.int32), p.box_type, p.box, p.r_max, p.n_bins)
    same(split[0:1], cdh_oracle.problem_histograms(a, "f32"), "config 5 block (A,A) vs oracle")
    # permutation invariance at full size (the pinned sequence is odd-symmetric): reversed particle order
    rev = inputs.Problem("cfg5_rev", np.ascontiguousarray(p.coords[:, ::-1]), p.species_offsets, p.box_type, p.box, p.r_max, p.n_bins)
    same(run(ctx, rev), got, "config 5 reversed particle order")


def test_config5_cluster_major_order_is_the_same_histogram(ctx):
    # adversarial order for the shared atomics (a warp's particles come from one cluster): same integers
    p, q = inputs.config5(n=200_000), inputs.config5(n=200_000, cluster_major=True)
    same(run(ctx, q), run(ctx, p), "cluster-major order")
    assert int(run(ctx, q).sum()) == 200_000 * 199_999 // 2
