"""-m gpu: the five BASELINE.json configs at FULL size, in the launch configuration bench.py times.

Config 1 and 2: the whole result against the fp32 oracle, run here.  Configs 3, 4, 5: every bin of every row against
the oracle's full-size histogram stored in tests/golden/cfg{3,4,5}_f32.npz (written once by tests/golden/make_fullsize.py,
which calls only oracle/; SURVEY.md 8d "compute once, cache on disk"); the stored file carries the sha256 of the input
bytes, re-checked here against the inputs the GPU is given.  On top of that, exact decompositions of the integer
histogram (kept from round 1; they exercise other launch shapes):
  * a species split (extra offsets) turns one row into three rows that must add up to it;
  * the sum over frames equals the sum of the per-chunk results, each chunk against the oracle's stored chunk sum;
  * the plain cross-validation kernel (CDH_FLAG_SIMPLE_KERNEL, library sqrtf / rintf / floorf, no pruning);
  * closed forms: total = N(N-1)/2 when r_max covers every pair, kept fraction = sphere / cell volume.
"""
import hashlib
import os
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


GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def golden(config, p, precision="f32"):
    """The oracle's stored full-size result; fails if the stored input hash is not that of ``p``."""
    d = np.load(os.path.join(GOLDEN, f"cfg{config}_{precision}.npz"))
    h = hashlib.sha256()
    h.update(np.ascontiguousarray(p.coords).tobytes())
    h.update(np.ascontiguousarray(p.species_offsets, dtype=np.int32).tobytes())
    h.update(b"" if p.box is None else np.ascontiguousarray(p.box, dtype=np.float64).tobytes())
    h.update(np.array([p.r_max], dtype=np.float64).tobytes())
    h.update(np.array([p.n_bins, p.box_type], dtype=np.int64).tobytes())
    assert h.hexdigest() == str(d["sha_inputs"]), "tests/golden was written for other inputs: rerun make_fullsize.py"
    return d


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
    same(got, golden(3, p)["hist"], "config 3, all three rows vs the oracle's full-size histogram")
    # and against the cross-validation kernel (27 shifts for every pair)
    same(got, run(ctx_simple, p), "config 3 vs plain kernel")
    assert got.sum() / p.evaluated_pairs == pytest.approx(math.pi / 12, rel=2e-3)     # V = d^3 sqrt(2)/2, r = d sqrt(2)/4


def test_config3_and_4_full_without_item_table():
    # the scheduler's other way to learn a work item (row search + Row + Seg instead of the descriptor table), many items per CTA
    with cdh.Context(0, cdh.FLAG_NO_ITEM_TABLE) as c:
        for k, p in ((3, inputs.config3()), (4, inputs.config4())):
            same(run(c, p), golden(k, p)["hist"], f"config {k} without the item table vs the oracle's full-size histogram")


def test_config4_full(ctx):
    p = inputs.config4()
    got = run(ctx, p)
    g = golden(4, p)
    same(got, g["hist"], "config 4, 64 frames in one call vs the oracle's full-size histogram")
    parts = np.zeros_like(got)
    for f0 in range(0, 64, 8):
        chunk = inputs.Problem(f"cfg4_{f0}", np.ascontiguousarray(p.coords[f0:f0 + 8]), p.species_offsets, p.box_type, p.box,
                               p.r_max, p.n_bins)
        h = run(ctx, chunk)
        same(h, g["chunk_hist"][f0 // 8], f"config 4 frames {f0}..{f0 + 7} vs the oracle's stored chunk sum")
        parts += h
    same(got, parts, "config 4: 64 frames in one call vs the sum of 8-frame calls (Eq. 2)")
    assert got.sum() / p.evaluated_pairs == pytest.approx(math.pi / 6, rel=2e-3)


def test_config5_full(ctx):
    p = inputs.config5()
    got = run(ctx, p)
    info = ctx.last_call_info()
    assert info["sweeps"] == 1 and info["fast"]
    assert int(got.sum()) == 499_999_500_000                     # P1: every pair is binned
    same(got, golden(5, p)["hist"], "config 5, all 5e11 pairs vs the oracle's full-size histogram")
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
