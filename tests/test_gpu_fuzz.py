"""-m gpu: seeded randomised differential test of the CUDA path against the oracle.

Many small problems with random box type and shape, species layout (empty / tiny / ragged species), frame count,
per-frame boxes, bin count, r_max (below and beyond half the box), coordinate spread (inside the cell, several cells
away), a few NaN coordinates and coincident points; fp32 and fp64, production kernels and forced variants.
Every histogram must equal the oracle's bin for bin.
"""
import os

import numpy as np
import pytest

import paper_1808_01478_b200 as cdh
from paper_1808_01478_b200 import inputs
from oracle import oracle as cdh_oracle

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

FLAGS = [0, 0, 0, cdh.FLAG_NO_PRUNE, cdh.FLAG_SIMPLE_KERNEL, cdh.FLAG_GLOBAL_HIST, 97 << cdh.FLAG_MAX_SMEM_BINS_SHIFT,
         cdh.FLAG_NO_ITEM_TABLE, cdh.FLAG_NO_PDL | cdh.FLAG_NO_ITEM_TABLE]


def random_problem(g):
    box_type = int(g.integers(0, 3))
    n_species = int(g.integers(1, 5))
    counts = [int(c) for c in g.choice([0, 1, 2, 3, 5, 31, 32, 33, 257, 600, 1023, 1025, 1500], size=n_species)]
    n = sum(counts)
    if n == 0:
        counts[0] = 7; n = 7
    n_frames = int(g.integers(1, 4))
    per_frame = box_type != 0 and n_frames > 1 and g.random() < 0.4
    n_boxes = n_frames if per_frame else 1
    spread = float(g.choice([1.0, 1.0, 1.3, 2.5, 6.0]))
    boxes, coords = [], np.empty((n_frames, n, 3), dtype=np.float32)
    for b in range(n_boxes):
        if box_type == 1:
            boxes.append(np.diag(g.uniform(2.0, 20.0, size=3) * g.choice([1.0, 1.0 / 3.0, np.pi])))
        elif box_type == 2:
            m = np.diag(g.uniform(4.0, 12.0, size=3))
            m[1, 0] = g.uniform(-2, 2); m[2, 0] = g.uniform(-2, 2); m[2, 1] = g.uniform(-2, 2)
            if g.random() < 0.5:
                m[0, 1] = g.uniform(-0.5, 0.5); m[0, 2] = g.uniform(-0.5, 0.5); m[1, 2] = g.uniform(-0.5, 0.5)
            boxes.append(m)
    for f in range(n_frames):
        s = (g.random((n, 3)) - 0.25) * spread
        if box_type == 0:
            coords[f] = (s * 3.0).astype(np.float32)
        else:
            coords[f] = (s @ boxes[f if per_frame else 0]).astype(np.float32)
    if n > 4 and g.random() < 0.3:
        coords[0, int(g.integers(0, n)), int(g.integers(0, 3))] = np.nan
    if n > 4 and g.random() < 0.3:
        coords[:, 1] = coords[:, 0]                                  # coincident points: d = 0
    if box_type == 0:
        box, scale = None, 3.0 * spread
    else:
        box = np.stack(boxes).reshape(n_boxes, 9)
        scale = float(min(np.linalg.norm(b, axis=1).min() for b in boxes))
    r_max = float(scale * g.choice([0.2, 0.45, 0.5, 0.8, 1.7]))
    n_bins = int(g.choice([1, 7, 100, 1000, 4097, 20000]))
    off = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
    return inputs.Problem("fuzz", coords, off, box_type, box, r_max, n_bins)


@pytest.mark.parametrize("chunk", range(8))
def test_fuzz_against_oracle(chunk):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    g = np.random.Generator(np.random.PCG64(int(os.environ.get("CDH_FUZZ_SEED", "20260000")) + chunk))   # other seeds: longer soaks
    for case in range(30):
        p = random_problem(g)
        flags = FLAGS[int(g.integers(0, len(FLAGS)))]
        f64 = g.random() < 0.3
        with cdh.Context(0, flags) as ctx:
            out = cdh.histograms_device(ctx, p, precision=cdh.F64 if f64 else cdh.F32)
            torch.cuda.synchronize()
            info = ctx.last_call_info()
        got = out.cpu().numpy().view(np.uint64)
        if f64:
            want = cdh_oracle.histograms(p.coords.astype(np.float64), p.species_offsets, p.box_type, p.box, p.r_max, p.n_bins,
                                         precision="f64")
        else:
            want = cdh_oracle.problem_histograms(p, "f32")
        if not np.array_equal(got, want):
            d = got.astype(np.int64) - want.astype(np.int64)
            raise AssertionError(f"chunk {chunk} case {case}: box_type {p.box_type}, counts {p.species_counts()}, frames {p.n_frames}, "
                                 f"boxes {p.n_boxes}, bins {p.n_bins}, r_max {p.r_max}, flags {flags:#x}, f64 {f64}, {info}: "
                                 f"{np.count_nonzero(d)} bins differ, L1 {int(np.abs(d).sum())}")
