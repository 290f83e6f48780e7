"""-m gpu: the double-precision path (precision CDH_F64) against the fp64 oracle, bin for bin.

Both sides run the pinned sequence in IEEE double; the float32 coordinates of the seeded
generators are widened to double exactly, so the histograms must be identical integers.
"""
import math

import numpy as np
import pytest

import paper_1808_01478_b200 as cdh
from paper_1808_01478_b200 import inputs
from oracle import oracle as cdh_oracle

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def gpu64(p, flags=0):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    with cdh.Context(0, flags) as ctx:
        out = cdh.histograms_device(ctx, p, precision=cdh.F64)
        torch.cuda.synchronize()
        return out.cpu().numpy().view(np.uint64), ctx.last_call_info()


def golden64(config, p):
    """The fp64 oracle's full-size histogram from tests/golden (written by make_fullsize.py, which calls only oracle/)."""
    from test_gpu_fullsize import golden
    return golden(config, p, "f64")


def oracle64(p):
    return cdh_oracle.histograms(p.coords.astype(np.float64), p.species_offsets, p.box_type, p.box, p.r_max, p.n_bins,
                                 precision="f64")


def same(got, want, what):
    if not np.array_equal(got, want):
        d = got.astype(np.int64) - want.astype(np.int64)
        raise AssertionError(f"{what}: {np.count_nonzero(d)} bins differ, L1 = {int(np.abs(d).sum())}, "
                             f"sums {int(got.sum())} / {int(want.sum())}")


@pytest.mark.parametrize("k", [1, 2, 3, 4, 5])
def test_reduced_configs_f64_bit_exact(k):
    p = inputs.reduced_config(k)
    got, info = gpu64(p)
    same(got, oracle64(p), f"{p.name} f64 {info}")


def test_f64_split_path_and_no_prune():
    p = inputs.reduced_config(3)
    want = oracle64(p)
    a, info = gpu64(p, 4000 << cdh.FLAG_MAX_SMEM_BINS_SHIFT)
    assert info["sweeps"] == 5
    same(a, want, "f64 bin-range split")
    b, _ = gpu64(p, cdh.FLAG_NO_PRUNE)
    same(b, want, "f64 27-shift search everywhere")


def test_f64_general_box_beyond_half_height_and_outside_coordinates():
    box = np.array([[9.0, 0.5, -0.25], [1.5, 8.0, 0.75], [-2.0, 2.5, 7.0]])
    for spread, r_max in ((1.0, 2.5), (3.5, 2.5), (1.0, 5.5)):
        p = inputs.uniform_problem(91, (700, 900), inputs.BOX_TRICLINIC, 3000, r_max, box=box, spread=spread)
        got, _ = gpu64(p)
        same(got, oracle64(p), f"general box spread={spread} r_max={r_max}")


def test_f64_hand_examples_and_total_count():
    pts = np.array([[1, 1, 1], [8, 8, 2], [2, 14, 9], [13, 3, 15]], dtype=np.float32)[None]
    box = np.array([[16.0, 0, 0], [0, 16.0, 0], [8.0, 8.0, 16.0]]).reshape(1, 9)
    p = inputs.Problem("p4", pts, np.array([0, 4], dtype=np.int32), inputs.BOX_TRICLINIC, box, 16.0, 16)
    got, _ = gpu64(p)
    want = np.zeros((1, 16), dtype=np.uint64); want[0, 5] = 1; want[0, 7] = 1; want[0, 8] = 1; want[0, 9] = 3   # pin P4
    same(got, want, "P4 in double")
    q = inputs.config1()
    got, _ = gpu64(q)
    assert int(got.sum()) == 1_999_000
    same(got, oracle64(q), "config 1 in double")


def test_f64_differs_from_f32_only_by_adjacent_bin_moves():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    p = inputs.reduced_config(2)
    with cdh.Context(0) as ctx:
        a = cdh.histograms_device(ctx, p).cpu().numpy().astype(np.int64)
        b = cdh.histograms_device(ctx, p, precision=cdh.F64).cpu().numpy().astype(np.int64)
    assert abs(int(a.sum()) - int(b.sum())) <= 8                     # pairs within a few ulp of r_max
    cum = np.abs(np.cumsum(a - b, axis=1))
    assert cum.max() <= 64                                           # moves between neighbouring bins only
    assert 0 < np.abs(a - b).sum() < 4 * p.n_bins * 2.0 ** -24 * p.evaluated_pairs * 2   # SURVEY.md 8c model bound


def test_f64_host_entry_point():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    p = inputs.reduced_config(4)
    with cdh.Context(0) as ctx:
        got = ctx.cdh_histograms_host(p.coords.astype(np.float64), p.species_offsets, p.box_type, p.box, p.r_max, p.n_bins,
                                      precision=cdh.F64)
    same(got, oracle64(p), "cdh_histograms_host in double")


def test_f64_config2_full_size():
    p = inputs.config2()
    got, info = gpu64(p)
    same(got, oracle64(p), f"config 2 full size in double {info}")
    assert got.sum() / p.evaluated_pairs == pytest.approx(math.pi / 6, rel=2e-3)


def test_f64_config3_full_size():
    """Config 3 at full size in double, tied to the fp64 oracle as tests/test_gpu_fullsize.py does in float: the
    (0,0) row outright, every row against the same kernels with the pruning off (27 shifts for every pair, the
    oracle's own order of work), and the closed-form kept fraction pi/12 (V = d^3 sqrt(2)/2, r_max = d sqrt(2)/4)."""
    p = inputs.config3()
    got, info = gpu64(p)
    assert info["sweeps"] == 1
    same(got, golden64(3, p)["hist"], "config 3 in double, all rows vs the oracle's full-size histogram")
    full, _ = gpu64(p, cdh.FLAG_NO_PRUNE)
    same(got, full, "config 3 in double: pruned vs 27-shift search everywhere")
    assert got.sum() / p.evaluated_pairs == pytest.approx(math.pi / 12, rel=2e-3)


def test_f64_config4_full_size():
    """Config 4 at full size in double: the 64-frame call equals the sum of 8-frame calls (Eq. 2) and the
    oracle computes one of the chunks outright."""
    p = inputs.config4()
    got, _ = gpu64(p)
    g = golden64(4, p)
    same(got, g["hist"], "config 4 in double, 64 frames in one call vs the oracle's full-size histogram")
    parts = np.zeros_like(got)
    for f0 in range(0, 64, 8):
        chunk = inputs.Problem(f"cfg4_{f0}", np.ascontiguousarray(p.coords[f0:f0 + 8]), p.species_offsets, p.box_type, p.box,
                               p.r_max, p.n_bins)
        h, _ = gpu64(chunk)
        same(h, g["chunk_hist"][f0 // 8], f"config 4 frames {f0}..{f0 + 7} in double vs the oracle's stored chunk sum")
        parts += h
    same(got, parts, "config 4 in double: 64 frames in one call vs the sum of 8-frame calls")
    assert got.sum() / p.evaluated_pairs == pytest.approx(math.pi / 6, rel=2e-3)


def test_f64_config5_full_size():
    """Config 5 at full size in double: every pair is binned, a species split adds up to the
    one-species histogram, and the oracle computes the (A, A) block outright."""
    p = inputs.config5()
    got, info = gpu64(p)
    assert info["sweeps"] == 1
    assert int(got.sum()) == 499_999_500_000
    same(got, golden64(5, p)["hist"], "config 5 in double, all 5e11 pairs vs the oracle's full-size histogram")
    n_a = 50_000
    sp = inputs.Problem("cfg5_split", p.coords, np.array([0, n_a, p.n_total], dtype=np.int32), p.box_type, p.box, p.r_max, p.n_bins)
    split, _ = gpu64(sp)
    same(split.sum(axis=0, keepdims=True), got, "config 5 in double: (A,A) + (A,B) + (B,B) vs the one-species call")
    a = inputs.Problem("cfg5_A", p.coords[:, :n_a], np.array([0, n_a], dtype=np.int32), p.box_type, p.box, p.r_max, p.n_bins)
    same(split[0:1], oracle64(a), "config 5 block (A,A) in double vs oracle")


def test_f64_sqrt_selftest_sample():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    assert cdh.cdh_selftest_sqrt_f64(7, 1 << 28) == 0


@pytest.mark.parametrize("seed", [21, 22, 23])
def test_f64_ortho_fused_and_plain_rint_awkward_boxes(seed):
    g = np.random.Generator(np.random.PCG64(seed))
    L = g.uniform(3.0, 40.0, size=3) * np.array([1.0, 1.0 / 3.0, math.pi])
    p = inputs.uniform_problem(seed, (1200, 1700), inputs.BOX_ORTHO, 5000, 0.5 * float(L.min()), box=np.diag(L))
    want = oracle64(p)
    a, _ = gpu64(p)                              # fused rint (coordinates inside the box)
    b, _ = gpu64(p, cdh.FLAG_NO_PRUNE)           # plain rint
    same(a, want, f"f64 fused rint L={L}")
    same(b, want, "f64 plain rint")
    q = inputs.uniform_problem(seed, (900, 800), inputs.BOX_ORTHO, 3000, 0.5 * float(L.min()), box=np.diag(L), spread=4.0)
    c, _ = gpu64(q)                              # range 4 > 1.49: the kernel itself falls back to the plain form
    same(c, oracle64(q), "f64 unwrapped coordinates")


def test_f64_ortho_half_box_switch_points():
    L = np.array([10.0, 7.3, 12.9])
    rows = [[0.0, 0.0, 0.0]]
    for ax in range(3):
        half = np.float64(L[ax] / 2)
        for k in range(-6, 7):
            v = half
            for _ in range(abs(k)):
                v = np.nextafter(v, np.inf if k > 0 else -np.inf)
            q = [0.0, 0.0, 0.0]; q[ax] = float(v)
            rows.append(q)
    pts = np.array(rows, dtype=np.float64)[None]
    off = np.array([0, 1, len(rows)], dtype=np.int32)
    box = np.diag(L).reshape(1, 9)
    want = cdh_oracle.histograms(pts, off, inputs.BOX_ORTHO, box, 30.0, 1 << 20, precision="f64")
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    with cdh.Context(0) as ctx:
        d = torch.from_numpy(pts).cuda()
        out = torch.empty((3, 1 << 20), dtype=torch.int64, device="cuda")
        ctx.cdh_histograms(d, 1, off, inputs.BOX_ORTHO, box, 30.0, 1 << 20, out, precision=cdh.F64)
        torch.cuda.synchronize()
    same(out.cpu().numpy().view(np.uint64), want, "f64 pairs within 6 ulp of L/2")


def test_f64_wide_histogram_global_and_split():
    p = inputs.uniform_problem(19, (4000,), inputs.BOX_NONE, 800_000, math.sqrt(3.0))
    want = oracle64(p)
    a, info = gpu64(p)
    assert info["hybrid"] and info["sweeps"] == 1             # a shared window of the bins + L2 updates, one sweep
    same(a, want, f"f64 800k bins, hybrid window {info}")
    g, info = gpu64(p, cdh.FLAG_GLOBAL_HIST)
    assert info["global_hist"] and info["sweeps"] == 1
    same(g, want, f"f64 800k bins, global histogram {info}")
    for nb in (60_000, 100_000, 200_000):                     # the bin counts just above one CTA's shared memory
        q = inputs.uniform_problem(23, (3000, 2000), inputs.BOX_ORTHO, nb, 3.0, box=np.diag([6.0, 7.0, 8.0]))
        h, info = gpu64(q)
        assert info["hybrid"] and info["sweeps"] == 1
        same(h, oracle64(q), f"f64 {nb} bins orthorhombic, hybrid window {info}")
    b, info = gpu64(p, 45000 << cdh.FLAG_MAX_SMEM_BINS_SHIFT)
    assert not info["global_hist"] and info["sweeps"] == 18
    same(b, want, f"f64 800k bins, 18 sweeps {info}")
    q = inputs.reduced_config(3)
    c, info = gpu64(q, cdh.FLAG_GLOBAL_HIST)
    same(c, oracle64(q), "f64 triclinic, forced global histogram")


@pytest.mark.parametrize("box_type", [inputs.BOX_NONE, inputs.BOX_ORTHO, inputs.BOX_TRICLINIC])
def test_f64_small_species_take_the_skip_variants(box_type):
    box = {inputs.BOX_NONE: None, inputs.BOX_ORTHO: np.diag([5.0, 6.0, 7.0]),
           inputs.BOX_TRICLINIC: np.array([[6.0, 0.0, 0.0], [1.0, 5.5, 0.0], [-0.5, 1.5, 5.0]])}[box_type]
    for counts in ((130,), (1025, 2047), (300, 1100, 2100), (4096, 3)):
        p = inputs.uniform_problem(sum(counts) + 1, counts, box_type, 1500, 2.2, box=box, n_frames=2)
        got, info = gpu64(p)
        assert info["skip"], f"{counts}: {info}"
        same(got, oracle64(p), f"f64 skip variant, box_type {box_type}, species {counts}")
    big = inputs.uniform_problem(9, (16000, 24000), box_type, 1500, 2.2, box=box)
    got, info = gpu64(big)
    assert not info["skip"], info
    same(got, oracle64(big), f"f64 large species, box_type {box_type}")


def test_f64_clean_forms_and_what_switches_them_off():
    """The double-precision kernels leave out the d < r_max compare where the call cannot drop a pair (no box: coordinate
    extent below r_max) or where dropped pairs have slots of their own (orthorhombic full-range histogram); NaN / inf
    coordinates, r_max inside the extent and inexact scales must fall back or stay exact."""
    g = np.random.Generator(np.random.PCG64(78))
    n = 6000
    base = g.random((n, 3)).astype(np.float32)
    cases = {"clean": (base, math.sqrt(3.0))}
    x = base.copy(); x[4321] = x[17]
    cases["coincident"] = (x, math.sqrt(3.0))
    x = base.copy(); x[5000, 1] = np.nan
    cases["nan"] = (x, math.sqrt(3.0))
    x = base.copy(); x[123, 0] = np.inf
    cases["inf"] = (x, math.sqrt(3.0))
    cases["r_max inside the extent"] = (base, 1.2)
    x = base.copy(); x[0] = (0.0, 0.0, 0.0); x[1] = (1.0, 1.0, 1.0)
    cases["corner to corner"] = (x, math.sqrt(3.0))            # d = sqrt(3) exactly in double: not below r_max, dropped
    for name, (pts, r_max) in cases.items():
        p = inputs.Problem(name, np.ascontiguousarray(pts[None]), np.array([0, 4097, n], dtype=np.int32), inputs.BOX_NONE, None,
                           r_max, 3000)
        got, info = gpu64(p)
        same(got, oracle64(p), f"f64 no box, {name}: {info}")
    for k, (diag, r_max, n_bins) in enumerate([((10.0, 10.0, 10.0), 5.0, 10000), ((8.0, 9.0, 7.5), 3.75, 3000),
                                               ((7.3, 8.1, 9.7), 3.65, 7777), ((6.0, 6.0, 6.0), 5.0, 2048)]):
        p = inputs.uniform_problem(600 + k, (2500, 1700), inputs.BOX_ORTHO, n_bins, r_max, box=np.diag(diag), n_frames=2, spread=1.2)
        got, info = gpu64(p)
        same(got, oracle64(p), f"f64 orthorhombic case {k}: {info}")
        if k == 0:
            assert info["full_range"]
            p.coords[1, 77, 0] = np.nan
            got, info = gpu64(p)
            same(got, oracle64(p), "f64 orthorhombic full-range histogram with a NaN coordinate")
