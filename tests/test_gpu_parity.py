"""-m gpu: parity of the CUDA path (through the C ABI, include/cdh.h) with the CPU oracle, bin for bin.

Bar (BASELINE.json north_star): uint64 histograms BIT-EXACT to the fp32 oracle.  Every kernel variant
(production packed-f32x2 kernel, the plain cross-validation kernel, the bin-range-split path, forced
27-shift triclinic search) must give the same integers ("cross validation").
"""
import hashlib
import math

import numpy as np
import pytest

import paper_1808_01478_b200 as cdh
from paper_1808_01478_b200 import inputs
from oracle import oracle as cdh_oracle

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def _need_gpu():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")


def gpu_hist(p, flags=0, host=False):
    _need_gpu()
    with cdh.Context(0, flags) as ctx:
        if host:
            return ctx.cdh_histograms_host(p.coords, p.species_offsets, p.box_type, p.box, p.r_max, p.n_bins), \
                ctx.last_call_info()
        out = cdh.histograms_device(ctx, p)
        torch.cuda.synchronize()
        return out.cpu().numpy().view(np.uint64), ctx.last_call_info()


def assert_same(got, want, what):
    if not np.array_equal(got, want):
        diff = got.astype(np.int64) - want.astype(np.int64)
        rows, bins = np.nonzero(diff)
        raise AssertionError(f"{what}: {len(rows)} bins differ, L1={int(np.abs(diff).sum())}, "
                             f"sum got={int(got.sum())} want={int(want.sum())}, first at row {rows[0]} bin {bins[0]}: "
                             f"{int(got[rows[0], bins[0]])} vs {int(want[rows[0], bins[0]])}")


_oracle_cache = {}


def oracle_hist(p):
    key = (hashlib.sha1(p.coords.tobytes()).hexdigest(), tuple(p.species_offsets.tolist()), p.n_bins, p.r_max,
           p.box_type, None if p.box is None else p.box.tobytes())
    if key not in _oracle_cache:
        _oracle_cache[key] = cdh_oracle.problem_histograms(p, "f32")
    return _oracle_cache[key]


FLAG_SETS = {
    "fast": 0,
    "simple": cdh.FLAG_SIMPLE_KERNEL,
    "split3000": 3000 << cdh.FLAG_MAX_SMEM_BINS_SHIFT,
    "simple_split700": cdh.FLAG_SIMPLE_KERNEL | (700 << cdh.FLAG_MAX_SMEM_BINS_SHIFT),
    "global_hist": cdh.FLAG_GLOBAL_HIST,
    "simple_global_hist": cdh.FLAG_GLOBAL_HIST | cdh.FLAG_SIMPLE_KERNEL,
    "match_any": cdh.FLAG_WARP_AGGREGATE,
    "plain_add": cdh.FLAG_NO_AGGREGATE,
    "no_item_table": cdh.FLAG_NO_ITEM_TABLE,      # every item looked up in the row / segment tables (calls with > 262,144 items)
    "no_pdl": cdh.FLAG_NO_PDL,                    # tile launches fully serialised behind the repack kernel
}


@pytest.mark.parametrize("variant", sorted(FLAG_SETS))
@pytest.mark.parametrize("k", [1, 2, 3, 4, 5])
def test_reduced_configs_bit_exact(k, variant):
    p = inputs.reduced_config(k)
    got, info = gpu_hist(p, FLAG_SETS[variant])
    assert_same(got, oracle_hist(p), f"{p.name} [{variant}] {info}")
    cap = FLAG_SETS[variant] >> cdh.FLAG_MAX_SMEM_BINS_SHIFT
    if cap and p.n_bins > cap:
        assert info["sweeps"] == -(-p.n_bins // cap)


@pytest.mark.parametrize("counts,n_frames", [((10000,), 1), ((30000,), 1), ((6000, 9000), 3), ((700, 1900), 40)])
def test_every_pair_once_with_few_and_many_items_per_cta(counts, n_frames):
    # the scheduler's two ways to claim work (one item ahead; late, where a CTA gets few items) and its two ways to learn an
    # item (descriptor table; row search): r_max covers the unit cube, so the total must be the closed form (P1),
    # and all variants must agree bin for bin
    p = inputs.uniform_problem(4242 + sum(counts), counts, inputs.BOX_NONE, 3000, math.sqrt(3.0) * 1.0001, n_frames=n_frames)
    got, info = gpu_hist(p)
    assert int(got.sum()) == p.evaluated_pairs, info
    assert_same(gpu_hist(p, cdh.FLAG_NO_ITEM_TABLE)[0], got, "row search vs descriptor table")
    assert_same(gpu_hist(p, cdh.FLAG_NO_PDL)[0], got, "serialised launch vs early launch")
    assert_same(gpu_hist(p, cdh.FLAG_SIMPLE_KERNEL)[0], got, "cross-validation kernel")


def test_config1_full_and_total_count():
    p = inputs.config1()
    got, _ = gpu_hist(p)
    assert int(got.sum()) == 1_999_000          # P1: N(N-1)/2, r_max covers all pairs
    assert_same(got, oracle_hist(p), p.name)


def test_host_entry_point_matches_device_entry_point():
    p = inputs.reduced_config(2)
    a, _ = gpu_hist(p)
    b, _ = gpu_hist(p, host=True)
    assert_same(b, a, "cdh_histograms_host vs cdh_histograms")
    assert_same(b, oracle_hist(p), "cdh_histograms_host")


def test_triclinic_no_prune_equals_prune_and_oracle():
    p = inputs.reduced_config(3)
    a, _ = gpu_hist(p)
    b, _ = gpu_hist(p, cdh.FLAG_NO_PRUNE)
    assert_same(b, a, "27-shift search vs exact pruning")
    assert_same(a, oracle_hist(p), p.name)


def test_triclinic_beyond_half_height_runs_full_search():
    # r_max > h_min/2: Eq. 5 alone is not exact; the neighbour search decides.
    p = inputs.config3(counts=(1500, 2100), n_bins=4000, r_max=6.0)
    got, _ = gpu_hist(p)
    assert_same(got, oracle_hist(p), "cfg3 r_max=6")


def test_triclinic_general_box_and_far_outside_coordinates():
    box = np.array([[9.0, 0.5, -0.25], [1.5, 8.0, 0.75], [-2.0, 2.5, 7.0]])
    heights_min = 5.0
    for spread, tag in ((1.0, "inside"), (3.5, "outside")):
        p = inputs.uniform_problem(77, (900, 1300), inputs.BOX_TRICLINIC, 3000, heights_min / 2, box=box, spread=spread)
        got, info = gpu_hist(p)
        assert_same(got, oracle_hist(p), f"general triclinic {tag} {info}")


def test_upper_triangular_box_variant():
    box = np.array([[10.0, 0.0, 0.0], [3.0, 9.0, 0.0], [-2.0, 4.0, 8.0]])
    p = inputs.uniform_problem(78, (1000, 1200), inputs.BOX_TRICLINIC, 2500, 3.9, box=box)
    got, info = gpu_hist(p)
    assert_same(got, oracle_hist(p), f"upper triangular {info}")


def test_ortho_unwrapped_coordinates_and_per_frame_boxes():
    g = np.random.Generator(np.random.PCG64(5))
    n, f = 2100, 3
    coords = (g.random((f, n, 3)) * 30.0 - 10.0).astype(np.float32)      # several box lengths outside
    boxes = np.stack([np.diag([6.0 + k, 7.0, 8.0 - k]) for k in range(f)]).reshape(f, 9)
    p = inputs.Problem("ortho_per_frame_boxes", coords, np.array([0, 600, n], dtype=np.int32), inputs.BOX_ORTHO,
                       boxes, 2.9, 1234)
    got, _ = gpu_hist(p)
    assert_same(got, oracle_hist(p), p.name)


@pytest.mark.parametrize("seed", [11, 12, 13, 14])
def test_ortho_awkward_box_lengths_fused_and_plain_rint(seed):
    # box lengths with full 24-bit mantissas: the fused rint needs a host-searched constant per axis; coordinates
    # wrapped into the box take the fused form, NO_PRUNE forces the plain magic-number form, both must equal the oracle
    g = np.random.Generator(np.random.PCG64(seed))
    L = g.uniform(3.0, 40.0, size=3) * np.array([1.0, 1.0 / 3.0, math.pi])
    p = inputs.uniform_problem(seed, (1500, 2100), inputs.BOX_ORTHO, 5000, 0.5 * float(L.min()), box=np.diag(L))
    a, info_a = gpu_hist(p)
    b, info_b = gpu_hist(p, cdh.FLAG_NO_PRUNE)
    assert info_a["form"] in (1, 2) and info_b["form"] == 0      # fused or exact-product form vs the pinned 5-operation form
    assert_same(a, oracle_hist(p), f"rint form {info_a['form']}, L={L}")
    assert_same(b, a, "plain vs fused / exact-product rint")


def test_ortho_rint_forms_all_occur():
    # over a handful of seeded boxes both the fused form (constants found for all axes) and the exact-product form occur
    forms = set()
    for seed in range(50, 62):
        g = np.random.Generator(np.random.PCG64(seed))
        L = g.uniform(3.0, 40.0, size=3)
        p = inputs.uniform_problem(seed, (700, 900), inputs.BOX_ORTHO, 3000, 0.5 * float(L.min()), box=np.diag(L))
        got, info = gpu_hist(p)
        forms.add(info["form"])
        assert_same(got, oracle_hist(p), f"form {info['form']} L={L}")
    assert forms == {1, 2}


def test_ortho_pairs_on_the_half_box_switch_point():
    # separations within a few ulps of L/2 on every axis: where n = rint(d/L) switches between 0 and +-1
    L = np.array([10.0, 7.3, 12.9])
    rows = [[0.0, 0.0, 0.0]]
    for ax in range(3):
        half = np.float32(L[ax] / 2)
        for k in range(-6, 7):
            v = half
            for _ in range(abs(k)):
                v = np.nextafter(v, np.float32(np.inf if k > 0 else -np.inf))
            q = [0.0, 0.0, 0.0]; q[ax] = float(v)
            rows.append(q)
    pts = np.array(rows, dtype=np.float32)[None]
    for r_max in (6.0, 30.0):
        p = inputs.Problem(f"halfbox{r_max}", pts, np.array([0, 1, len(rows)], dtype=np.int32), inputs.BOX_ORTHO,
                           np.diag(L).reshape(1, 9), r_max, 1 << 20)
        got, _ = gpu_hist(p)
        assert_same(got, oracle_hist(p), p.name)


def test_p2_hand_example_species_split():
    pts = np.array([[0, 0, 0], [3, 4, 0], [3, 4, 12], [0, 0, 12]], dtype=np.float32)[None]
    p = inputs.Problem("p2", pts, np.array([0, 2, 4], dtype=np.int32), inputs.BOX_NONE, None, 16.0, 16)
    got, _ = gpu_hist(p)
    want = np.zeros((3, 16), dtype=np.uint64)
    want[0, 5] = 1; want[1, 12] = 2; want[1, 13] = 2; want[2, 5] = 1          # SURVEY.md 8c pin P2
    assert_same(got, want, "P2 hand example")
    p13 = inputs.Problem("p2b", pts, np.array([0, 4], dtype=np.int32), inputs.BOX_NONE, None, 13.0, 13)
    got, _ = gpu_hist(p13)
    want = np.zeros((1, 13), dtype=np.uint64); want[0, 5] = 2; want[0, 12] = 2   # d = 13 dropped (Q2)
    assert_same(got, want, "P2 r_max=13")


def test_p4_triclinic_hand_example():
    pts = np.array([[1, 1, 1], [8, 8, 2], [2, 14, 9], [13, 3, 15]], dtype=np.float32)[None]
    box = np.array([[16.0, 0, 0], [0, 16.0, 0], [8.0, 8.0, 16.0]]).reshape(1, 9)
    p = inputs.Problem("p4", pts, np.array([0, 4], dtype=np.int32), inputs.BOX_TRICLINIC, box, 16.0, 16)
    got, _ = gpu_hist(p)
    want = np.zeros((1, 16), dtype=np.uint64); want[0, 5] = 1; want[0, 7] = 1; want[0, 8] = 1; want[0, 9] = 3
    assert_same(got, want, "P4 hand example")


def test_p8_single_bin_exceeds_uint32():
    # 100,000 identical points: bin 0 = 4,999,950,000 > 2^32 (flush rule)
    pts = np.full((1, 100_000, 3), 0.25, dtype=np.float32)
    p = inputs.Problem("p8", pts, np.array([0, 100_000], dtype=np.int32), inputs.BOX_NONE, None, 1.0, 64)
    got, _ = gpu_hist(p)
    assert int(got[0, 0]) == 4_999_950_000 and int(got.sum()) == 4_999_950_000


def test_p9_wide_histogram_global_and_split_paths():
    # 1,000,000 bins = 4 MB >> shared memory: beyond 16 shared windows the global-histogram mode takes over by itself;
    # a cap on the shared bins forces the bin-range-split path (20 sweeps) instead; both must equal the oracle
    p = inputs.uniform_problem(9, (6000,), inputs.BOX_NONE, 1_000_000, math.sqrt(3.0))
    got, info = gpu_hist(p)
    assert info["global_hist"] and info["sweeps"] == 1
    assert_same(got, oracle_hist(p), f"1M bins, global histogram {info}")
    got, info = gpu_hist(p, 50000 << cdh.FLAG_MAX_SMEM_BINS_SHIFT)
    assert not info["global_hist"] and info["sweeps"] == 20
    assert_same(got, oracle_hist(p), f"1M bins, 20 sweeps {info}")
    q = inputs.uniform_problem(10, (2500, 3000), inputs.BOX_ORTHO, 400_000, 3.0, box=np.diag([6.0, 7.0, 8.0]))
    got, info = gpu_hist(q)
    assert info["hybrid"] and info["sweeps"] == 1
    assert_same(got, oracle_hist(q), f"400k bins orthorhombic, hybrid window {info}")
    got, info = gpu_hist(q, cdh.FLAG_GLOBAL_HIST)
    assert info["global_hist"]
    assert_same(got, oracle_hist(q), f"400k bins orthorhombic, forced global histogram {info}")


@pytest.mark.parametrize("n_bins", [56_000, 60_000, 100_000, 200_000])
@pytest.mark.parametrize("box_type", [inputs.BOX_NONE, inputs.BOX_ORTHO, inputs.BOX_TRICLINIC])
def test_hybrid_window_single_sweep(n_bins, box_type):
    """Bin counts just above what one CTA's shared memory holds (the paper's staircase of sweeps,
    PAPER.md:205, 308-316): one sweep with the most populated window of every row in shared memory and the rest in L2.
    Several species, so that every row picks its own window; also a clustered set (config-5 recipe), whose first bins
    are far more populated than a uniform set's."""
    box = {inputs.BOX_NONE: None, inputs.BOX_ORTHO: np.diag([5.0, 6.0, 7.0]),
           inputs.BOX_TRICLINIC: np.array([[6.0, 0.0, 0.0], [1.0, 5.5, 0.0], [-0.5, 1.5, 5.0]])}[box_type]
    r_max = 9.0 if box_type == inputs.BOX_NONE else 2.4
    p = inputs.uniform_problem(n_bins + box_type, (2100, 4200, 900), box_type, n_bins, r_max, box=box, spread=5.0 if box_type == inputs.BOX_NONE else 1.0)
    got, info = gpu_hist(p)
    assert info["sweeps"] == 1 and info["hybrid"] == (n_bins > 56_402), info
    assert_same(got, oracle_hist(p), f"{n_bins} bins, box {box_type}: {info}")
    if box_type == inputs.BOX_NONE:
        c = inputs.config5(n=12_000, n_bins=n_bins, n_clusters=25)
        got, info = gpu_hist(c)
        assert_same(got, oracle_hist(c), f"{n_bins} bins, clustered set: {info}")
        assert int(got.sum()) == 12_000 * 11_999 // 2


@pytest.mark.parametrize("box_type", [inputs.BOX_ORTHO, inputs.BOX_TRICLINIC])
@pytest.mark.parametrize("n_bins", [40_000, 70_000])
@pytest.mark.parametrize("spread", [1.0, 5.0, 200.0, 3.0e6])
def test_one_cta_per_sm_plans_in_every_range_tier(box_type, n_bins, spread):
    """40,000 bins: one 512-thread CTA per SM (periodic boxes); 70,000 bins: the hybrid plans (1,024 threads orthorhombic, 512
    triclinic).  The work tables of a plan are built for ONE i-tile size, so the launch that owns the measured coordinate range
    -- fast narrow form, wide / plain-rint form, or the cross-validation kernel far outside -- must have the CTA size of the
    plan's first launch.  Coordinates inside the cell, a few cells away, hundreds of cells away, millions of cells away."""
    box = np.diag([5.0, 6.0, 7.0]) if box_type == inputs.BOX_ORTHO else np.array([[6.0, 0.0, 0.0], [1.0, 5.5, 0.0], [-0.5, 1.5, 5.0]])
    p = inputs.uniform_problem(int(n_bins + spread) % 9973, (1300, 2900), box_type, n_bins, 2.4, box=box, spread=spread)
    got, info = gpu_hist(p)
    assert info["ctas"] <= 148 and info["threads"] in (512, 1024) and info["hybrid"] == (n_bins > 56_402), info
    assert_same(got, oracle_hist(p), f"{n_bins} bins, box {box_type}, spread {spread}: {info}")


def test_empty_species_tiny_inputs_and_nan():
    pts = np.array([[0.1, 0.2, 0.3], [0.5, 0.5, 0.5], [np.nan, 0.0, 0.0], [0.9, 0.1, 0.4]], dtype=np.float32)[None]
    p = inputs.Problem("tiny", pts, np.array([0, 0, 1, 1, 4], dtype=np.int32), inputs.BOX_NONE, None, 2.0, 7)
    got, _ = gpu_hist(p)
    assert_same(got, oracle_hist(p), "empty species + NaN")
    one = inputs.Problem("one", pts[:, :1], np.array([0, 1], dtype=np.int32), inputs.BOX_NONE, None, 2.0, 7)
    got, _ = gpu_hist(one)
    assert int(got.sum()) == 0


def test_q3_clamp_and_rmax_cut():
    # distances at and just below r_max; scale rounding can push d*scale to n_bins (Q3)
    r = np.float32(0.7)
    xs = [np.nextafter(r, np.float32(0)), r, np.nextafter(r, np.float32(1)), np.float32(0.35), np.float32(0.0)]
    pts = np.zeros((1, 1 + len(xs), 3), dtype=np.float32)
    pts[0, 1:, 0] = xs
    for n_bins in (1, 3, 7, 1000, 4097):
        p = inputs.Problem(f"q3_{n_bins}", pts, np.array([0, 1, 1 + len(xs)], dtype=np.int32), inputs.BOX_NONE, None,
                           float(r), n_bins)
        got, _ = gpu_hist(p)
        assert_same(got, oracle_hist(p), p.name)


def test_sqrt_selftest_sample():
    _need_gpu()
    # full range is bench.py --selftest; here 2^26 patterns around 1.0 and the low end of the range
    assert cdh.cdh_selftest_sqrt(0x3F000000, 0x3F000000 + (1 << 26)) == 0
    assert cdh.cdh_selftest_sqrt(0x0D800000, 0x0D800000 + (1 << 24)) == 0


def test_argument_errors_leave_out_untouched():
    _need_gpu()
    p = inputs.reduced_config(1)
    dev = torch.device("cuda", 0)
    coords = torch.from_numpy(p.coords).to(dev)
    out = torch.full((1, p.n_bins), -7, dtype=torch.int64, device=dev)
    c_ptr, o_ptr = int(coords.data_ptr()), int(out.data_ptr())     # raw pointers: the C library's own checks are under test
    with cdh.Context(0) as ctx:
        for kw in (dict(n_bins=0), dict(r_max=-1.0), dict(r_max=float("nan")), dict(n_bins=(1 << 22) + 1)):
            args = dict(r_max=p.r_max, n_bins=p.n_bins)
            args.update(kw)
            with pytest.raises(cdh.CdhError) as e:
                ctx.cdh_histograms(c_ptr, 1, p.species_offsets, p.box_type, None, args["r_max"], args["n_bins"], o_ptr)
            assert e.value.code == cdh.binding.ERR_INVALID_ARG
        with pytest.raises(cdh.CdhError) as e:
            ctx.cdh_histograms(c_ptr, 1, p.species_offsets, p.box_type, None, p.r_max, p.n_bins, o_ptr, precision=7)
        assert e.value.code == cdh.binding.ERR_INVALID_ARG
        with pytest.raises(cdh.CdhError):       # singular box
            ctx.cdh_histograms(c_ptr, 1, p.species_offsets, inputs.BOX_TRICLINIC, np.zeros((1, 9)), 1.0, 10, o_ptr)
        with pytest.raises(cdh.CdhError):       # off-diagonal with ORTHO
            ctx.cdh_histograms(c_ptr, 1, p.species_offsets, inputs.BOX_ORTHO,
                               np.array([[1.0, 0.1, 0, 0, 1, 0, 0, 0, 1]]), 1.0, 10, o_ptr)
        with pytest.raises(ValueError):         # the binding refuses a tensor the call would overrun
            ctx.cdh_histograms(coords, 1, p.species_offsets, p.box_type, None, p.r_max, p.n_bins + 1, out)
        with pytest.raises(ValueError):         # ... and one of the wrong element type
            ctx.cdh_histograms(coords.double(), 1, p.species_offsets, p.box_type, None, p.r_max, p.n_bins, out)
    torch.cuda.synchronize()
    assert bool((out == -7).all())


def test_context_reuse_growing_and_shrinking_problems():
    _need_gpu()
    with cdh.Context(0) as ctx:
        for k in (1, 3, 2, 1, 5, 4):
            p = inputs.reduced_config(k)
            out = cdh.histograms_device(ctx, p)
            torch.cuda.synchronize()
            assert_same(out.cpu().numpy().view(np.uint64), oracle_hist(p), f"reuse {p.name}")


def test_user_stream_and_back_to_back_calls():
    _need_gpu()
    p = inputs.reduced_config(2)
    s = torch.cuda.Stream()
    with cdh.Context(0) as ctx:
        with torch.cuda.stream(s):
            outs = [cdh.histograms_device(ctx, p, stream=s) for _ in range(3)]
        s.synchronize()
        for o in outs:
            assert_same(o.cpu().numpy().view(np.uint64), oracle_hist(p), "stream")


def test_many_species_and_ragged_sizes():
    # 12 species of very different sizes (some empty, some of one particle): 78 histograms in one call
    counts = (0, 1, 2, 3, 511, 512, 513, 1023, 1025, 0, 2047, 4097)
    p = inputs.uniform_problem(21, counts, inputs.BOX_ORTHO, 777, 2.0, box=np.diag([4.0, 5.0, 6.0]))
    got, info = gpu_hist(p)
    assert got.shape == (78, 777)
    assert_same(got, oracle_hist(p), f"12 species {info}")


def test_per_frame_triclinic_boxes_and_frame_sum():
    g = np.random.Generator(np.random.PCG64(33))
    f, n = 4, 1500
    boxes = np.stack([np.array([[7.0 + k, 0, 0], [1.0, 6.5, 0], [0.5 * k, -1.0, 8.0 - k]]) for k in range(f)])
    coords = np.stack([(g.random((n, 3)) @ boxes[k]).astype(np.float32) for k in range(f)])
    p = inputs.Problem("tri_per_frame", coords, np.array([0, 400, n], dtype=np.int32), inputs.BOX_TRICLINIC,
                       boxes.reshape(f, 9), 2.4, 999)
    got, _ = gpu_hist(p)
    assert_same(got, oracle_hist(p), p.name)
    # Eq. 2: the call sums the frames
    parts = sum(gpu_hist(inputs.Problem(f"fr{k}", coords[k:k + 1], p.species_offsets, p.box_type, p.box[k:k + 1], p.r_max,
                                        p.n_bins))[0] for k in range(f))
    assert_same(got, parts, "sum over frames")


def test_maximum_bin_count_and_single_bin():
    p = inputs.uniform_problem(5, (3000,), inputs.BOX_NONE, 1 << 22, math.sqrt(3.0))      # n_bins = 2^22, the API maximum
    got, info = gpu_hist(p)
    assert info["global_hist"]
    assert_same(got, oracle_hist(p), f"2^22 bins {info}")
    q = inputs.uniform_problem(6, (3000, 10), inputs.BOX_NONE, 1, 0.5)
    got, _ = gpu_hist(q)
    assert_same(got, oracle_hist(q), "one bin")


def test_tiny_rmax_keeps_nothing_and_huge_rmax_keeps_everything():
    p = inputs.uniform_problem(8, (2500,), inputs.BOX_NONE, 100, 1e-6)
    got, _ = gpu_hist(p)
    assert_same(got, oracle_hist(p), "r_max = 1e-6")
    q = inputs.uniform_problem(8, (2500,), inputs.BOX_NONE, 100, 1e6)
    got, _ = gpu_hist(q)
    assert int(got.sum()) == 2500 * 2499 // 2 and int(got[0, 0]) == int(got.sum())
    assert_same(got, oracle_hist(q), "r_max = 1e6")


def test_periodic_boxes_far_from_the_origin():
    # compact systems translated far away: fp32 coordinates get coarse (ulp(x) up to a fraction of the bin width) and the
    # measured fractional range loses accuracy; the launch plan must leave the fused / pruned paths early enough
    base = inputs.uniform_problem(41, (900, 1100), inputs.BOX_ORTHO, 2000, 3.0, box=np.diag([6.0, 7.3, 9.1]))
    tri_box = np.array([[7.0, 0.0, 0.0], [1.0, 6.5, 0.0], [0.5, -1.0, 8.0]])
    tri = inputs.uniform_problem(42, (800, 1000), inputs.BOX_TRICLINIC, 2000, 3.0, box=tri_box)
    for shift in (1.0e2, 3.0e3, 1.0e4, 3.0e5, 1.0e7):
        for p in (base, tri):
            q = inputs.Problem(f"far{shift}", (p.coords.astype(np.float64) + shift).astype(np.float32), p.species_offsets,
                               p.box_type, p.box, p.r_max, p.n_bins)
            got, info = gpu_hist(q)
            assert_same(got, oracle_hist(q), f"box_type {p.box_type} shifted by {shift} {info}")


def test_accumulate_flag_sums_chunks_of_a_trajectory():
    _need_gpu()
    p = inputs.reduced_config(4)                     # 3 frames
    dev = torch.device("cuda", 0)
    out = torch.zeros((p.n_hist, p.n_bins), dtype=torch.int64, device=dev)
    with cdh.Context(0, cdh.FLAG_ACCUMULATE) as ctx:
        for f in range(p.n_frames):                  # one frame per call, all into the same result
            c = torch.from_numpy(np.ascontiguousarray(p.coords[f:f + 1])).to(dev)
            ctx.cdh_histograms(c, 1, p.species_offsets, p.box_type, p.box, p.r_max, p.n_bins, out)
        torch.cuda.synchronize()
    assert_same(out.cpu().numpy().view(np.uint64), oracle_hist(p), "accumulated over three calls")


@pytest.mark.parametrize("spread", [1.6, 3.0, 12.0, 40.0, 90.0])
def test_triclinic_unwrapped_coordinates_wide_tier(spread):
    # coordinates spanning several cells (unwrapped trajectories): range 1.49 .. 64 takes the wide fast path (pinned B*n
    # chain, pruning margin grown with the range), beyond 64 the plain kernel; all must equal the oracle
    box = np.array([[9.0, 0.0, 0.0], [1.5, 8.0, 0.0], [-2.0, 2.5, 7.0]])
    p = inputs.uniform_problem(88, (1500, 2300), inputs.BOX_TRICLINIC, 4000, 3.4, box=box, spread=spread)
    got, info = gpu_hist(p)
    assert_same(got, oracle_hist(p), f"triclinic spread {spread} {info}")
    q = inputs.config3(counts=(1700, 2100), n_bins=5000)
    g = np.random.Generator(np.random.PCG64(int(spread * 10)))
    shifts = g.integers(-int(spread), int(spread) + 1, size=(q.n_total, 3)).astype(np.float64) @ q.box.reshape(3, 3)
    q = inputs.Problem("cfg3_unwrapped", (q.coords.astype(np.float64) + shifts[None]).astype(np.float32), q.species_offsets,
                       q.box_type, q.box, q.r_max, q.n_bins)
    got, info = gpu_hist(q)
    assert_same(got, oracle_hist(q), f"config 3 shifted by up to {int(spread)} cells {info}")


@pytest.mark.parametrize("r_max", [7.0, 12.0])
def test_triclinic_pairs_on_the_half_cell_switch_points(r_max):
    # fractional separations within a few ulps of 1/2 on each axis of a dyadic cell (all coordinates exact): exactly where
    # Eq. 5 can pick the far image and where the pruning test has to hand the pair to the 27-shift search
    box = np.array([[16.0, 0.0, 0.0], [0.0, 16.0, 0.0], [8.0, 8.0, 16.0]])        # heights 14.3, 14.3, 16
    rows = [np.zeros(3)]
    for ax in range(3):
        for k in range(-8, 9):
            for other in (0.0, 0.125, 0.4375):
                s = np.array([other, other / 2, other / 4])
                s[ax] = 0.5 + k * 2.0 ** -23
                rows.append(s @ box)
                rows.append(-(s @ box))
    pts = np.array(rows, dtype=np.float32)[None]
    p = inputs.Problem("tri_half", pts, np.array([0, 1, len(rows)], dtype=np.int32), inputs.BOX_TRICLINIC, box.reshape(1, 9),
                       r_max, 1 << 16)
    want = oracle_hist(p)
    for flags in (0, cdh.FLAG_NO_PRUNE, cdh.FLAG_SIMPLE_KERNEL):
        got, info = gpu_hist(p, flags)
        assert_same(got, want, f"flags {flags:#x} {info}")


def test_triclinic_rare_pairs_in_the_large_problem_kernel():
    """The large-problem kernel of the TRI_UPPER_B01 form bins a group first and MOVES the rare pair the neighbour search
    corrects afterwards (csrc/cdh_math32.cuh, CDH_TRI_FIXUP).  Half of the points sit within a few ulps of the half-cell
    lattice of a dyadic cell, so that a large share of the pairs -- in diagonal (masked), full and ragged stages -- has a
    fractional separation at the switch point 1/2; big enough for the large-problem kernel (not the SKIP one)."""
    box = np.array([[16.0, 0.0, 0.0], [0.0, 16.0, 0.0], [8.0, 8.0, 16.0]])        # heights 14.3, 14.3, 16; B upper triangular, B01 = 0
    g = np.random.Generator(np.random.PCG64(424242))
    n, f = 26_000, 3
    frac = g.random((f, n, 3))
    lattice = g.integers(0, 2, size=(f, n // 2, 3)) * 0.5 + g.integers(-8, 9, size=(f, n // 2, 3)) * 2.0 ** -23
    frac[:, : n // 2] = lattice
    coords = (frac @ box).astype(np.float32)
    p = inputs.Problem("tri_rare_large", coords, np.array([0, n], dtype=np.int32), inputs.BOX_TRICLINIC, box.reshape(1, 9), 7.0, 20_000)
    got, info = gpu_hist(p)
    assert not info["skip"] and info["form"] == 2 and info["threads"] == 256, info
    assert_same(got, oracle_hist(p), f"rare pairs, large-problem kernel: {info}")
    assert_same(gpu_hist(p, cdh.FLAG_NO_PRUNE)[0], got, "27-shift search for every pair")


@pytest.mark.parametrize("box_type", [inputs.BOX_NONE, inputs.BOX_ORTHO, inputs.BOX_TRICLINIC])
def test_small_species_take_the_skip_variants(box_type):
    # species of a few i-tiles each: the launch plan takes the kernels whose warps skip the j-groups below the diagonal
    # and the padding-only warps of a ragged i-tile (info["skip"]); same integers as the oracle, and as the plain kernel
    box = {inputs.BOX_NONE: None, inputs.BOX_ORTHO: np.diag([5.0, 6.0, 7.0]),
           inputs.BOX_TRICLINIC: np.array([[6.0, 0.0, 0.0], [1.0, 5.5, 0.0], [-0.5, 1.5, 5.0]])}[box_type]
    for counts in ((130,), (1024,), (1025, 2047), (300, 1100, 2100), (4096, 3), (2500, 2500)):
        p = inputs.uniform_problem(sum(counts), counts, box_type, 1500, 2.2, box=box, n_frames=2)
        got, info = gpu_hist(p)
        assert info["skip"], f"{counts}: {info}"
        assert_same(got, oracle_hist(p), f"skip variant, box_type {box_type}, species {counts}")
        # info[7]: the pair slots the 1024-particle i-tiles are scheduled to walk: at least the pairs, at most full tiles
        tiles = [-(-c // 1024) for c in counts]
        full = p.n_frames * sum(1024 * t * sum(c + 3 for c in counts[k:]) for k, t in enumerate(tiles))
        assert p.evaluated_pairs <= info["padded_pairs"] <= full, (p.evaluated_pairs, info["padded_pairs"], full)
    big = inputs.uniform_problem(7, (16000, 24000), box_type, 1500, 2.2, box=box)
    got, info = gpu_hist(big)
    assert not info["skip"], info
    assert_same(got, oracle_hist(big), f"large species, box_type {box_type}")


def test_no_box_clean_form_and_everything_that_must_switch_it_off():
    """No box: when every distance of the call is provably below r_max and no coordinate is NaN the kernel leaves out the
    threshold compare (KIND_CLEAN, cdh_sched.cuh).  The device decides from the coordinate extent the repack kernel
    measures; each of these inputs must give the oracle's integers whichever form runs."""
    g = np.random.Generator(np.random.PCG64(77))
    n = 9000                                                    # several i-tiles and a ragged tail
    base = g.random((n, 3)).astype(np.float32)
    cases = {"clean": (base, math.sqrt(3.0))}
    x = base.copy(); x[4321] = x[17]; x[8999] = x[17]           # coincident particles: d2 = 0 inside the clean form
    cases["coincident"] = (x, math.sqrt(3.0))
    x = base.copy(); x[5000, 1] = np.nan                        # a NaN coordinate: its pairs are dropped, the form is general
    cases["nan"] = (x, math.sqrt(3.0))
    x = base.copy(); x[123, 0] = np.inf
    cases["inf"] = (x, math.sqrt(3.0))
    cases["r_max inside the extent"] = (base, 1.2)              # some pairs are beyond r_max
    x = base.copy(); x[0] = (0.0, 0.0, 0.0); x[1] = (1.0, 1.0, 1.0)
    cases["corner to corner"] = (x, math.sqrt(3.0))             # d = fl(sqrt(3)) is NOT below (float)r_max: dropped
    for name, (pts, r_max) in cases.items():
        for offsets in ([0, n], [0, 4097, n]):
            p = inputs.Problem(name, np.ascontiguousarray(pts[None]), np.array(offsets, dtype=np.int32), inputs.BOX_NONE, None,
                               r_max, 3000)
            got, info = gpu_hist(p)
            assert_same(got, oracle_hist(p), f"{name}, offsets {offsets}: {info}")
    p = inputs.Problem("clean", np.ascontiguousarray(base[None]), np.array([0, n], dtype=np.int32), inputs.BOX_NONE, None,
                       math.sqrt(3.0), 3000)
    assert int(gpu_hist(p)[0].sum()) == n * (n - 1) // 2


def test_hybrid_window_with_frames_accumulate_and_per_frame_boxes():
    """MODE_HYBRID next to the other features: several frames with their own boxes, CDH_FLAG_ACCUMULATE (the result is
    not zeroed), and a bin count one above what the shared memory holds."""
    _need_gpu()
    f, counts = 3, (1500, 700)
    g = np.random.Generator(np.random.PCG64(5))
    boxes = np.stack([np.diag([4.0 + 0.1 * k, 4.5, 5.0 - 0.1 * k]) for k in range(f)]).reshape(f, 9)
    coords = (g.random((f, sum(counts), 3)) * 5.0).astype(np.float32)
    for n_bins in (56_403, 90_000):
        p = inputs.Problem("hyb_frames", coords, np.array([0, 1500, 2200], dtype=np.int32), inputs.BOX_ORTHO, boxes, 2.0, n_bins)
        want = oracle_hist(p)
        got, info = gpu_hist(p)
        assert info["hybrid"], info
        assert_same(got, want, f"{n_bins} bins, per-frame boxes: {info}")
        with cdh.Context(0, cdh.FLAG_ACCUMULATE) as ctx:
            dev = torch.device("cuda", 0)
            out = torch.zeros((p.n_hist, n_bins), dtype=torch.int64, device=dev)
            for k in range(f):                                   # frame by frame into the same result
                c = torch.from_numpy(np.ascontiguousarray(coords[k:k + 1])).to(dev)
                ctx.cdh_histograms(c, 1, p.species_offsets, p.box_type, boxes[k:k + 1], p.r_max, n_bins, out)
            torch.cuda.synchronize()
            assert_same(out.cpu().numpy().view(np.uint64), want, f"{n_bins} bins, accumulated frame by frame")


def test_orthorhombic_full_range_private_histogram():
    """Orthorhombic box: when no dropped pair can share a bin slot with a kept one (the host checks bin(thr2) >= n_bins and
    that no kept pair rounds up into slot n_bins) the private histogram gets a slot for every reachable distance and stages
    without padding skip the threshold compare (info["full_range"]).  Taken or not, the integers are the oracle's."""
    _need_gpu()
    cases = [
        # (box diag, r_max, n_bins, counts): dyadic scale -> the form is taken
        ((10.0, 10.0, 10.0), 5.0, 10000, (3000, 5200)),
        ((8.0, 9.0, 7.5), 3.75, 3000, (4100, 1000)),           # anisotropic box, r_max = half the shortest edge
        ((6.0, 6.0, 6.0), 1.0, 512, (5000,)),                  # few pairs kept: most updates land beyond n_bins
        ((6.0, 6.0, 6.0), 5.0, 2048, (5000,)),                 # r_max beyond half the box: nearly every pair is kept
        # scales that are not exact in fp32: taken or not depending on the rounding, exact either way
        ((7.3, 8.1, 9.7), 3.65, 7777, (2500, 2600)),
        ((5.123, 5.123, 5.123), 2.5615, 9999, (4097,)),
        ((11.0, 11.0, 11.0), 5.5, 30011, (3000,)),             # the full-range histogram needs the one-CTA-per-SM shape
    ]
    taken = 0
    for k, (diag, r_max, n_bins, counts) in enumerate(cases):
        p = inputs.uniform_problem(500 + k, counts, inputs.BOX_ORTHO, n_bins, r_max, box=np.diag(diag), n_frames=2, spread=1.2)
        got, info = gpu_hist(p)
        taken += info["full_range"]
        assert_same(got, oracle_hist(p), f"case {k} {diag} r_max {r_max} bins {n_bins}: {info}")
        plain, info2 = gpu_hist(p, cdh.FLAG_NO_PRUNE)           # the pinned 5-operation form, no full-range histogram
        assert not info2["full_range"]
        assert_same(plain, got, f"case {k}: plain form")
    assert taken >= 4
    # a NaN coordinate switches the form off on the device (its pairs are dropped by the threshold compare)
    p = inputs.uniform_problem(77, (3000, 1200), inputs.BOX_ORTHO, 4096, 4.0, box=np.diag((8.0, 8.0, 8.0)))
    p.coords[0, 1234, 2] = np.nan
    got, info = gpu_hist(p)
    assert info["full_range"]
    assert_same(got, oracle_hist(p), "NaN coordinate with the full-range histogram")
