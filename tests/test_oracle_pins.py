"""Pins for the CPU oracle (oracle/cdh_oracle.c): everything here is fixed by the paper or by
mathematics, not by the oracle itself and never by the CUDA path.

P1 total counts N(N-1)/2, N1*N2          P5 125-image brute force, dyadic boxes
P2-P4 hand-computed 4-particle examples (tests/golden)      P6 permutation / species-swap symmetry
P7 reductions to numpy / the ideal-gas shell count          P8 one bin > 2^32
P10 fp32 vs fp64 oracle: adjacent-bin moves only, bounded L1
"""
import itertools
import json
import math
import os

import numpy as np
import pytest

import oracle
from paper_1808_01478_b200 import inputs
from paper_1808_01478_b200.inputs import BOX_NONE, BOX_ORTHO, BOX_TRICLINIC


# ------------------------------------------------------------------ helpers (independent of the oracle)
def load_golden(golden_dir, name):
    out = {}
    with open(os.path.join(golden_dir, name)) as fh:
        for line in fh:
            line = line.split("#", 1)[0].strip()
            if not line:
                continue
            key, val = line.split(":", 1)
            out[key.strip()] = json.loads(val)
    return out


def sparse(hist_row):
    return {str(int(b)): int(hist_row[b]) for b in np.flatnonzero(hist_row)}


def brute_min_image_d2(xi, xj, box_rows, shell=2):
    """float64 minimum over (2*shell+1)^3 lattice translates of |xj - xi + i a + j b + k c|^2."""
    d = np.asarray(xj, dtype=np.float64) - np.asarray(xi, dtype=np.float64)
    rng = range(-shell, shell + 1)
    shifts = np.array([i * box_rows[0] + j * box_rows[1] + k * box_rows[2]
                       for i, j, k in itertools.product(rng, rng, rng)])
    c = d[None, :] + shifts
    return float((c * c).sum(axis=1).min())


def brute_hist(points, offsets, box_rows, r_max, n_bins, shell=2):
    """Histograms by the plain definition in float64 (dyadic inputs: exact before the sqrt): every pair,
    minimum over (2*shell+1)^3 lattice translates, floor(d * n_bins / r_max), d >= r_max dropped."""
    pts = np.asarray(points, dtype=np.float64)
    ns = len(offsets) - 1
    scale = n_bins / r_max
    rng = range(-shell, shell + 1)
    shifts = np.zeros((1, 3)) if box_rows is None else np.array(
        [i * box_rows[0] + j * box_rows[1] + k * box_rows[2] for i, j, k in itertools.product(rng, rng, rng)])
    hists = []
    for p in range(ns):
        for q in range(p, ns):
            if p == q:
                i, j = np.triu_indices(offsets[p + 1] - offsets[p], k=1)
                i, j = i + offsets[p], j + offsets[p]
            else:
                i, j = np.meshgrid(np.arange(offsets[p], offsets[p + 1]), np.arange(offsets[q], offsets[q + 1]),
                                   indexing="ij")
                i, j = i.ravel(), j.ravel()
            c = (pts[j] - pts[i])[:, None, :] + shifts[None, :, :]
            d = np.sqrt((c * c).sum(axis=2).min(axis=1))
            d = d[d < r_max]
            bins = np.minimum(np.floor(d * scale).astype(np.int64), n_bins - 1)
            hists.append(np.bincount(bins, minlength=n_bins).astype(np.uint64))
    return np.array(hists)


PRECS = ["f32", "f64"]


# ------------------------------------------------------------------ P1 total counts
@pytest.mark.parametrize("prec", PRECS)
def test_p1_total_count_single_species(prec):
    p = inputs.config1()
    h = oracle.problem_histograms(p, prec)
    assert h.shape == (1, 1000)
    assert int(h.sum()) == 2000 * 1999 // 2       # N(N-1)/2


@pytest.mark.parametrize("prec", PRECS)
def test_p1_total_count_multi_species(prec):
    counts = (37, 1, 250, 0, 113)
    p = inputs.uniform_problem(11, counts, BOX_NONE, n_bins=64, r_max=2.0)
    h = oracle.problem_histograms(p, prec)
    k = 0
    for a in range(len(counts)):
        for b in range(a, len(counts)):
            want = counts[a] * (counts[a] - 1) // 2 if a == b else counts[a] * counts[b]
            assert int(h[k].sum()) == want, (a, b)
            k += 1
    assert k == h.shape[0] == 15


def test_p1_clustered_config_total():
    p = inputs.reduced_config(5)
    h = oracle.problem_histograms(p)
    n = p.n_total
    assert int(h.sum()) == n * (n - 1) // 2


# ------------------------------------------------------------------ P2-P4 hand examples
def _run_points(points, offsets, box_type, box, r_max, n_bins, prec):
    pts = np.asarray(points, dtype=np.float32)
    return oracle.histograms(pts, offsets, box_type, None if box is None else np.asarray(box, float),
                             r_max, n_bins, precision=prec)


@pytest.mark.parametrize("prec", PRECS)
def test_p2_nonperiodic_hand_example(golden_dir, prec):
    g = load_golden(golden_dir, "p2_nonperiodic_4particles.txt")
    pts = g["points"]
    for (i, j) in itertools.combinations(range(4), 2):
        assert oracle.pair_d2(pts[i], pts[j], BOX_NONE, None, prec) == g["d2"][f"{i}{j}"]
    for case in ("case_a", "case_b"):
        c = g[case]
        h = _run_points(pts, [0, 4], BOX_NONE, None, c["r_max"], c["n_bins"], prec)
        assert sparse(h[0]) == c["hist"], case
    c = g["case_c"]
    h = _run_points(pts, c["species_offsets"], BOX_NONE, None, c["r_max"], c["n_bins"], prec)
    assert [sparse(r) for r in h] == c["hist"]


@pytest.mark.parametrize("prec", PRECS)
def test_p3_orthorhombic_hand_example(golden_dir, prec):
    g = load_golden(golden_dir, "p3_orthorhombic_4particles.txt")
    pts, box = g["points"], np.array(g["box"], float)
    for (i, j) in itertools.combinations(range(4), 2):
        assert oracle.pair_d2(pts[i], pts[j], BOX_ORTHO, box, prec) == g["d2"][f"{i}{j}"]
        assert brute_min_image_d2(pts[i], pts[j], box) == g["d2"][f"{i}{j}"]
    c = g["case_a"]
    h = _run_points(pts, [0, 4], BOX_ORTHO, box, c["r_max"], c["n_bins"], prec)
    assert sparse(h[0]) == c["hist"]
    t = g["tie"]
    assert oracle.pair_d2(t["points"][0], t["points"][1], BOX_ORTHO, box, prec) == t["d2"]
    assert oracle.pair_d2(t["points"][1], t["points"][0], BOX_ORTHO, box, prec) == t["d2"]


@pytest.mark.parametrize("prec", PRECS)
def test_p4_triclinic_needs_neighbour_shift(golden_dir, prec):
    g = load_golden(golden_dir, "p4_triclinic_4particles.txt")
    pts, box = g["points"], np.array(g["box"], float)
    for (i, j) in itertools.combinations(range(4), 2):
        want = g["d2"][f"{i}{j}"]
        assert brute_min_image_d2(pts[i], pts[j], box) == want          # the fixture is right
        assert oracle.pair_d2(pts[i], pts[j], BOX_TRICLINIC, box, prec) == want
        assert oracle.pair_d2(pts[j], pts[i], BOX_TRICLINIC, box, prec) == want
    # Eq. 5 alone really is insufficient here: columns of b are the box vectors (Q6).
    b = box.T
    for key, want in g["eq5_only_d2"].items():
        i, j = int(key[0]), int(key[1])
        dx = np.array(pts[j], float) - np.array(pts[i], float)
        e = dx - b @ np.rint(np.linalg.solve(b, dx))
        assert float(e @ e) == want
    c = g["case_a"]
    h = _run_points(pts, [0, 4], BOX_TRICLINIC, box, c["r_max"], c["n_bins"], prec)
    assert sparse(h[0]) == c["hist"]


def test_row_vs_column_convention_matters(golden_dir):
    """Passing the transposed box must change the answer (guards Q6 against a silent transpose)."""
    g = load_golden(golden_dir, "p4_triclinic_4particles.txt")
    pts, box = g["points"], np.array(g["box"], float)
    c = g["case_a"]
    h = _run_points(pts, [0, 4], BOX_TRICLINIC, box.T.copy(), c["r_max"], c["n_bins"], "f32")
    assert sparse(h[0]) != c["hist"]


# ------------------------------------------------------------------ P5 brute force on tiny dyadic periodic boxes
DYADIC_BOXES = {
    "ortho": (BOX_ORTHO, np.diag([8.0, 16.0, 4.0])),
    "tric_a": (BOX_TRICLINIC, np.array([[16.0, 0, 0], [0, 16.0, 0], [8.0, 8.0, 16.0]])),
    "tric_b": (BOX_TRICLINIC, np.array([[8.0, 0, 0], [4.0, 8.0, 0], [4.0, 4.0, 8.0]])),
    "tric_full": (BOX_TRICLINIC, np.array([[8.0, 0, 2.0], [2.0, 8.0, 0], [0, 2.0, 8.0]])),
}


def _heights(box_rows):
    a, b, c = box_rows
    vol = abs(np.dot(a, np.cross(b, c)))
    return [vol / np.linalg.norm(np.cross(b, c)), vol / np.linalg.norm(np.cross(c, a)),
            vol / np.linalg.norm(np.cross(a, b))]


@pytest.mark.parametrize("name", sorted(DYADIC_BOXES))
@pytest.mark.parametrize("regime", ["half_min_height", "beyond"])
@pytest.mark.parametrize("prec", PRECS)
def test_p5_bruteforce_periodic(name, regime, prec):
    box_type, box = DYADIC_BOXES[name]
    if name == "tric_full":
        # b^-1 of this cell is not dyadic: only the fp64 oracle is compared exactly (fp32 differs by rounding).
        if prec == "f32":
            pytest.skip("non-dyadic inverse: exact comparison only in fp64")
    g = np.random.Generator(np.random.PCG64(5000 + len(name)))
    n = 60
    # dyadic coordinates (multiples of 1/64), deliberately up to 1.5 cells outside the box (|dx| < 4 cells)
    frac = g.integers(-96, 160, size=(n, 3)) / 64.0
    pts = frac @ box if box_type == BOX_TRICLINIC else frac * np.diag(box)
    pts = np.round(pts * 64) / 64
    assert np.array_equal(pts.astype(np.float32).astype(np.float64), pts)
    hmin = min(_heights(box))
    # r_max a multiple of 1/4 and scale = n_bins / r_max = 16 exactly: with d^2 a multiple of 1/4096 a
    # distance is either exactly on a bin edge (exact sqrt) or > 1e-5 away from one, so fp32 and fp64
    # must both reproduce the brute-force bins exactly.
    r_max = math.floor((hmin / 2 if regime == "half_min_height" else hmin * 0.9375) * 4) / 4
    n_bins = int(r_max * 16)
    offsets = [0, 25, 60]
    want = brute_hist(pts, offsets, box, r_max, n_bins, shell=4)
    got = oracle.histograms(pts.astype(np.float32), offsets, box_type, box, r_max, n_bins, precision=prec)
    assert np.array_equal(got, want)
    assert want.sum() > 0


# ------------------------------------------------------------------ P6 symmetry
@pytest.mark.parametrize("k", [2, 3, 5])
def test_p6_permutation_and_species_swap(k):
    p = inputs.reduced_config(k)
    if k == 5:
        p = inputs.config5(n=3001, n_bins=5000, n_clusters=10)
    if k == 2:
        p = inputs.config2(counts=(300, 900, 1500), n_bins=2000)
    if k == 3:
        p = inputs.config3(counts=(700, 1100), n_bins=4000)
    base = oracle.problem_histograms(p)
    g = np.random.Generator(np.random.PCG64(99))
    c = p.coords.copy()
    off = p.species_offsets
    for s in range(p.n_species):
        perm = g.permutation(off[s + 1] - off[s]) + off[s]
        c[:, off[s]:off[s + 1]] = p.coords[:, perm]
    assert np.array_equal(oracle.histograms(c, off, p.box_type, p.box, p.r_max, p.n_bins), base)
    if p.n_species > 1:
        # reverse the species order: histogram rows are permuted accordingly
        order = list(range(p.n_species))[::-1]
        blocks = [p.coords[:, off[s]:off[s + 1]] for s in order]
        counts = [b.shape[1] for b in blocks]
        c2 = np.concatenate(blocks, axis=1)
        off2 = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
        h2 = oracle.histograms(c2, off2, p.box_type, p.box, p.r_max, p.n_bins)
        ns = p.n_species
        for a in range(ns):
            for b in range(a, ns):
                src = inputs.hist_index(order[a], order[b], ns)
                row = a * ns - a * (a - 1) // 2 + (b - a)
                assert np.array_equal(h2[row], base[src]), (a, b)


def test_p6_lattice_shift_invariance_dyadic():
    """Shifting particles by integer lattice vectors changes nothing when all products are exact."""
    box = DYADIC_BOXES["tric_b"][1]
    g = np.random.Generator(np.random.PCG64(7))
    pts = (g.integers(0, 64, size=(80, 3)) / 64.0) @ box
    shifts = g.integers(-2, 3, size=(80, 3)).astype(np.float64) @ box
    a = oracle.histograms(pts.astype(np.float32), [0, 80], BOX_TRICLINIC, box, 3.5, 50)
    b = oracle.histograms((pts + shifts).astype(np.float32), [0, 80], BOX_TRICLINIC, box, 3.5, 50)
    assert np.array_equal(a, b) and a.sum() > 0


# ------------------------------------------------------------------ P7 reductions to library routines / closed forms
def test_p7_nonperiodic_fp64_equals_numpy():
    from scipy.spatial.distance import cdist, pdist
    p = inputs.uniform_problem(21, (1500, 800), BOX_NONE, n_bins=777, r_max=1.1)
    x = p.coords[0].astype(np.float64)
    a, b = x[:1500], x[1500:]
    scale = 777 / 1.1

    def binned(d):
        d = d[d < 1.1]
        return np.bincount(np.minimum(np.floor(d * scale).astype(np.int64), 776), minlength=777)

    got = oracle.problem_histograms(p, "f64")
    # scipy's euclidean kernels sum squares in a different order; allow a handful of edge pairs to move
    # to the neighbouring bin, nothing else.
    for row, d in zip(got, (pdist(a), cdist(a, b).ravel(), pdist(b))):
        want = binned(d)
        assert int(row.sum()) == int(want.sum()) or abs(int(row.sum()) - int(want.sum())) <= 2
        assert np.abs(np.cumsum(row.astype(np.int64)) - np.cumsum(want)).max() <= 3


def test_p7_nonperiodic_fp64_exact_small():
    """Same reduction written out with numpy in the oracle's own summation order: exact."""
    p = inputs.uniform_problem(22, (400,), BOX_NONE, n_bins=100, r_max=0.9)
    x = p.coords[0].astype(np.float64)
    i, j = np.triu_indices(400, k=1)
    d = x[j] - x[i]
    d2 = (d[:, 0] * d[:, 0] + d[:, 1] * d[:, 1]) + d[:, 2] * d[:, 2]
    r = np.sqrt(d2)
    keep = r < 0.9
    want = np.bincount(np.minimum(np.floor(r[keep] * (100 / 0.9)).astype(np.int64), 99), minlength=100)
    assert np.array_equal(oracle.problem_histograms(p, "f64")[0], want.astype(np.uint64))


@pytest.mark.parametrize("k,frac", [(2, math.pi / 6), (3, math.pi / 12), (4, math.pi / 6)])
def test_p7_ideal_gas_shell_counts(k, frac):
    """Uniform points in a periodic box, r_max <= half the minimum height: the expected count of bin
    kappa is N_pairs * (4 pi / 3)(r_{k+1}^3 - r_k^3) / V (Eq. 1 with g(r) = 1)."""
    p = inputs.reduced_config(k)
    h = oracle.problem_histograms(p).astype(np.float64)
    box = p.box.reshape(-1, 3, 3)[0]
    vol = abs(np.linalg.det(box))
    edges = np.arange(p.n_bins + 1) * (p.r_max / p.n_bins)
    shell = 4 * math.pi / 3 * (edges[1:] ** 3 - edges[:-1] ** 3) / vol
    for row, npairs in zip(h, p.pairs_per_hist()):
        npairs *= p.n_frames
        kept = row.sum() / npairs
        assert abs(kept - frac) < 4 * math.sqrt(frac / npairs) + 2e-3, (kept, frac)
        # coarse chi^2 over 50 groups of bins
        gexp = (shell * npairs).reshape(50, -1).sum(axis=1)
        gobs = row.reshape(50, -1).sum(axis=1)
        big = gexp > 50
        chi2 = (((gobs - gexp) ** 2) / gexp)[big].sum()
        dof = int(big.sum())
        if k != 4:                      # cfg 4 frames are correlated (shared base): kept-fraction check only
            assert chi2 < dof + 6 * math.sqrt(2 * dof), (chi2, dof)


# ------------------------------------------------------------------ P8 a single bin beyond 2^32
@pytest.mark.slow
def test_p8_bin_exceeds_uint32():
    n = 100_000
    pts = np.full((n, 3), 0.25, dtype=np.float32)
    h = oracle.histograms(pts, [0, n], BOX_NONE, None, 1.0, 16)
    assert int(h[0, 0]) == 4_999_950_000 and int(h[0, 1:].sum()) == 0


# ------------------------------------------------------------------ P10 fp32 vs fp64
@pytest.mark.parametrize("k", [1, 2, 3])
def test_p10_fp32_vs_fp64_adjacent_bins_only(k):
    p = inputs.reduced_config(k)
    h32 = oracle.problem_histograms(p, "f32").astype(np.int64)
    h64 = oracle.problem_histograms(p, "f64").astype(np.int64)
    pairs = np.array(p.pairs_per_hist()) * p.n_frames
    l1 = np.abs(h32 - h64).sum(axis=1)
    bound = 4 * p.n_bins * 2.0 ** -24              # model bound of DESIGN.md "fp32 vs fp64"
    assert (l1 <= bound * pairs + 8).all(), (l1 / pairs, bound)
    # every discrepancy is a move between adjacent bins: cumulative histograms differ by a few counts
    cum = np.abs(np.cumsum(h32, axis=1) - np.cumsum(h64, axis=1))
    per_bin = pairs / p.n_bins
    assert (cum.max(axis=1) <= np.maximum(8, 0.02 * per_bin)).all()
    # kept totals differ at most by pairs within a few ulp of r_max
    assert (np.abs(h32.sum(axis=1) - h64.sum(axis=1)) <= 4).all()


# ------------------------------------------------------------------ edge cases of the readings
def test_empty_species_and_single_bin():
    p = inputs.uniform_problem(3, (0, 50, 0), BOX_NONE, n_bins=1, r_max=5.0)
    h = oracle.problem_histograms(p)
    assert h.shape == (6, 1)
    assert [int(v) for v in h[:, 0]] == [0, 0, 0, 50 * 49 // 2, 0, 0]


def test_frames_sum_and_per_frame_boxes():
    """Eq. 2's sum over frames: one call over F frames == sum of F single-frame calls,
    with one shared box and with one box per frame."""
    g = np.random.Generator(np.random.PCG64(4))
    coords = (g.random((3, 200, 3)) * 9).astype(np.float32)
    boxes = np.array([np.diag([6.0, 7.0, 8.0]), np.diag([7.0, 7.0, 7.0]), np.diag([8.0, 6.5, 9.0])]).reshape(3, 9)
    off = [0, 80, 200]
    whole = oracle.histograms(coords, off, BOX_ORTHO, boxes, 3.0, 40)
    parts = sum(oracle.histograms(coords[f], off, BOX_ORTHO, boxes[f:f + 1], 3.0, 40).astype(np.int64)
                for f in range(3))
    assert np.array_equal(whole.astype(np.int64), parts)
    shared = oracle.histograms(coords, off, BOX_ORTHO, boxes[:1], 3.0, 40)
    parts1 = sum(oracle.histograms(coords[f], off, BOX_ORTHO, boxes[:1], 3.0, 40).astype(np.int64)
                 for f in range(3))
    assert np.array_equal(shared.astype(np.int64), parts1)
    assert not np.array_equal(whole, shared)


def test_q3_clamp_and_q2_cut_at_rmax():
    """A pair with d < (float)r_max whose d*scale rounds up to n_bins lands in the last bin (Q3); a pair
    with d == (float)r_max is dropped (Q2).  Expected values from IEEE float32 arithmetic in numpy."""
    found = None
    for n_bins in range(3, 4000):
        for r_max in (0.1, 0.3, 0.7, 1.1, 1.3):
            rm = np.float32(r_max)
            sc = np.float32(n_bins / r_max)
            d = np.nextafter(rm, np.float32(0))
            if np.float32(d * sc) >= np.float32(n_bins):
                found = (n_bins, r_max, d)
                break
        if found:
            break
    assert found, "no clamp case in the search range"
    n_bins, r_max, d = found
    pts = np.array([[0, 0, 0], [d, 0, 0], [0, np.float32(r_max), 0]], dtype=np.float32)
    # pairs: (0,1) distance d -> clamped into the last bin; (0,2) distance (float)r_max -> dropped;
    # (1,2) distance sqrt(d^2 + r_max^2) > r_max -> dropped
    h = oracle.histograms(pts, [0, 3], BOX_NONE, None, r_max, n_bins)
    assert int(h.sum()) == 1 and int(h[0, n_bins - 1]) == 1


def test_nan_pairs_are_dropped():
    pts = np.array([[0, 0, 0], [np.nan, 0, 0], [0.5, 0, 0]], dtype=np.float32)
    for bt, box in ((BOX_NONE, None), (BOX_ORTHO, np.diag([4.0, 4, 4])),
                    (BOX_TRICLINIC, np.diag([4.0, 4, 4]))):
        h = oracle.histograms(pts, [0, 3], bt, box, 1.0, 4)
        assert int(h.sum()) == 1 and int(h[0, 2]) == 1


def test_triclinic_with_diagonal_box_equals_ortho():
    """A triclinic box with a diagonal matrix is the orthorhombic special case; inside
    r_max <= L/2 both modes must bin identically in fp64 (fp32: the operation sequences differ)."""
    p = inputs.uniform_problem(8, (500,), BOX_ORTHO, n_bins=128, r_max=2.0, box=np.diag([4.0, 5.0, 6.0]),
                               spread=1.7)
    a = oracle.problem_histograms(p, "f64")
    b = oracle.histograms(p.coords, p.species_offsets, BOX_TRICLINIC, p.box, p.r_max, p.n_bins, precision="f64")
    assert np.abs(np.cumsum(a.astype(np.int64)) - np.cumsum(b.astype(np.int64))).max() <= 2
    assert abs(int(a.sum()) - int(b.sum())) <= 2


# ---- the stored full-size oracle histograms (tests/golden/cfg{3,4,5}_{f32,f64}.npz, make_fullsize.py) ------------------
@pytest.mark.parametrize("config,precision", [(c, p) for c in (3, 4, 5) for p in ("f32", "f64")])
def test_fullsize_goldens_belong_to_these_inputs_and_this_oracle(config, precision):
    """The files the GPU full-size tests compare against: written by the oracle source as it stands (sha256), for the
    inputs the generators produce today (sha256), and consistent with what the mathematics fixes at full size --
    the closed-form total where r_max covers every pair or the sphere/cell volume ratio of uniform
    points, and the chunk sums adding up to the whole (Eq. 2)."""
    import hashlib
    import importlib.util
    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    spec = importlib.util.spec_from_file_location("make_fullsize", os.path.join(here, "make_fullsize.py"))
    mf = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mf)
    d = np.load(mf.path(config, precision))
    assert str(d["sha_oracle"]) == mf.sha_oracle(), "oracle/cdh_oracle.c changed: rerun tests/golden/make_fullsize.py"
    p = inputs.make_config(config)
    assert str(d["sha_inputs"]) == mf.sha_inputs(p), "the seeded inputs changed: rerun tests/golden/make_fullsize.py"
    h = d["hist"]
    assert h.shape == (p.n_hist, p.n_bins) and h.dtype == np.uint64
    kept = int(h.sum())
    if config == 5:
        assert kept == 1_000_000 * 999_999 // 2                         # every pair is within sqrt(3) of every other
    else:
        want = math.pi / 12 if config == 3 else math.pi / 6               # sphere of radius r_max / cell volume
        assert kept / p.evaluated_pairs == pytest.approx(want, rel=2e-3)
        per_row = h.sum(axis=1) / (np.array(p.pairs_per_hist(), dtype=np.float64) * p.n_frames)
        assert np.allclose(per_row, want, rtol=1e-2)                      # every species pair separately
    if config == 4:
        assert d["chunk_hist"].shape == (8, p.n_hist, p.n_bins)
        assert np.array_equal(d["chunk_hist"].sum(axis=0, dtype=np.uint64), h)
    # ideal-gas shape of a uniform periodic system: counts grow like r^2 (compare two wide shells)
    if config in (3, 4):
        n = p.n_bins
        a, b = h[:, n // 4: n // 4 + n // 8].sum(), h[:, n // 2: n // 2 + n // 8].sum()
        r1, r2 = (n // 4, n // 4 + n // 8), (n // 2, n // 2 + n // 8)
        want_ratio = (r2[1] ** 3 - r2[0] ** 3) / (r1[1] ** 3 - r1[0] ** 3)
        assert b / a == pytest.approx(want_ratio, rel=5e-3)
