"""-m "not gpu": the host logic of libcdh (csrc/cdh_host.h) through its test hooks (include/cdh_bench.h); no GPU.

  * the d2 threshold that replaces "d < r_max" in the kernels,
  * the constant of the fused rint,
  * the work list: every pair of every species pair, sweep and frame is covered exactly once.
"""
import ctypes

import numpy as np
import pytest

from paper_1808_01478_b200 import binding
from paper_1808_01478_b200 import build as cdh_build

f32 = np.float32


@pytest.fixture(scope="module")
def lib():
    cdh_build.build()
    return binding.load()


def test_d2_threshold_is_the_exact_cut(lib):
    g = np.random.Generator(np.random.PCG64(3))
    rmaxs = np.concatenate([g.uniform(1e-3, 1e3, 400), [1.0, 0.7, 5.0, 4.0, np.sqrt(3.0), 4.242640687119285, 1e-20, 1e18]])
    for r in rmaxs.astype(np.float32):
        bits = lib.cdh_host_d2_threshold_bits(ctypes.c_float(float(r)))
        thr = np.uint32(bits).view(np.float32)
        below = np.nextafter(thr, f32(0))
        # numpy's float32 sqrt is correctly rounded: thr is the smallest d2 with sqrt(d2) >= r_max
        assert np.sqrt(thr) >= r and np.sqrt(below) < r, (r, thr)


def pinned_n(d, inv_l):
    return np.rint((d.astype(np.float32) * f32(inv_l)).astype(np.float32))


def fused_n(d, inv_lf):
    return np.rint(d.astype(np.float64) * np.float64(inv_lf))        # exact product of two floats in double, one rint


def test_fused_rint_constant_agrees_with_the_pinned_form(lib):
    g = np.random.Generator(np.random.PCG64(4))
    found = 0
    for L in np.concatenate([g.uniform(0.5, 200.0, 300), [10.0, 8.0, 12.0, 6.0, 7.3]]):
        inv_l = f32(1.0 / L)
        out = ctypes.c_float()
        if not lib.cdh_host_fused_rint_constant(ctypes.c_float(float(inv_l)), ctypes.byref(out)):
            continue
        found += 1
        inv_lf = f32(out.value)
        half = f32(0.5 / np.float64(inv_l))
        # every float within 200 ulps of the 0 -> 1 switch, both signs, plus a coarse sweep of the whole range |t| < 1.49
        near = half.view(np.uint32).astype(np.int64) + np.arange(-200, 201)
        d = np.concatenate([near.astype(np.uint32).view(np.float32), np.linspace(0.0, 1.49 * L, 20001).astype(np.float32)])
        d = np.concatenate([d, -d])
        assert np.array_equal(pinned_n(d, inv_l), fused_n(d, inv_lf)), L
    assert found > 200                      # ~81 % of random box lengths have a constant


def covered_pairs(items, ni, nj, same, ti):
    """pairs (i, j) of one species pair covered by the given items, counted with multiplicity"""
    count = np.zeros((ni, nj), dtype=np.int32)
    for it in items:
        i0, j0, j1 = int(it[3]), int(it[4]), int(it[5])
        i1 = min(ni, i0 + ti)
        if j1 <= j0:
            continue
        blk = count[i0:i1, j0:j1]
        if same:
            ii, jj = np.meshgrid(np.arange(i0, i1), np.arange(j0, j1), indexing="ij")
            blk += (jj > ii)
        else:
            blk += 1
    return count


@pytest.mark.parametrize("counts,ti,tj", [((700,), 256, 256), ((1030, 517), 1024, 256), ((5, 0, 2100, 1), 1024, 512),
                                          ((3000,), 4096, 1024), ((2000,), 1024, 32), ((700, 130), 1024, 64)])
def test_work_list_covers_every_pair_exactly_once(lib, counts, ti, tj):
    off = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
    n_species, n_frames, n_bins, cap = len(counts), 2, 1000, 300            # 4 sweeps
    items = np.zeros((200000, 8), dtype=np.int64)
    n = lib.cdh_host_work_items(n_frames, off.ctypes.data, n_species, n_bins, cap, ti, tj, items.ctypes.data, len(items))
    assert 0 <= n <= len(items)
    items = items[:n]
    sweeps = sorted({(int(a), int(b)) for a, b in items[:, 1:3]}) if n else []
    if n:
        assert sum(b for _, b in sweeps) == n_bins and sweeps[0][0] == 0       # the sweeps tile [0, n_bins)
    h = 0
    for p in range(n_species):
        for q in range(p, n_species):
            ni, nj = counts[p], counts[q]
            mine = items[items[:, 0] == h]
            want_pairs = ni * (ni - 1) // 2 if p == q else ni * nj
            if want_pairs == 0:
                assert len(mine) == 0
            else:
                for lo, cnt in sweeps:
                    sel = mine[(mine[:, 1] == lo) & (mine[:, 2] == cnt)]
                    assert (sel[:, 6] == (p == q)).all()
                    frames = sorted(set(sel[:, 7].tolist()))                 # group offsets differ per frame
                    per_frame = [sel[sel[:, 7] == fkey] for fkey in frames]
                    assert len(per_frame) == n_frames
                    for chunk in per_frame:
                        c = covered_pairs(chunk, ni, nj, p == q, ti)
                        expect = np.triu(np.ones((ni, nj), dtype=np.int32), 1) if p == q else np.ones((ni, nj), dtype=np.int32)
                        assert np.array_equal(c, expect), (p, q, lo)
            h += 1
