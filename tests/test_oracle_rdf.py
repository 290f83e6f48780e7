"""-m "not gpu": pins of the oracle's g(r) post-processing (Eqs. 1-3).

What fixes it with no implementation to compare against:
  * ideal gas: uniform points in a periodic box have g(r) = 1 for r < L/2 (the textbook limit of Eq. 1);
  * a simple-cubic crystal has delta peaks exactly at a*sqrt(h^2+k^2+l^2) with known coordination numbers 6, 12, 8, 6;
  * closed form: with r at the bin centre, 4 pi r^2 dr equals the exact shell volume minus pi dr^3 / 3;
  * scaling laws of Eq. 1 / Eq. 2: g is linear in the counts and in V, inversely linear in N_frames and N_pairs.
"""
import math

import numpy as np

from oracle import oracle as cdh_oracle
from paper_1808_01478_b200 import inputs


def test_ideal_gas_is_one():
    p = inputs.config2(counts=(1500, 2500, 3000), n_bins=50)
    h = cdh_oracle.problem_histograms(p, "f64")
    g = cdh_oracle.rdf(h, p.r_max, 1, p.pairs_per_hist(), 10.0 ** 3)
    # expected counts per bin are 10^3..10^5 here: 5 sigma of the Poisson noise plus the finite-bin bias
    counts = h.astype(np.float64)
    tol = 5.0 / np.sqrt(np.maximum(counts, 1.0)) + 1e-3
    assert (np.abs(g - 1.0)[:, 5:] < tol[:, 5:]).all()
    assert abs(g[:, 5:].mean() - 1.0) < 2e-3


def test_simple_cubic_crystal_peaks_and_coordination_numbers():
    n, a = 6, 1.0                                    # 6^3 sites, lattice constant 1, periodic box of edge 6
    idx = np.arange(n)
    pts = np.stack(np.meshgrid(idx, idx, idx, indexing="ij"), axis=-1).reshape(-1, 3).astype(np.float32) * a
    n_bins, r_max = 300, 3.0                         # dr = 0.01
    h = cdh_oracle.histograms(pts[None], [0, len(pts)], inputs.BOX_ORTHO, np.diag([6.0, 6.0, 6.0]), r_max, n_bins, "f64")
    npairs = len(pts) * (len(pts) - 1) / 2
    g = cdh_oracle.rdf(h, r_max, 1, [npairs], 6.0 ** 3)[0]
    shells = {1.0: 6, math.sqrt(2.0): 12, math.sqrt(3.0): 8, 2.0: 6}        # distance -> coordination number
    nz = set(np.flatnonzero(g).tolist())
    dr = r_max / n_bins
    for r, z in shells.items():
        k = int(math.floor(r / dr + 1e-9))
        assert k in nz
        # Eq. 1 inverted: neighbours per atom in the bin = g * 4 pi rho r_c^2 dr with rho = N / V
        r_c = (k + 0.5) * dr
        neigh = g[k] * 4.0 * math.pi * (npairs / 6.0 ** 3) * r_c * r_c * dr * 2.0 / len(pts)
        assert neigh == pytest_approx(z)
    assert all(abs(((k + 0.5) * dr) ** 2 - round(((k + 0.5) * dr) ** 2)) < 0.05 for k in nz)   # peaks only at sqrt(integer)


def pytest_approx(x):
    import pytest
    return pytest.approx(x, rel=1e-12)


def test_bin_centre_shell_identity_and_scaling_laws():
    rng = np.random.default_rng(7)
    h = rng.integers(0, 10 ** 12, size=(2, 64), dtype=np.uint64)
    r_max, frames, npairs, vol = 2.5, 7, [1.5e9, 3.0e9], 321.0
    g = cdh_oracle.rdf(h, r_max, frames, npairs, vol)
    dr = r_max / 64
    k = np.arange(64)
    exact_shell = 4.0 * math.pi / 3.0 * (((k + 1) * dr) ** 3 - (k * dr) ** 3)
    g_exact = h / frames / ((np.array(npairs)[:, None] / vol) * exact_shell[None, :])
    ratio = g / g_exact                                       # = 1 + dr^2 / (12 r_c^2)
    want = 1.0 + dr * dr / (12.0 * ((k + 0.5) * dr) ** 2)
    assert np.allclose(ratio, want[None, :], rtol=1e-13, atol=0)
    assert np.array_equal(cdh_oracle.rdf(h, r_max, frames, npairs, 2 * vol), 2 * g)          # exact powers of two
    assert np.array_equal(cdh_oracle.rdf(h, r_max, 2 * frames, npairs, vol), g / 2)
    assert np.array_equal(cdh_oracle.rdf(h, r_max, frames, [2 * n for n in npairs], vol), g / 2)
    assert np.array_equal(cdh_oracle.rdf(h // 2 * 2, r_max, frames, npairs, vol)[0] > 0, h[0] // 2 * 2 > 0)
