"""Seeded synthetic input generators for the five BASELINE.json configs.

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA
path: it draws particle coordinates and states the problem parameters.  It holds
none of the method's arithmetic (no distances, no minimum image, no binning).

Recipe: every config uses
``numpy.random.Generator(PCG64(SEED_BASE + config))``, draws in float64, casts to
float32 once; a value that rounds up to an exclusive upper bound is replaced by
``nextafter(bound, 0)``.  The inputs stand in for the paper's "particles at
pseudo-random coordinates in a unit box" (section 4) and for its MD
and astrophysics use cases; nothing from the paper's
F1-ATPase trajectory is reproduced.

A ``Problem`` carries exactly the arguments of ``cdh_histograms`` (include/cdh.h).
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np

SEED_BASE = 1808014780

BOX_NONE = 0
BOX_ORTHO = 1
BOX_TRICLINIC = 2


@dataclasses.dataclass
class Problem:
    name: str
    coords: np.ndarray            # float32 [n_frames, n_total, 3], C-contiguous
    species_offsets: np.ndarray   # int32 [n_species + 1]
    box_type: int
    box: Optional[np.ndarray]     # float64 [n_boxes, 9] row-major, rows = box vectors; None for BOX_NONE
    r_max: float
    n_bins: int

    @property
    def n_frames(self) -> int:
        return int(self.coords.shape[0])

    @property
    def n_total(self) -> int:
        return int(self.coords.shape[1])

    @property
    def n_species(self) -> int:
        return int(len(self.species_offsets) - 1)

    @property
    def n_boxes(self) -> int:
        return 0 if self.box is None else int(self.box.shape[0])

    @property
    def n_hist(self) -> int:
        s = self.n_species
        return s * (s + 1) // 2

    def species_counts(self):
        o = self.species_offsets
        return [int(o[k + 1] - o[k]) for k in range(self.n_species)]

    def pairs_per_hist(self):
        """Evaluated pairs per histogram (row-major upper triangle p <= q), one frame."""
        n = self.species_counts()
        out = []
        for p in range(self.n_species):
            for q in range(p, self.n_species):
                out.append(n[p] * (n[p] - 1) // 2 if p == q else n[p] * n[q])
        return out

    @property
    def evaluated_pairs(self) -> int:
        return self.n_frames * sum(self.pairs_per_hist())


def hist_index(p: int, q: int, n_species: int) -> int:
    """Row-major upper-triangle index of species pair (p <= q); include/cdh.h."""
    if p > q:
        p, q = q, p
    return p * n_species - p * (p - 1) // 2 + (q - p)


def _to_f32_below(x64: np.ndarray, bound: float) -> np.ndarray:
    """float64 -> float32 once; values that round up to ``bound`` become nextafter(bound, 0)."""
    x32 = x64.astype(np.float32)
    b32 = np.float32(bound)
    hit = x32 >= b32
    if hit.any():
        x32[hit] = np.nextafter(b32, np.float32(0.0))
    return x32


def _rng(config: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(SEED_BASE + config))


def _offsets(counts) -> np.ndarray:
    return np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)


def config1(n: int = 2000, n_bins: int = 1000) -> Problem:
    """1 species, uniform in [0,1)^3, non-periodic, bins over [0, sqrt(3))."""
    g = _rng(1)
    x = _to_f32_below(g.random((n, 3)), 1.0)
    return Problem("cfg1_uniform_nobox", x[None].copy(), _offsets([n]), BOX_NONE, None,
                   math.sqrt(3.0), n_bins)


def config2(counts=(5000, 30000, 60000), n_bins: int = 10000, edge: float = 10.0,
            r_max: Optional[float] = None) -> Problem:
    """Water-box-like MD frame: 3 species uniform in an orthorhombic periodic box."""
    g = _rng(2)
    n = int(sum(counts))
    x = _to_f32_below(edge * g.random((n, 3)), edge)
    box = np.diag([edge, edge, edge]).astype(np.float64).reshape(1, 9)
    return Problem("cfg2_waterbox_ortho", x[None].copy(), _offsets(counts), BOX_ORTHO, box,
                   edge / 2 if r_max is None else r_max, n_bins)


def rhombic_dodecahedron_box(d: float) -> np.ndarray:
    """Rows a=(d,0,0), b=(0,d,0), c=(d/2,d/2,d*sqrt(2)/2) (BASELINE.json config 3)."""
    return np.array([[d, 0.0, 0.0], [0.0, d, 0.0], [d / 2, d / 2, d * math.sqrt(2.0) / 2]],
                    dtype=np.float64)


def config3(counts=(40000, 60000), n_bins: int = 20000, d: float = 12.0,
            r_max: Optional[float] = None) -> Problem:
    """Triclinic periodic frame (rhombic dodecahedron), uniform in fractional coordinates.

    Default r_max = half the minimum box height = d*sqrt(2)/4.
    """
    g = _rng(3)
    n = int(sum(counts))
    s = g.random((n, 3))
    box = rhombic_dodecahedron_box(d)
    x64 = s @ box                     # x = s0*a + s1*b + s2*c (rows are the box vectors)
    x = x64.astype(np.float32)
    return Problem("cfg3_triclinic_rhombdodec", x[None].copy(), _offsets(counts), BOX_TRICLINIC,
                   box.reshape(1, 9), d * math.sqrt(2.0) / 4 if r_max is None else r_max, n_bins)


def config4(n_frames: int = 64, counts=(10000, 40000), n_bins: int = 8000, edge: float = 8.0,
            sigma: float = 0.05) -> Problem:
    """Trajectory batch: a seeded base configuration plus per-frame Gaussian jitter (NOT re-wrapped)."""
    g = _rng(4)
    n = int(sum(counts))
    base = edge * g.random((n, 3))
    frames = np.empty((n_frames, n, 3), dtype=np.float32)
    for f in range(n_frames):
        frames[f] = (base + sigma * g.standard_normal((n, 3))).astype(np.float32)
    box = np.diag([edge, edge, edge]).astype(np.float64).reshape(1, 9)
    return Problem("cfg4_trajectory_ortho", frames, _offsets(counts), BOX_ORTHO, box, edge / 2, n_bins)


def config5(n: int = 1_000_000, n_bins: int = 50000, n_clusters: int = 2000,
            sigma: float = 0.005, background: float = 0.2, cluster_major: bool = False) -> Problem:
    """Astrophysics-like clustered set: Gaussian clusters + uniform background in the unit cube.

    Each point independently: with probability ``background`` uniform in the cube, else a uniformly
    chosen centre + sigma*N(0, I3), redrawn until inside [0,1)^3.  Emitted in draw order (spatially
    shuffled); ``cluster_major=True`` sorts by component id (the adversarial order for shared atomics).
    """
    g = _rng(5)
    centres = g.random((n_clusters, 3))
    is_bg = g.random(n) < background
    comp = np.where(is_bg, -1, g.integers(0, n_clusters, size=n))
    x = np.empty((n, 3), dtype=np.float64)
    x[is_bg] = g.random((int(is_bg.sum()), 3))
    todo = np.flatnonzero(~is_bg)
    while todo.size:
        cand = centres[comp[todo]] + sigma * g.standard_normal((todo.size, 3))
        c32 = cand.astype(np.float32)
        ok = ((c32 >= 0.0) & (c32 < 1.0)).all(axis=1)
        x[todo[ok]] = cand[ok]
        todo = todo[~ok]
    x32 = _to_f32_below(x, 1.0)
    if cluster_major:
        x32 = x32[np.argsort(comp, kind="stable")]
    name = "cfg5_clustered_nobox" + ("_clustermajor" if cluster_major else "")
    return Problem(name, x32[None].copy(), _offsets([n]), BOX_NONE, None, math.sqrt(3.0), n_bins)


def make_config(k: int, **kw) -> Problem:
    return {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}[k](**kw)


def reduced_config(k: int) -> Problem:
    """Same recipe, shrunk so the CPU oracle finishes in seconds while still spanning several
    tiles, a ragged tail and every species pair."""
    if k == 1:
        return config1()
    if k == 2:
        return config2(counts=(700, 3100, 5300), n_bins=10000)
    if k == 3:
        return config3(counts=(2300, 3700), n_bins=20000)
    if k == 4:
        return config4(n_frames=3, counts=(1100, 4300), n_bins=8000)
    if k == 5:
        return config5(n=21001, n_bins=50000, n_clusters=40)
    raise ValueError(k)


def uniform_problem(seed: int, counts, box_type: int, n_bins: int, r_max: float,
                    box: Optional[np.ndarray] = None, n_frames: int = 1, spread: float = 1.0) -> Problem:
    """Generic seeded uniform points (tests): coordinates uniform in [0, spread)^3 (BOX_NONE / ORTHO)
    or uniform in fractional coordinates times ``spread`` (TRICLINIC; spread > 1 leaves the cell)."""
    g = np.random.Generator(np.random.PCG64(seed))
    n = int(sum(counts))
    frames = np.empty((n_frames, n, 3), dtype=np.float32)
    for f in range(n_frames):
        s = g.random((n, 3)) * spread
        if box_type == BOX_TRICLINIC:
            frames[f] = (s @ np.asarray(box, dtype=np.float64).reshape(-1, 3, 3)[0]).astype(np.float32)
        elif box_type == BOX_ORTHO:
            diag = np.asarray(box, dtype=np.float64).reshape(-1, 3, 3)[0].diagonal()
            frames[f] = (s * diag).astype(np.float32)
        else:
            frames[f] = s.astype(np.float32)
    b = None if box_type == BOX_NONE else np.asarray(box, dtype=np.float64).reshape(-1, 9)
    return Problem(f"uniform_seed{seed}", frames, _offsets(counts), box_type, b, float(r_max), int(n_bins))
