"""ctypes front end of ``cdh_oracle.c`` (test infrastructure; see the C file's header)."""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cdh_oracle.c")
_LIB = os.path.join(_HERE, "libcdh_oracle.so")

# No FMA contraction, no fast-math, default rounding; -fno-math-errno only lets gcc inline sqrtss /
# roundss (value-preserving).  Baseline x86-64 + SSE4.1 so the library runs on any host of the image.
CFLAGS = ["-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-msse4.1", "-ffp-contract=off",
          "-fno-fast-math", "-fno-unsafe-math-optimizations", "-fno-math-errno", "-Wall", "-Wextra"]

_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc if the shared object is missing or older than its source."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.run(["gcc", *CFLAGS, "-o", tmp, _SRC, "-lm"], check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.cdh_oracle_histograms.restype = ctypes.c_int
        lib.cdh_oracle_histograms.argtypes = [
            ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_int, ctypes.c_int,
            ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_int, ctypes.c_int, ctypes.c_int,
            ctypes.c_void_p]
        lib.cdh_oracle_pair_d2.restype = ctypes.c_double
        lib.cdh_oracle_pair_d2.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int,
                                           ctypes.c_void_p, ctypes.c_int]
        lib.cdh_oracle_rdf.restype = ctypes.c_int
        lib.cdh_oracle_rdf.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_int,
                                       ctypes.c_void_p, ctypes.c_double, ctypes.c_void_p]
        lib.cdh_oracle_max_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def max_threads() -> int:
    return int(_load().cdh_oracle_max_threads())


def histograms(coords: np.ndarray, species_offsets, box_type: int, box: Optional[np.ndarray],
               r_max: float, n_bins: int, precision: str = "f32", n_threads: int = 0) -> np.ndarray:
    """uint64 [n_hist, n_bins]: all species-pair histograms summed over the frames of ``coords``.

    coords: float32 or float64 [n_frames, n_total, 3] (or [n_total, 3]); precision "f32" is the pinned
    fp32 sequence, "f64" the same sequence in double (inputs converted exactly).
    """
    lib = _load()
    c = np.ascontiguousarray(coords)
    if c.ndim == 2:
        c = c[None]
    if c.dtype not in (np.float32, np.float64) or c.ndim != 3 or c.shape[2] != 3:
        raise ValueError("coords must be float32/float64 [n_frames, n_total, 3]")
    off = np.ascontiguousarray(species_offsets, dtype=np.int32)
    n_species = len(off) - 1
    if off[0] != 0 or off[-1] != c.shape[1] or (np.diff(off) < 0).any():
        raise ValueError("bad species_offsets")
    n_hist = n_species * (n_species + 1) // 2
    out = np.zeros((n_hist, n_bins), dtype=np.uint64)
    if box_type == 0:
        b, n_boxes, bp = None, 0, None
    else:
        b = np.ascontiguousarray(box, dtype=np.float64).reshape(-1, 9)
        n_boxes, bp = b.shape[0], b.ctypes.data
    rc = lib.cdh_oracle_histograms(c.ctypes.data, int(c.dtype == np.float64), c.shape[0],
                                   off.ctypes.data, n_species, int(box_type), bp, n_boxes,
                                   float(r_max), int(n_bins), {"f32": 0, "f64": 1}[precision],
                                   int(n_threads), out.ctypes.data)
    if rc != 0:
        raise ValueError(f"cdh_oracle_histograms rejected its arguments (rc={rc})")
    return out


def problem_histograms(p, precision: str = "f32", n_threads: int = 0) -> np.ndarray:
    """``histograms`` on a ``paper_1808_01478_b200.inputs.Problem``-shaped object."""
    return histograms(p.coords, p.species_offsets, p.box_type, p.box, p.r_max, p.n_bins,
                      precision=precision, n_threads=n_threads)


def pair_d2(pi, pj, box_type: int, box: Optional[np.ndarray], precision: str = "f32") -> float:
    """Squared minimum-image distance of one pair by the pinned sequence."""
    lib = _load()
    a = np.ascontiguousarray(pi, dtype=np.float64)
    b = np.ascontiguousarray(pj, dtype=np.float64)
    bx = None if box_type == 0 else np.ascontiguousarray(box, dtype=np.float64).reshape(9)
    return float(lib.cdh_oracle_pair_d2(a.ctypes.data, b.ctypes.data, int(box_type),
                                        None if bx is None else bx.ctypes.data,
                                        {"f32": 0, "f64": 1}[precision]))


def rdf(hist: np.ndarray, r_max: float, n_frames: int, n_pairs, volume: float) -> np.ndarray:
    """g(r) per histogram row from summed uint64 counts (Eqs. 1-3); float64 [n_hist, n_bins]."""
    lib = _load()
    h = np.ascontiguousarray(hist, dtype=np.uint64)
    if h.ndim == 1:
        h = h[None]
    npairs = np.ascontiguousarray(n_pairs, dtype=np.float64).reshape(-1)
    if npairs.shape[0] != h.shape[0]:
        raise ValueError("one pair count per histogram row")
    g = np.empty(h.shape, dtype=np.float64)
    rc = lib.cdh_oracle_rdf(h.ctypes.data, h.shape[0], h.shape[1], float(r_max), int(n_frames), npairs.ctypes.data,
                            float(volume), g.ctypes.data)
    if rc != 0:
        raise ValueError("cdh_oracle_rdf rejected its arguments")
    return g
