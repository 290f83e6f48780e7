"""Writes tests/golden/cfg{3,4,5}_{f32,f64}.npz: the CPU oracle's histograms of configs 3, 4, 5 at FULL size.

SURVEY.md 8(d): "Full-size oracle histograms are needed for parity on every config ... compute once, cache on disk
keyed by a hash of (input bytes, parameters, oracle source)".  Every stored value is produced by ``oracle/`` alone, on
the seeded inputs of ``paper_1808_01478_b200/inputs.py`` (generators only; no arithmetic of the method).  This script
imports nothing else of the package and never touches the CUDA library.

Each file holds
    hist        uint64 [n_hist, n_bins]   the oracle's result (config 4: summed over the 64 frames, Eq. 2)
    chunk_hist  uint64 [n_frames / 8, n_hist, n_bins]  (config 4 only: the sum over each run of 8 consecutive frames, so that
                chunked calls can be checked against the oracle too)
    sha_inputs  sha256 of coords bytes + species offsets + box + r_max + n_bins
    sha_oracle  sha256 of oracle/cdh_oracle.c
    seconds, threads  how long the oracle took here

Run (CPU only, minutes to tens of minutes on 8 cores):
    python tests/golden/make_fullsize.py [--configs 3 4 5] [--precisions f32 f64]

tests/test_gpu_fullsize.py / test_gpu_f64.py compare the CUDA result with ``hist`` bin by bin, and
tests/test_oracle_pins.py (CPU) re-checks the hashes and the closed-form totals of the stored histograms.
"""
from __future__ import annotations

import argparse
import hashlib
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

# inputs.py is loaded by path so that the package's __init__ (which loads the CUDA binding) is not imported
import importlib.util  # noqa: E402

_spec = importlib.util.spec_from_file_location("cdh_inputs_for_golden", os.path.join(ROOT, "paper_1808_01478_b200", "inputs.py"))
inputs = importlib.util.module_from_spec(_spec)
sys.modules[_spec.name] = inputs
_spec.loader.exec_module(inputs)

from oracle import oracle as cdh_oracle  # noqa: E402


CHUNK_FRAMES = 8


def sha_inputs(p) -> str:
    h = hashlib.sha256()
    h.update(np.ascontiguousarray(p.coords).tobytes())
    h.update(np.ascontiguousarray(p.species_offsets, dtype=np.int32).tobytes())
    h.update(b"" if p.box is None else np.ascontiguousarray(p.box, dtype=np.float64).tobytes())
    h.update(np.array([p.r_max], dtype=np.float64).tobytes())
    h.update(np.array([p.n_bins, p.box_type], dtype=np.int64).tobytes())
    return h.hexdigest()


def sha_oracle() -> str:
    with open(os.path.join(ROOT, "oracle", "cdh_oracle.c"), "rb") as f:
        return hashlib.sha256(f.read()).hexdigest()


def path(config: int, precision: str) -> str:
    return os.path.join(HERE, f"cfg{config}_{precision}.npz")


def make(config: int, precision: str) -> None:
    p = inputs.make_config(config)
    t0 = time.time()
    extra = {}
    if p.n_frames > 1:
        frames = np.zeros((p.n_frames, p.n_hist, p.n_bins), dtype=np.uint64)
        for f in range(p.n_frames):
            frames[f] = cdh_oracle.histograms(p.coords[f:f + 1], p.species_offsets, p.box_type, p.box, p.r_max, p.n_bins,
                                              precision=precision)
            print(f"  cfg{config} {precision} frame {f + 1}/{p.n_frames}  {time.time() - t0:.0f} s", flush=True)
        hist = frames.sum(axis=0, dtype=np.uint64)
        extra["chunk_hist"] = frames.reshape(p.n_frames // CHUNK_FRAMES, CHUNK_FRAMES, p.n_hist, p.n_bins).sum(axis=1, dtype=np.uint64)
        extra["chunk_frames"] = CHUNK_FRAMES
    else:
        hist = cdh_oracle.problem_histograms(p, precision)
    dt = time.time() - t0
    np.savez_compressed(path(config, precision), hist=hist, sha_inputs=sha_inputs(p), sha_oracle=sha_oracle(),
                        seconds=dt, threads=cdh_oracle.max_threads(), **extra)
    print(f"cfg{config} {precision}: {p.evaluated_pairs} pairs, kept {int(hist.sum())}, {dt:.0f} s "
          f"({p.evaluated_pairs / dt / 1e9:.2f} Gpairs/s on {cdh_oracle.max_threads()} threads) -> {path(config, precision)}",
          flush=True)


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", type=int, nargs="+", default=[3, 4, 5])
    ap.add_argument("--precisions", nargs="+", default=["f32", "f64"])
    a = ap.parse_args()
    cdh_oracle.build()
    for prec in a.precisions:
        for c in a.configs:
            make(c, prec)


if __name__ == "__main__":
    main()
