"""CPU oracle for the pair-distance histogram -- TEST INFRASTRUCTURE, not the product.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It shares no code with ``paper_1808_01478_b200/csrc`` and never
imports the CUDA binding.  See ``cdh_oracle.c`` for what it computes and the passages it follows.
"""
from .oracle import build, histograms, problem_histograms, pair_d2, max_threads  # noqa: F401
