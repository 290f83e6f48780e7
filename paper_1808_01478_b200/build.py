"""Build libcdh.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

``python -m paper_1808_01478_b200.build`` or ``build()``; nvcc cross-compiles without a GPU.
The host code derives constants of the pinned sequence in double, so it is compiled without FP
contraction (-ffp-contract=off).
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libcdh.so")
# cdh_api.cu: the C ABI and host dispatch; cdh_k_*.cu: the tile-kernel instantiations, one translation unit per box
# type so that they compile in parallel; cdh_bench.cu: the roofline microbenchmarks and self-tests.
SOURCES = ["cdh_api.cu", "cdh_bench.cu", "cdh_k_none.cu", "cdh_k_ortho.cu", "cdh_k_tri.cu", "cdh_k_tri_wide.cu",
           "cdh_k_simple.cu", "cdh_k_f64.cu", "cdh_noalloc.cu"]
INCLUDE = os.path.join(_HERE, "..", "include")


def deps():
    """Every source and header the library is built from (all of csrc/ and include/)."""
    out = [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC)) if f.endswith((".cu", ".cuh", ".h"))]
    out += [os.path.join(INCLUDE, f) for f in sorted(os.listdir(INCLUDE)) if f.endswith(".h")]
    return out


NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC,-ffp-contract=off,-fno-fast-math"]
LINK_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static"]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in deps())


def build(force: bool = False, verbose: bool = False, extra_flags=(), out: str = LIB) -> str:
    """Compile if the library is missing or older than a source; returns its path.  ``extra_flags`` / ``out``
    build an experimental copy (e.g. ``-DCDH_MINB=3``) next to the product library.  The translation units are
    compiled concurrently (one nvcc process each), then linked into one shared object."""
    if force or out != LIB or is_stale():
        import concurrent.futures
        import tempfile
        nvcc = nvcc_path()
        with tempfile.TemporaryDirectory(prefix="cdh_build_") as tmpdir:
            def compile_one(src):
                obj = os.path.join(tmpdir, src.replace(".cu", ".o"))
                cmd = [nvcc, *NVCC_FLAGS, *extra_flags, "-c", "-o", obj, os.path.join(CSRC, src)]
                if verbose:
                    cmd.insert(1, "-Xptxas=-v")
                    print(" ".join(cmd), file=sys.stderr)
                r = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
                return src, obj, r
            with concurrent.futures.ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 1)) as pool:
                results = list(pool.map(compile_one, SOURCES))
            for src, _obj, r in results:
                if verbose or r.returncode != 0:
                    sys.stderr.write(r.stdout + r.stderr)
                if r.returncode != 0:
                    raise subprocess.CalledProcessError(r.returncode, f"nvcc -c {src}")
            tmp = out + f".tmp{os.getpid()}"
            subprocess.run([nvcc, *LINK_FLAGS, "-o", tmp, *[obj for _s, obj, _r in results]], check=True, cwd=CSRC)
            os.replace(tmp, out)
    return out


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
