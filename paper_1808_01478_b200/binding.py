"""ctypes binding of libcdh.so: same names as include/cdh.h, argument marshalling only.

Every step of the path runs inside the CUDA library; there is no CPU fallback.  Loading or calling
without the built library / without a CUDA device raises (``CdhError`` or ``OSError``).
PyTorch is used by callers for device buffers and streams only; this module accepts torch CUDA
tensors or raw device pointers (ints).
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcdh.so")

BOX_NONE, BOX_ORTHO, BOX_TRICLINIC = 0, 1, 2
F32, F64 = 0, 1
OK, ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_ALLOC, ERR_CUDA = 0, -1, -2, -3, -4
FLAG_SIMPLE_KERNEL = 1 << 0
FLAG_NO_PRUNE = 1 << 1
FLAG_WARP_AGGREGATE = 1 << 2
FLAG_NO_AGGREGATE = 1 << 3
FLAG_TIME_KERNELS = 1 << 4
FLAG_GLOBAL_HIST = 1 << 5
FLAG_ACCUMULATE = 1 << 6
FLAG_NO_PDL = 1 << 7
FLAG_NO_ITEM_TABLE = 1 << 8
FLAG_MAX_SMEM_BINS_SHIFT = 12

EXPORTS = ["cdh_create", "cdh_histograms", "cdh_histograms_host", "cdh_histograms_stream", "cdh_destroy", "cdh_strerror",
           "cdh_last_error", "cdh_last_call_info", "cdh_call_kernel_ms", "cdh_rdf", "cdh_histograms_noalloc", "cdh_noalloc_last_error",
           "cdh_bench_fp32_rate", "cdh_bench_shared_atomics", "cdh_bench_inner_loop", "cdh_bench_dsmem_atomics", "cdh_selftest_sqrt", "cdh_selftest_sqrt_f64",
           "cdh_host_d2_threshold_bits", "cdh_host_fused_rint_constant", "cdh_host_work_items"]


class CdhError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"cdh error {code}: {text}")
        self.code = code


_lib = None


def load(path: Optional[str] = None) -> ctypes.CDLL:
    """dlopen libcdh.so and declare the signatures.  Fails loudly if it was not built."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or LIB_PATH
    if not os.path.exists(p):
        raise OSError(f"{p} not found: build it with `python -m paper_1808_01478_b200.build` "
                      "(there is no CPU fallback)")
    lib = ctypes.CDLL(p)
    vp, i32, u32, dbl = ctypes.c_void_p, ctypes.c_int32, ctypes.c_uint32, ctypes.c_double
    lib.cdh_create.restype = ctypes.c_int
    lib.cdh_create.argtypes = [ctypes.POINTER(vp), ctypes.c_int, u32]
    hist_args = [vp, vp, i32, vp, i32, i32, vp, i32, dbl, i32, i32, vp, vp]
    lib.cdh_histograms.restype = ctypes.c_int
    lib.cdh_histograms.argtypes = hist_args
    lib.cdh_histograms_host.restype = ctypes.c_int
    lib.cdh_histograms_host.argtypes = hist_args
    lib.cdh_histograms_stream.restype = ctypes.c_int
    lib.cdh_histograms_stream.argtypes = hist_args[:11] + [i32, vp, vp]
    lib.cdh_histograms_noalloc.restype = ctypes.c_int
    lib.cdh_histograms_noalloc.argtypes = [ctypes.c_int, vp, i32, vp, i32, i32, vp, i32, dbl, i32, vp, vp]
    lib.cdh_noalloc_last_error.restype = ctypes.c_char_p
    lib.cdh_noalloc_last_error.argtypes = []
    lib.cdh_destroy.restype = ctypes.c_int
    lib.cdh_destroy.argtypes = [vp]
    lib.cdh_strerror.restype = ctypes.c_char_p
    lib.cdh_strerror.argtypes = [ctypes.c_int]
    lib.cdh_last_error.restype = ctypes.c_char_p
    lib.cdh_last_error.argtypes = [vp]
    lib.cdh_last_call_info.restype = ctypes.c_int
    lib.cdh_last_call_info.argtypes = [vp, ctypes.POINTER(ctypes.c_int64)]
    lib.cdh_call_kernel_ms.restype = ctypes.c_int
    lib.cdh_call_kernel_ms.argtypes = [vp, ctypes.c_int, ctypes.POINTER(dbl)]
    lib.cdh_rdf.restype = ctypes.c_int
    lib.cdh_rdf.argtypes = [vp, vp, i32, i32, dbl, i32, vp, dbl, vp, vp]
    lib.cdh_bench_fp32_rate.restype = ctypes.c_int
    lib.cdh_bench_fp32_rate.argtypes = [ctypes.c_int, ctypes.c_int, vp, ctypes.POINTER(dbl), ctypes.POINTER(dbl)]
    lib.cdh_bench_shared_atomics.restype = ctypes.c_int
    lib.cdh_bench_shared_atomics.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, vp, ctypes.c_int, dbl,
                                             ctypes.c_int, ctypes.c_int, ctypes.c_int, vp,
                                             ctypes.POINTER(dbl), ctypes.POINTER(dbl), ctypes.POINTER(dbl)]
    lib.cdh_bench_dsmem_atomics.restype = ctypes.c_int
    lib.cdh_bench_dsmem_atomics.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, vp, ctypes.POINTER(dbl), ctypes.POINTER(dbl)]
    lib.cdh_bench_inner_loop.restype = ctypes.c_int
    lib.cdh_bench_inner_loop.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, vp, ctypes.POINTER(dbl), ctypes.POINTER(dbl)]
    lib.cdh_selftest_sqrt.restype = ctypes.c_int
    lib.cdh_selftest_sqrt.argtypes = [u32, u32, vp, ctypes.POINTER(ctypes.c_uint64)]
    lib.cdh_host_d2_threshold_bits.restype = ctypes.c_uint32
    lib.cdh_host_d2_threshold_bits.argtypes = [ctypes.c_float]
    lib.cdh_host_fused_rint_constant.restype = ctypes.c_int
    lib.cdh_host_fused_rint_constant.argtypes = [ctypes.c_float, ctypes.POINTER(ctypes.c_float)]
    lib.cdh_host_work_items.restype = ctypes.c_int64
    lib.cdh_host_work_items.argtypes = [i32, vp, i32, i32, i32, i32, i32, vp, ctypes.c_int64]
    lib.cdh_selftest_sqrt_f64.restype = ctypes.c_int
    lib.cdh_selftest_sqrt_f64.argtypes = [ctypes.c_uint64, ctypes.c_uint64, vp, ctypes.POINTER(ctypes.c_uint64)]
    if path is None:
        _lib = lib
    return lib


def cdh_strerror(code: int) -> str:
    return load().cdh_strerror(int(code)).decode()


def _ptr(x) -> int:
    """Device/host address of a torch tensor, numpy array or int."""
    if x is None:
        return 0
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return int(x.data_ptr())
    if isinstance(x, np.ndarray):
        return int(x.ctypes.data)
    raise TypeError(f"cannot take the address of {type(x)}")


def _check_device_tensor(x, what: str, device: int, dtype_name: str, min_numel: int) -> None:
    """A torch tensor handed to a device entry point must be what the C call will read or write: CUDA memory of the
    context's device, contiguous, of the precision's element type and large enough.  Raw integer pointers pass
    through unchecked (the caller vouches for them)."""
    if x is None or isinstance(x, int) or not hasattr(x, "data_ptr"):
        return
    if not getattr(x, "is_cuda", False):
        raise ValueError(f"{what} must be a CUDA tensor (cdh_histograms_host takes host buffers)")
    if x.device.index != device:
        raise ValueError(f"{what} lives on cuda:{x.device.index}, the context on cuda:{device}")
    if not x.is_contiguous():
        raise ValueError(f"{what} must be contiguous")
    if str(x.dtype).replace("torch.", "") not in dtype_name.split("|"):
        raise ValueError(f"{what} must have dtype {dtype_name}, not {x.dtype}")
    if x.numel() < min_numel:
        raise ValueError(f"{what} has {x.numel()} elements, the call needs {min_numel}")


def _stream_ptr(stream) -> int:
    if stream is None:
        return 0
    if isinstance(stream, int):
        return stream
    return int(stream.cuda_stream)          # torch.cuda.Stream


class Context:
    """Owns one ``cdh_ctx`` (device scratch).  One per device; not thread-safe."""

    def __init__(self, device: int = 0, flags: int = 0):
        self._lib = load()
        h = ctypes.c_void_p()
        rc = self._lib.cdh_create(ctypes.byref(h), int(device), int(flags))
        if rc != OK:
            raise CdhError(rc, cdh_strerror(rc))
        self._h = h
        self.device = int(device)

    def _check(self, rc: int):
        if rc != OK:
            detail = self._lib.cdh_last_error(self._h).decode() if self._h else ""
            raise CdhError(rc, cdh_strerror(rc) + (f" [{detail}]" if detail else ""))

    def _marshal(self, species_offsets, box, n_frames):
        off = np.ascontiguousarray(species_offsets, dtype=np.int32)
        if box is None:
            b, n_boxes = None, 0
        else:
            b = np.ascontiguousarray(box, dtype=np.float64).reshape(-1, 9)
            n_boxes = int(b.shape[0])
        return off, b, n_boxes

    def cdh_histograms(self, coords, n_frames: int, species_offsets: Sequence[int], box_type: int,
                       box, r_max: float, n_bins: int, out, precision: int = F32, stream=None) -> None:
        """include/cdh.h ``cdh_histograms``: coords / out are DEVICE buffers (torch CUDA tensors or ints).
        Asynchronous on ``stream``."""
        off, b, n_boxes = self._marshal(species_offsets, box, n_frames)
        n_species = len(off) - 1
        _check_device_tensor(coords, "coords", self.device, "float64" if precision == F64 else "float32",
                             int(n_frames) * int(off[-1]) * 3)
        _check_device_tensor(out, "out", self.device, "int64|uint64", n_species * (n_species + 1) // 2 * int(n_bins))
        rc = self._lib.cdh_histograms(self._h, _ptr(coords), int(n_frames), off.ctypes.data, len(off) - 1,
                                      int(box_type), None if b is None else b.ctypes.data, n_boxes,
                                      float(r_max), int(n_bins), int(precision), _stream_ptr(stream), _ptr(out))
        self._check(rc)

    def cdh_histograms_host(self, coords: np.ndarray, species_offsets: Sequence[int], box_type: int, box,
                            r_max: float, n_bins: int, precision: int = F32, stream=None,
                            out: Optional[np.ndarray] = None) -> np.ndarray:
        """include/cdh.h ``cdh_histograms_host``: HOST numpy coords [n_frames, n_total, 3] -> HOST uint64
        [n_hist, n_bins]; H2D, kernels and D2H inside the call; synchronises ``stream``."""
        c = np.ascontiguousarray(coords)
        if c.ndim == 2:
            c = c[None]
        want = np.float64 if precision == F64 else np.float32
        if c.dtype != want or c.ndim != 3 or c.shape[2] != 3:
            raise ValueError(f"coords must be {np.dtype(want).name} [n_frames, n_total, 3] for this precision")
        off, b, n_boxes = self._marshal(species_offsets, box, c.shape[0])
        n_species = len(off) - 1
        n_hist = n_species * (n_species + 1) // 2
        if out is None:
            out = np.empty((n_hist, int(n_bins)), dtype=np.uint64)
        rc = self._lib.cdh_histograms_host(self._h, c.ctypes.data, int(c.shape[0]), off.ctypes.data, n_species,
                                           int(box_type), None if b is None else b.ctypes.data, n_boxes,
                                           float(r_max), int(n_bins), int(precision), _stream_ptr(stream),
                                           out.ctypes.data)
        self._check(rc)
        return out

    def cdh_histograms_stream(self, coords: np.ndarray, species_offsets: Sequence[int], box_type: int, box,
                              r_max: float, n_bins: int, precision: int = F32, frames_per_chunk: int = 0,
                              stream=None, out: Optional[np.ndarray] = None) -> np.ndarray:
        """include/cdh.h ``cdh_histograms_stream``: HOST coords [n_frames, n_total, 3] (numpy, or a pinned CPU torch
        tensor for overlapped copies) -> HOST uint64 [n_hist, n_bins]; frames go to the device chunk by chunk."""
        want = np.float64 if precision == F64 else np.float32
        if hasattr(coords, "data_ptr"):                      # torch tensor (pinned host memory)
            if coords.is_cuda or not coords.is_contiguous():
                raise ValueError("coords must be a contiguous CPU tensor")
            shape, dt, addr = tuple(coords.shape), np.dtype(str(coords.dtype).replace("torch.", "")), coords.data_ptr()
        else:
            coords = np.ascontiguousarray(coords)
            shape, dt, addr = coords.shape, coords.dtype, coords.ctypes.data
        if dt != want or len(shape) != 3 or shape[2] != 3:
            raise ValueError(f"coords must be {np.dtype(want).name} [n_frames, n_total, 3] for this precision")
        off, b, n_boxes = self._marshal(species_offsets, box, shape[0])
        n_species = len(off) - 1
        n_hist = n_species * (n_species + 1) // 2
        if out is None:
            out = np.empty((n_hist, int(n_bins)), dtype=np.uint64)
        rc = self._lib.cdh_histograms_stream(self._h, addr, int(shape[0]), off.ctypes.data, n_species,
                                             int(box_type), None if b is None else b.ctypes.data, n_boxes,
                                             float(r_max), int(n_bins), int(precision), int(frames_per_chunk),
                                             _stream_ptr(stream), out.ctypes.data)
        self._check(rc)
        return out

    def cdh_rdf(self, hist, n_hist: int, n_bins: int, r_max: float, n_frames: int, n_pairs, volume: float, g,
                stream=None) -> None:
        """include/cdh.h ``cdh_rdf``: hist (uint64) and g (float64) are DEVICE buffers [n_hist, n_bins]."""
        npairs = np.ascontiguousarray(n_pairs, dtype=np.float64).reshape(-1)
        if npairs.shape[0] != int(n_hist):
            raise ValueError("one pair count per histogram row")
        _check_device_tensor(hist, "hist", self.device, "int64|uint64", int(n_hist) * int(n_bins))
        _check_device_tensor(g, "g", self.device, "float64", int(n_hist) * int(n_bins))
        rc = self._lib.cdh_rdf(self._h, _ptr(hist), int(n_hist), int(n_bins), float(r_max), int(n_frames),
                               npairs.ctypes.data, float(volume), _stream_ptr(stream), _ptr(g))
        self._check(rc)

    def last_call_info(self) -> dict:
        arr = (ctypes.c_int64 * 8)()
        self._check(self._lib.cdh_last_call_info(self._h, arr))
        v = list(arr)
        return {"launches": v[0], "items": v[1], "sweeps": v[2], "ctas": v[3], "threads": v[4],
                "smem_bytes": v[5], "variant": v[6], "tj": v[6] >> 16, "fast": bool(v[6] & 1), "global_hist": bool(v[6] & 4), "hybrid": bool(v[6] & 8), "form": (v[6] >> 8) & 15, "skip": bool(v[6] & (1 << 14)), "full_range": bool(v[6] & (1 << 15)),
                "padded_pairs": v[7]}

    def call_kernel_ms(self, calls_back: int = 0):
        """(tile kernel ms, whole call ms) of a recent call (0 = last); needs FLAG_TIME_KERNELS; waits for it."""
        arr = (ctypes.c_double * 2)()
        self._check(self._lib.cdh_call_kernel_ms(self._h, int(calls_back), arr))
        return float(arr[0]), float(arr[1])

    def cdh_destroy(self) -> None:
        if self._h:
            self._lib.cdh_destroy(self._h)
            self._h = None

    close = cdh_destroy

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.cdh_destroy()

    def __del__(self):
        try:
            self.cdh_destroy()
        except Exception:
            pass


def cdh_create(device: int = 0, flags: int = 0) -> Context:
    return Context(device, flags)


# ---- microbenchmarks (include/cdh_bench.h) ---------------------------------------------------------
def cdh_bench_fp32_rate(kind: int, iters: int = 2048, stream=None):
    lib = load()
    r, ms = ctypes.c_double(), ctypes.c_double()
    rc = lib.cdh_bench_fp32_rate(int(kind), int(iters), _stream_ptr(stream), ctypes.byref(r), ctypes.byref(ms))
    if rc != OK:
        raise CdhError(rc, cdh_strerror(rc))
    return r.value, ms.value


def cdh_bench_shared_atomics(pattern: int, op: int, n_bins: int, samples=None, n_samples: int = 0,
                             active_fraction: float = 1.0, threads: int = 512, ctas_per_sm: int = 1,
                             iters: int = 4096, stream=None):
    lib = load()
    r, ms, ms0 = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
    rc = lib.cdh_bench_shared_atomics(int(pattern), int(op), int(n_bins), _ptr(samples), int(n_samples),
                                      float(active_fraction), int(threads), int(ctas_per_sm), int(iters),
                                      _stream_ptr(stream), ctypes.byref(r), ctypes.byref(ms), ctypes.byref(ms0))
    if rc != OK:
        raise CdhError(rc, cdh_strerror(rc))
    return r.value, ms.value, ms0.value


NOALLOC_MAX_PADDED_PARTICLES = 131072
NOALLOC_MAX_BINS = 32768


def cdh_histograms_noalloc(device: int, coords, n_frames: int, species_offsets: Sequence[int], box_type: int, box,
                           r_max: float, n_bins: int, out, stream=None) -> None:
    """include/cdh.h ``cdh_histograms_noalloc``: ``cdh_histograms`` (CDH_F32) without a context and without any
    allocation -- the scratch is a static device array inside the library, shared by all calls on the device (calls that
    overlap on the GPU race).  coords / out are DEVICE buffers (torch CUDA tensors or ints).  Asynchronous on ``stream``."""
    lib = load()
    off = np.ascontiguousarray(species_offsets, dtype=np.int32)
    n_species = len(off) - 1
    if box is None:
        b, n_boxes = None, 0
    else:
        b = np.ascontiguousarray(box, dtype=np.float64).reshape(-1, 9)
        n_boxes = int(b.shape[0])
    _check_device_tensor(coords, "coords", int(device), "float32", int(n_frames) * int(off[-1]) * 3)
    _check_device_tensor(out, "out", int(device), "int64|uint64", n_species * (n_species + 1) // 2 * int(n_bins))
    rc = lib.cdh_histograms_noalloc(int(device), _ptr(coords), int(n_frames), off.ctypes.data, n_species, int(box_type),
                                    None if b is None else b.ctypes.data, n_boxes, float(r_max), int(n_bins),
                                    _stream_ptr(stream), _ptr(out))
    if rc != OK:
        detail = lib.cdh_noalloc_last_error().decode()
        raise CdhError(rc, cdh_strerror(rc) + (f" [{detail}]" if detail else ""))


def cdh_bench_dsmem_atomics(cluster_size: int, bins_per_cta: int = 25000, iters: int = 512, stream=None):
    """include/cdh_bench.h ``cdh_bench_dsmem_atomics``: (updates per second, kernel ms) of cluster-distributed shared atomics."""
    lib = load()
    r, ms = ctypes.c_double(), ctypes.c_double()
    rc = lib.cdh_bench_dsmem_atomics(int(cluster_size), int(bins_per_cta), int(iters), _stream_ptr(stream), ctypes.byref(r), ctypes.byref(ms))
    if rc != OK:
        raise CdhError(rc, cdh_strerror(rc))
    return r.value, ms.value


def cdh_bench_inner_loop(box: int, level: int, free_alu: int = 0, iters: int = 40, stream=None):
    """include/cdh_bench.h ``cdh_bench_inner_loop``: (pairs per second, kernel ms) of one layer of the tile kernel's inner loop."""
    lib = load()
    r, ms = ctypes.c_double(), ctypes.c_double()
    rc = lib.cdh_bench_inner_loop(int(box), int(level), int(free_alu), int(iters), _stream_ptr(stream), ctypes.byref(r), ctypes.byref(ms))
    if rc != OK:
        raise CdhError(rc, cdh_strerror(rc))
    return r.value, ms.value


def cdh_selftest_sqrt(first_bits: int = 0x0D800000, last_bits: int = 0x7F7FFFFF, stream=None) -> int:
    lib = load()
    bad = ctypes.c_uint64()
    rc = lib.cdh_selftest_sqrt(int(first_bits), int(last_bits), _stream_ptr(stream), ctypes.byref(bad))
    if rc != OK:
        raise CdhError(rc, cdh_strerror(rc))
    return int(bad.value)


def cdh_selftest_sqrt_f64(seed: int = 1808, count: int = 1 << 32, stream=None) -> int:
    lib = load()
    bad = ctypes.c_uint64()
    rc = lib.cdh_selftest_sqrt_f64(int(seed), int(count), _stream_ptr(stream), ctypes.byref(bad))
    if rc != OK:
        raise CdhError(rc, cdh_strerror(rc))
    return int(bad.value)
