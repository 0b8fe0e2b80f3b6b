"""Thin ctypes binding of libhec.so (include/hec.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  There is no CPU fallback: if
libhec.so is missing the first call raises, and on a box without a GPU `count`,
`histogram` and `gather_bench` raise HecError(HEC_ERR_CUDA) (only `build_field`, which is
host code by design, works without a device).  Arrays may be numpy arrays (host pointers)
or torch CUDA tensors (device pointers, passed as data_ptr()); results come back the
same way.
"""
from __future__ import annotations

import ctypes
from pathlib import Path

import numpy as np

_PKG = Path(__file__).resolve().parent
LIB_PATH = _PKG / "libhec.so"
_lib = None
_cap_hint: dict = {}     # (n, g, merge?) -> distinct tuples of the last histogram call of that shape

HEC_OK = 0
HEC_ERR_INVALID_FIELD, HEC_ERR_INVALID_ARG, HEC_ERR_COEFF_RANGE, HEC_ERR_DEGREE = -1, -2, -3, -4
HEC_ERR_CAPACITY, HEC_ERR_UNSUPPORTED, HEC_ERR_CUDA, HEC_ERR_NOMEM = -5, -6, -7, -8
REGIME_AUTO, REGIME_SMEM, REGIME_L2, REGIME_SMEM_HALF = 0, 1, 2, 3
EVAL_AUTO, EVAL_HORNER, EVAL_RADIX2, EVAL_RADIX4, EVAL_RADIX8, EVAL_ORBIT = 0, 1, 2, 4, 8, 16
TABLE_MODES = {0: "global32-extended", 1: "smem16-extended", 2: "smem32-half", 3: "smem16+8-half",
               4: "smem2x16-pair", 5: "smem32-rhalf", 6: "smem16+1-rhalf", 7: "global2x32-pair", 8: "smem2x16-pair-scalar"}
MAX_GENUS = 5

# every symbol include/hec.h declares (tests check the library exports all of them)
SYMBOLS = [
    "hec_last_error", "hec_last_error_index", "hec_build_field", "hec_build_field_device", "hec_free_field", "hec_field_p",
    "hec_field_degree", "hec_field_q", "hec_field_Q", "hec_field_embed_unit", "hec_field_modulus",
    "hec_field_antilog", "hec_field_log", "hec_field_zech", "hec_field_embed", "hec_count", "hec_histogram",
    "hec_histogram_merge", "hec_histogram_static", "hec_reduced_total", "hec_reduced_rows", "hec_curve_map",
    "hec_count_ex", "hec_lambda_partitions", "hec_curve_map_lambda", "hec_set_map_chunk_rows", "hec_curve_map_range", "hec_curve_map_all", "hec_set_shift", "hec_shift_rows", "hec_set_fast_tables", "hec_count_histogram", "hec_set_field_variant",
    "hec_set_stream", "hec_set_regime", "hec_set_eval", "hec_last_count_stats", "hec_launch_count", "hec_gather_bench",
    "hec_shutdown",
]


class HecError(RuntimeError):
    def __init__(self, code: int, msg: str, index: int | None = None):
        super().__init__(f"libhec error {code}: {msg}" + (f" (row {index})" if index is not None else ""))
        self.code, self.index = code, index


class CountStats(ctypes.Structure):
    _fields_ = [("count_kernel_ms", ctypes.c_float), ("squarefree_kernel_ms", ctypes.c_float),
                ("launches", ctypes.c_uint32), ("regime", ctypes.c_uint32), ("smem_bytes", ctypes.c_uint32),
                ("grid", ctypes.c_uint32), ("block", ctypes.c_uint32), ("chains_per_lane", ctypes.c_uint32),
                ("table_mode", ctypes.c_uint32), ("radix_fields", ctypes.c_uint32), ("splits", ctypes.c_uint32),
                ("fast_fields", ctypes.c_uint32), ("chunks", ctypes.c_uint32)]


def lib():
    """Load libhec.so (built in-tree by paper_1805_11991_b200/build.py); fail loudly if absent."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise ImportError(f"{LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                              "(nvcc, sm_100a). libhec has no CPU fallback.")
        L = ctypes.CDLL(str(LIB_PATH))
        u32, vp, sz = ctypes.c_uint32, ctypes.c_void_p, ctypes.c_size_t
        L.hec_last_error.restype = ctypes.c_char_p
        L.hec_last_error_index.restype = sz
        L.hec_build_field.restype = vp
        L.hec_build_field.argtypes = [u32, u32, u32]
        L.hec_build_field_device.restype = vp
        L.hec_build_field_device.argtypes = [u32, u32, u32]
        L.hec_free_field.argtypes = [vp]
        for name in ("p", "degree", "q", "Q", "embed_unit"):
            f = getattr(L, f"hec_field_{name}")
            f.restype, f.argtypes = u32, [vp]
        for name in ("modulus", "antilog", "log", "zech", "embed"):
            f = getattr(L, f"hec_field_{name}")
            f.restype, f.argtypes = None, [vp, vp]
        L.hec_count.argtypes = [u32, u32, vp, sz, vp, vp]
        L.hec_histogram.argtypes = [vp, vp, sz, u32, vp, vp, sz, ctypes.POINTER(sz)]
        L.hec_count_histogram.argtypes = [u32, u32, vp, sz, vp, vp, vp, vp, sz, ctypes.POINTER(sz)]
        L.hec_histogram_merge.argtypes = [vp, vp, sz, u32, vp, vp, sz, ctypes.POINTER(sz)]
        L.hec_histogram_static.argtypes = [vp, vp, sz, u32, vp, vp, sz, ctypes.POINTER(sz)]
        L.hec_reduced_total.argtypes = [u32, u32, u32, ctypes.POINTER(ctypes.c_uint64)]
        L.hec_reduced_rows.argtypes = [u32, u32, u32, ctypes.c_uint64, sz, vp, vp]
        L.hec_curve_map.argtypes = [u32, u32, u32, vp, vp, sz, ctypes.POINTER(sz)]
        L.hec_curve_map_lambda.argtypes = [u32, u32, u32, vp, vp, sz, ctypes.POINTER(sz)]
        L.hec_count_ex.argtypes = [u32, u32, vp, sz, vp, vp, vp, vp]
        L.hec_lambda_partitions.argtypes = [u32, vp, sz, ctypes.POINTER(sz)]
        L.hec_set_map_chunk_rows.argtypes = [sz]
        L.hec_set_shift.argtypes = [ctypes.c_int]
        L.hec_set_fast_tables.argtypes = [ctypes.c_int]
        L.hec_set_field_variant.argtypes = [ctypes.c_uint32]
        L.hec_shift_rows.argtypes = [u32, u32, vp, sz, vp]
        L.hec_curve_map_all.argtypes = [u32, u32, ctypes.c_int, vp, vp, sz, ctypes.POINTER(sz)]
        L.hec_curve_map_range.argtypes = [u32, u32, u32, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_int, vp, vp, sz, ctypes.POINTER(sz)]
        L.hec_set_stream.argtypes = [vp]
        L.hec_set_regime.argtypes = [ctypes.c_int]
        L.hec_set_eval.argtypes = [ctypes.c_int]
        L.hec_last_count_stats.argtypes = [ctypes.POINTER(CountStats)]
        L.hec_launch_count.restype = ctypes.c_uint64
        L.hec_gather_bench.argtypes = [ctypes.c_int, u32, u32, u32, u32, u32, u32,
                                       ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_float)]
        L.hec_shutdown.restype = None
        _lib = L
    return _lib


def _check(rc: int):
    if rc != HEC_OK:
        L = lib()
        idx = L.hec_last_error_index()
        raise HecError(rc, L.hec_last_error().decode(), None if idx == ctypes.c_size_t(-1).value else idx)


def _is_torch(x) -> bool:
    return type(x).__module__.startswith("torch")


def _ptr(x):
    if x is None:
        return None
    return x.data_ptr() if _is_torch(x) else x.ctypes.data


class Field:
    """hec_build_field handle with the read-only accessors of hec.h (paper's conventions)."""

    def __init__(self, p: int, r: int, k: int, device: bool = False):
        L = lib()
        self._h = (L.hec_build_field_device if device else L.hec_build_field)(p, r, k)
        if not self._h:
            raise HecError(HEC_ERR_INVALID_FIELD, L.hec_last_error().decode())
        self.p, self.r, self.k = p, r, k
        self.n = L.hec_field_degree(self._h)
        self.q = L.hec_field_q(self._h)
        self.Q = L.hec_field_Q(self._h)
        self.embed_unit = L.hec_field_embed_unit(self._h)

    def _arr(self, name: str, size: int) -> np.ndarray:
        out = np.empty(size, dtype=np.uint32)
        getattr(lib(), f"hec_field_{name}")(self._h, out.ctypes.data)
        return out

    @property
    def modulus(self):
        return self._arr("modulus", self.n + 1).tolist()

    @property
    def antilog(self):
        return self._arr("antilog", self.Q - 1)

    @property
    def log(self):
        return self._arr("log", self.Q)

    @property
    def zech(self):
        return self._arr("zech", self.Q - 1)

    @property
    def embed(self):
        return self._arr("embed", self.q)

    def close(self):
        if self._h:
            lib().hec_free_field(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def build_field(p: int, r: int, k: int) -> Field:
    return Field(p, r, k)


def build_field_device(p: int, r: int, k: int) -> Field:
    """hec_build_field_device: same tables, built by CUDA kernels on the current stream (needs a GPU)."""
    return Field(p, r, k, device=True)


def set_stream(cuda_stream: int | None):
    """cuda_stream: a cudaStream_t as an integer (e.g. torch.cuda.current_stream().cuda_stream) or None."""
    _check(lib().hec_set_stream(ctypes.c_void_p(cuda_stream or 0)))


def set_regime(regime: int):
    _check(lib().hec_set_regime(regime))


def set_eval(scheme: int):
    _check(lib().hec_set_eval(scheme))


def count(q: int, g: int, coeffs, out_counts=None, out_squarefree=None, want_squarefree: bool = True):
    """hec_count.  coeffs: uint16 [n][2g+3], numpy (host) or torch CUDA tensor (device).
    Returns (counts uint32-valued [n][g], squarefree uint8 [n] or None) of the same kind as coeffs
    (torch has no uint32 arithmetic: device counts come back as an int32 tensor holding the same bits)."""
    n = int(coeffs.shape[0])
    if tuple(coeffs.shape[1:]) != (2 * g + 3,):
        raise ValueError("coeffs must be [n][2g+3]")
    if _is_torch(coeffs):
        import torch
        if coeffs.dtype not in (torch.uint16, torch.int16) or not coeffs.is_contiguous():
            raise ValueError("device coeffs must be a contiguous uint16/int16 tensor")
        if out_counts is None:
            out_counts = torch.empty((n, g), dtype=torch.int32, device=coeffs.device)
        if out_squarefree is None and want_squarefree:
            out_squarefree = torch.empty((n,), dtype=torch.uint8, device=coeffs.device)
    else:
        coeffs = np.ascontiguousarray(coeffs, dtype=np.uint16)
        if out_counts is None:
            out_counts = np.empty((n, g), dtype=np.uint32)
        if out_squarefree is None and want_squarefree:
            out_squarefree = np.empty((n,), dtype=np.uint8)
    _check(lib().hec_count(q, g, _ptr(coeffs), n, _ptr(out_counts), _ptr(out_squarefree)))
    return out_counts, out_squarefree


def histogram(counts, mask=None, _weights=None):
    """hec_histogram with the two-call pattern.  Returns (tuples [m][g], multiplicities [m])."""
    n, g = int(counts.shape[0]), int(counts.shape[1])
    L = lib()
    m = ctypes.c_size_t(0)
    if not _is_torch(counts):
        counts = np.ascontiguousarray(counts, dtype=np.uint32)
    if _weights is not None:
        def call(*a):
            return L.hec_histogram_merge(_ptr(counts), _ptr(_weights), n, g, *a)
    else:
        def call(*a):
            return L.hec_histogram(_ptr(counts), _ptr(mask), n, g, *a)
    def buffers(cap):
        if _is_torch(counts):
            import torch
            return (torch.empty((cap, g), dtype=torch.int32, device=counts.device),
                    torch.empty((cap,), dtype=torch.int64, device=counts.device))
        return np.empty((cap, g), dtype=np.uint32), np.empty((cap,), dtype=np.uint64)

    # Capacity protocol of hec.h.  A repeated call on a batch of the same shape first tries the capacity the
    # last one needed (+25 %), so the steady state is ONE library call; otherwise size with cap = 0 first.
    key = (n, g, _weights is not None)
    hint = _cap_hint.get(key)
    if hint is None:
        rc = call(None, None, 0, ctypes.byref(m))
        if rc not in (HEC_OK, HEC_ERR_CAPACITY):
            _check(rc)
        cap = m.value
    else:
        cap = min(n, hint + hint // 4 + 1024)
    tup, mult = buffers(cap)
    if cap:
        rc = call(_ptr(tup), _ptr(mult), cap, ctypes.byref(m))
        if rc == HEC_ERR_CAPACITY:
            cap = m.value
            tup, mult = buffers(cap)
            rc = call(_ptr(tup), _ptr(mult), cap, ctypes.byref(m))
        _check(rc)
    _cap_hint[key] = m.value
    return tup[: m.value], mult[: m.value]


def count_histogram(q: int, g: int, coeffs, out_counts=None, out_squarefree=None, want_squarefree: bool = True,
                    out_tuples=None, out_mult=None):
    """hec_count_histogram: one pass of the whole hot path in one library call.  Returns (counts, squarefree, tuples,
    multiplicities), all of the same kind as coeffs (numpy: host; torch CUDA tensor: device).  out_tuples [cap][g] /
    out_mult [cap]: caller-owned result buffers (e.g. pinned host memory), used when their capacity suffices."""
    n = int(coeffs.shape[0])
    if tuple(coeffs.shape[1:]) != (2 * g + 3,):
        raise ValueError("coeffs must be [n][2g+3]")
    dev = _is_torch(coeffs)
    if dev:
        import torch
        if coeffs.dtype not in (torch.uint16, torch.int16) or not coeffs.is_contiguous():
            raise ValueError("device coeffs must be a contiguous uint16/int16 tensor")
        if out_counts is None:
            out_counts = torch.empty((n, g), dtype=torch.int32, device=coeffs.device)
        if out_squarefree is None and want_squarefree:
            out_squarefree = torch.empty((n,), dtype=torch.uint8, device=coeffs.device)
    else:
        coeffs = np.ascontiguousarray(coeffs, dtype=np.uint16)
        if out_counts is None:
            out_counts = np.empty((n, g), dtype=np.uint32)
        if out_squarefree is None and want_squarefree:
            out_squarefree = np.empty((n,), dtype=np.uint8)

    def buffers(cap):
        if dev:
            return (torch.empty((cap, g), dtype=torch.int32, device=coeffs.device),
                    torch.empty((cap,), dtype=torch.int64, device=coeffs.device))
        return np.empty((cap, g), dtype=np.uint32), np.empty((cap,), dtype=np.uint64)

    key = (n, g, "count_histogram", q)
    hint = _cap_hint.get(key)
    cap = min(n, hint + hint // 4 + 1024) if hint is not None else min(n, 1 << 20)
    if out_tuples is not None and out_mult is not None:
        tup, mult, cap = out_tuples, out_mult, min(int(out_tuples.shape[0]), int(out_mult.shape[0]))
    else:
        tup, mult = buffers(cap)
    m = ctypes.c_size_t(0)
    rc = lib().hec_count_histogram(q, g, _ptr(coeffs), n, _ptr(out_counts), _ptr(out_squarefree), _ptr(tup), _ptr(mult),
                                   cap, ctypes.byref(m))
    if rc == HEC_ERR_CAPACITY:          # counts and flags are complete: only the histogram is repeated, at the right size
        tup, mult = buffers(m.value)
        rc = lib().hec_histogram(_ptr(out_counts), _ptr(out_squarefree), n, g, _ptr(tup), _ptr(mult), m.value, ctypes.byref(m))
    _check(rc)
    _cap_hint[key] = m.value
    return out_counts, out_squarefree, tup[: m.value], mult[: m.value]


HISTOGRAM_STATIC_MAX_ROWS = 131072   # HEC_HISTOGRAM_STATIC_MAX_ROWS of hec.h


def histogram_static(counts, mask, out_tuples, out_mult):
    """hec_histogram_static: hec_histogram for code that may not allocate device memory -- e.g. inside a process whose
    HBM is already owned by another allocator, or where cudaMalloc's device-wide sync is unwelcome (hec.h has the
    details).  The library works in a fixed 8 MiB device array; this wrapper allocates nothing either: counts
    [n][g] (n <= HISTOGRAM_STATIC_MAX_ROWS), mask [n] or None, and the result buffers out_tuples [cap][g] / out_mult [cap]
    are the caller's CUDA tensors.  Returns m, the number of distinct tuples now in out_tuples[:m] / out_mult[:m];
    raises HecError(HEC_ERR_CAPACITY) if cap < m or n is above the limit.  Calls must not overlap on the GPU."""
    n, g = int(counts.shape[0]), int(counts.shape[1])
    cap = int(out_mult.shape[0])
    if int(out_tuples.shape[0]) != cap:
        raise ValueError("out_tuples and out_mult must have the same capacity")
    m = ctypes.c_size_t(0)
    _check(lib().hec_histogram_static(_ptr(counts), _ptr(mask), n, g, _ptr(out_tuples), _ptr(out_mult), cap, ctypes.byref(m)))
    return int(m.value)


def histogram_merge(tuples, mult):
    """hec_histogram_merge: (tuples [n][g], mult [n]) with repeats -> sorted distinct tuples, summed mult."""
    if not _is_torch(mult):
        mult = np.ascontiguousarray(mult, dtype=np.uint64)
    return histogram(tuples, None, _weights=mult)


def reduced_total(q: int, g: int, d: int) -> int:
    """hec_reduced_total: number of reduced polynomials of degree d (before the squarefree filter)."""
    t = ctypes.c_uint64(0)
    _check(lib().hec_reduced_total(q, g, d, ctypes.byref(t)))
    return int(t.value)


def reduced_rows(q: int, g: int, d: int, first: int, n: int, device=None):
    """hec_reduced_rows: rows [first, first + n) of the enumeration as (coeffs [n][2g+3], mult [n]); numpy arrays,
    or torch tensors on `device` when given."""
    if device is not None:
        import torch
        rows = torch.empty((n, 2 * g + 3), dtype=torch.int16, device=device)
        mult = torch.empty((n,), dtype=torch.int64, device=device)
    else:
        rows = np.empty((n, 2 * g + 3), dtype=np.uint16)
        mult = np.empty((n,), dtype=np.uint64)
    _check(lib().hec_reduced_rows(q, g, d, ctypes.c_uint64(first), ctypes.c_size_t(n), _ptr(rows), _ptr(mult)))
    return rows, mult


def curve_map(q: int, g: int, d: int, with_lambda: bool = False, index_range=None, device: bool = False):
    """hec_curve_map / hec_curve_map_lambda / hec_curve_map_range (two-call capacity protocol): (keys [m][g (+1)] uint32,
    weights [m] uint64) on the host; with_lambda appends the lambda index (see lambda_partitions) as the last key
    column; index_range = (first, n) restricts to those reduced polynomials (one rank's share).
    device=True: the outputs stay on the current CUDA device (int32 / int64 torch tensors holding the same bits)."""
    L = lib()
    if device:
        import torch

        def alloc(cap, cols):
            return (torch.empty((cap, cols), dtype=torch.int32, device="cuda"), torch.empty((cap,), dtype=torch.int64, device="cuda"))
    else:
        def alloc(cap, cols):
            return np.empty((cap, cols), dtype=np.uint32), np.empty((cap,), dtype=np.uint64)
    if index_range is not None:
        first, cnt = index_range

        def fn(q_, g_, d_, *rest):
            return L.hec_curve_map_range(q_, g_, d_, ctypes.c_uint64(first), ctypes.c_uint64(cnt), int(with_lambda), *rest)
    else:
        fn = L.hec_curve_map_lambda if with_lambda else L.hec_curve_map
    cols = g + 1 if with_lambda else g
    m = ctypes.c_size_t(0)
    # Capacity protocol of hec.h.  Every call does the whole computation, so start with a capacity that is almost
    # always enough (at most two keys per reduced polynomial) instead of asking for the size first.
    n_red = index_range[1] if index_range is not None else reduced_total(q, g, d)
    cap = max(1024, min(2 * n_red, 1 << 24))
    tup, w = alloc(cap, cols)
    rc = fn(q, g, d, _ptr(tup), _ptr(w), ctypes.c_size_t(cap), ctypes.byref(m))
    if rc == HEC_ERR_CAPACITY:
        cap = m.value
        tup, w = alloc(cap, cols)
        rc = fn(q, g, d, _ptr(tup), _ptr(w), ctypes.c_size_t(cap), ctypes.byref(m))
    _check(rc)
    if device:
        return tup[: m.value].clone(), w[: m.value].clone()
    return tup[: m.value].copy(), w[: m.value].copy()


def curve_map_all(q: int, g: int, with_lambda: bool = False):
    """hec_curve_map_all: both degrees 2g+1 and 2g+2 merged (Algorithm 1 in full)."""
    L = lib()
    cols = g + 1 if with_lambda else g
    m = ctypes.c_size_t(0)
    cap = max(1024, min(2 * (reduced_total(q, g, 2 * g + 1) + reduced_total(q, g, 2 * g + 2)), 1 << 24))
    tup = np.empty((cap, cols), dtype=np.uint32)
    w = np.empty((cap,), dtype=np.uint64)
    rc = L.hec_curve_map_all(q, g, int(with_lambda), _ptr(tup), _ptr(w), ctypes.c_size_t(cap), ctypes.byref(m))
    if rc == HEC_ERR_CAPACITY:
        cap = m.value
        tup = np.empty((cap, cols), dtype=np.uint32)
        w = np.empty((cap,), dtype=np.uint64)
        rc = L.hec_curve_map_all(q, g, int(with_lambda), _ptr(tup), _ptr(w), ctypes.c_size_t(cap), ctypes.byref(m))
    _check(rc)
    return tup[: m.value].copy(), w[: m.value].copy()


def set_shift(on: bool):
    _check(lib().hec_set_shift(int(on)))


def set_fast_tables(on: bool):
    _check(lib().hec_set_fast_tables(int(on)))


def set_field_variant(v: int):
    """hec_set_field_variant: the library's own fields use the (v+1)-th smallest primitive polynomial (0: the smallest)."""
    _check(lib().hec_set_field_variant(int(v)))


def shift_rows(q: int, g: int, coeffs):
    """hec_shift_rows: the rows hec_count evaluates after its shift pre-pass (same container type as coeffs)."""
    n = int(coeffs.shape[0])
    if _is_torch(coeffs):
        import torch
        out = torch.empty_like(coeffs)
    else:
        coeffs = np.ascontiguousarray(coeffs, dtype=np.uint16)
        out = np.empty_like(coeffs)
    _check(lib().hec_shift_rows(q, g, _ptr(coeffs), n, _ptr(out)))
    return out


def set_map_chunk_rows(rows: int):
    _check(lib().hec_set_map_chunk_rows(rows))


def lambda_partitions(g: int) -> list:
    """hec_lambda_partitions: list of multiplicity vectors (n_1..n_{2g+2}); the position is the lambda index."""
    L = lib()
    m = ctypes.c_size_t(0)
    rc = L.hec_lambda_partitions(g, None, ctypes.c_size_t(0), ctypes.byref(m))
    if rc not in (HEC_OK, HEC_ERR_CAPACITY):
        _check(rc)
    out = np.empty((m.value, 2 * g + 2), dtype=np.uint8)
    _check(L.hec_lambda_partitions(g, out.ctypes.data, ctypes.c_size_t(m.value), ctypes.byref(m)))
    return [tuple(int(v) for v in row) for row in out]


def count_ex(q: int, g: int, coeffs):
    """hec_count_ex with every output: (counts [n][g], squarefree [n], roots [n][g], lambda index [n])."""
    n = int(coeffs.shape[0])
    if _is_torch(coeffs):
        import torch
        dev = coeffs.device
        cnt = torch.empty((n, g), dtype=torch.int32, device=dev)
        sf = torch.empty((n,), dtype=torch.uint8, device=dev)
        r0 = torch.empty((n, g), dtype=torch.int32, device=dev)
        lam = torch.empty((n,), dtype=torch.uint8, device=dev)
    else:
        coeffs = np.ascontiguousarray(coeffs, dtype=np.uint16)
        cnt, sf = np.empty((n, g), dtype=np.uint32), np.empty((n,), dtype=np.uint8)
        r0, lam = np.empty((n, g), dtype=np.uint32), np.empty((n,), dtype=np.uint8)
    _check(lib().hec_count_ex(q, g, _ptr(coeffs), n, _ptr(cnt), _ptr(sf), _ptr(r0), _ptr(lam)))
    return cnt, sf, r0, lam


def last_count_stats() -> dict:
    s = CountStats()
    _check(lib().hec_last_count_stats(ctypes.byref(s)))
    return {name: getattr(s, name) for name, _ in s._fields_}


def launch_count() -> int:
    return int(lib().hec_launch_count())


def gather_bench(where: int, entries: int, entry_bytes: int, block: int = 1024, ctas_per_sm: int = 1,
                 chains: int = 4, lookups_per_lane: int = 4096) -> tuple[float, float]:
    """Returns (lookups per second, kernel ms) of the dependent random-gather micro-benchmark."""
    rate, ms = ctypes.c_double(0), ctypes.c_float(0)
    _check(lib().hec_gather_bench(where, entries, entry_bytes, block, ctas_per_sm, chains, lookups_per_lane,
                                  ctypes.byref(rate), ctypes.byref(ms)))
    return rate.value, ms.value


def shutdown():
    lib().hec_shutdown()
