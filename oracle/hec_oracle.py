"""TEST INFRASTRUCTURE ONLY -- ctypes front end of oracle/hec_oracle.c.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It imports nothing from paper_1805_11991_b200 and the
CUDA path imports nothing from here.

The arithmetic lives in hec_oracle.c (polynomial-basis F_{q^k}, Horner at every x,
Euler's criterion, Euclid for gcd(f, f')).  This file
only compiles it, marshals arrays and adds the histogram oracle, which is the plain
definition "sort the rows, run-length encode" (eq. (1.2) / Algorithm 1
line 20 with m = 1 and without lambda; numpy's sort is the library primitive).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "hec_oracle.c"
_LIB = _HERE / "libhec_oracle.so"
_lib = None


def build(force: bool = False) -> Path:
    """Compile hec_oracle.c with gcc (plain C, OpenMP over curves)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".tmp{os.getpid()}.so")
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fopenmp", "-shared", "-fPIC", "-o", str(tmp), str(_SRC)]
        )
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(str(_LIB))
        u32, u64, sz = ctypes.c_uint32, ctypes.c_uint64, ctypes.c_size_t
        vp = ctypes.c_void_p
        lib.orc_smallest_irreducible.argtypes = [u32, u32, vp]
        lib.orc_smallest_primitive.argtypes = [u32, u32, vp]
        lib.orc_is_primitive.argtypes = [u32, u32, vp]
        lib.orc_mul_encoded.argtypes = [u32, u32, vp, u64, u64]
        lib.orc_mul_encoded.restype = ctypes.c_int64
        lib.orc_count_range.argtypes = [u32, u32, u32, vp, sz, u32, u32, u32, vp, vp, ctypes.c_int, vp]
        lib.orc_roots_range.argtypes = [u32, u32, u32, vp, sz, u32, u32, u32, vp, ctypes.c_int]
        _lib = lib
    return _lib


def _factor_prime_power(q: int) -> tuple[int, int]:
    """q = p^r with p an odd prime (trial division; q is tiny)."""
    for p in range(3, q + 1, 2):
        if q % p == 0:
            r, v = 0, q
            while v % p == 0:
                v //= p
                r += 1
            if v != 1:
                break
            return p, r
    raise ValueError(f"q={q} is not an odd prime power")


def smallest_irreducible(p: int, n: int) -> list[int]:
    """Coefficients [a_0..a_{n-1}, 1] of the lexicographically smallest monic irreducible."""
    out = (ctypes.c_uint32 * (n + 1))()
    if _load().orc_smallest_irreducible(p, n, out):
        raise ValueError("no irreducible found")
    return list(out)


def smallest_primitive(p: int, n: int) -> list[int]:
    """Coefficients [a_0..a_{n-1}, 1] of the lexicographically smallest monic primitive
    polynomial (reading G7 in DESIGN.md)."""
    out = (ctypes.c_uint32 * (n + 1))()
    if _load().orc_smallest_primitive(p, n, out):
        raise ValueError("no primitive polynomial found")
    return list(out)


def is_primitive(p: int, mod: list[int]) -> bool:
    n = len(mod) - 1
    arr = (ctypes.c_uint32 * (n + 1))(*mod)
    return _load().orc_is_primitive(p, n, arr) == 1


def mul_encoded(p: int, mod: list[int], a: int, b: int) -> int:
    """Product in F_p[t]/(mod) of two elements given as integers sum a_i p^i."""
    n = len(mod) - 1
    arr = (ctypes.c_uint32 * (n + 1))(*mod)
    v = _load().orc_mul_encoded(p, n, arr, a, b)
    if v < 0:
        raise ValueError("bad modulus")
    return int(v)


def count(q: int, g: int, coeffs, k_lo: int = 1, k_hi: int | None = None, nthreads: int = 0,
          want_squarefree: bool = True):
    """(N_1..N_g) and the squarefree flag for each row of coeffs[n][2g+3] (uint16).

    Returns (counts uint32 [n][max(g, k_hi)], squarefree uint8 [n] or None, threads_used).
    Columns outside k_lo..k_hi are left 0.  k_hi > g asks for N_k beyond the genus (the
    formula of PAPER.md:41 holds for every extension E); tests use it for Newton-identity pins.
    """
    p, r = _factor_prime_power(q)
    c = np.ascontiguousarray(coeffs, dtype=np.uint16)
    if c.ndim != 2 or c.shape[1] != 2 * g + 3:
        raise ValueError("coeffs must be [n][2g+3]")
    n = c.shape[0]
    k_hi = g if k_hi is None else k_hi
    width = max(g, k_hi)
    out = np.zeros((n, width), dtype=np.uint32)
    sf = np.zeros(n, dtype=np.uint8) if want_squarefree else None
    used = ctypes.c_int(0)
    rc = _load().orc_count_range(
        p, r, g, c.ctypes.data, n, k_lo, k_hi, width, out.ctypes.data,
        sf.ctypes.data if sf is not None else None, nthreads, ctypes.byref(used))
    if rc:
        raise ValueError({-10: "bad field parameters", -11: "coefficient >= q",
                          -12: "degree < 2g+1", -13: "bad k range"}.get(rc, f"error {rc}"))
    return out, sf, used.value


def roots(q: int, g: int, coeffs, k_hi: int | None = None, nthreads: int = 0):
    """r0_k = #{x in F_{q^k}: f(x) = 0} (affine zeros) for k = 1..k_hi (default g): uint32 [n][k_hi]."""
    p, r = _factor_prime_power(q)
    c = np.ascontiguousarray(coeffs, dtype=np.uint16)
    if c.ndim != 2 or c.shape[1] != 2 * g + 3:
        raise ValueError("coeffs must be [n][2g+3]")
    k_hi = g if k_hi is None else k_hi
    out = np.zeros((c.shape[0], k_hi), dtype=np.uint32)
    rc = _load().orc_roots_range(p, r, g, c.ctypes.data, c.shape[0], 1, k_hi, k_hi, out.ctypes.data, nthreads)
    if rc:
        raise ValueError(f"orc_roots_range: error {rc}")
    return out


def histogram(counts, mask=None):
    """Distinct rows of counts[n][g] in ascending lexicographic order + multiplicities.

    Rows with mask == 0 are skipped when a mask is given (the paper's N map only counts
    squarefree f).  Returns (tuples uint32 [m][g], mult uint64 [m]).
    """
    c = np.asarray(counts, dtype=np.uint32)
    if mask is not None:
        c = c[np.asarray(mask) != 0]
    if c.shape[0] == 0:
        return np.zeros((0, c.shape[1]), dtype=np.uint32), np.zeros(0, dtype=np.uint64)
    tup, mult = np.unique(c, axis=0, return_counts=True)
    return tup.astype(np.uint32), mult.astype(np.uint64)
