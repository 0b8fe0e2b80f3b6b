"""Seeded synthetic workloads (numpy only; none of the method's arithmetic lives here).

This module is the ONE piece shared by the oracle-side tests and the CUDA-side tests and
bench: it only produces coefficient rows.  The five workloads are BASELINE.json's
`configs`; they stand in for the paper's own workload -- the enumeration of reduced
polynomials P~'_d(F_q) at q < 300 (g=2), q < 50 (g=3), q < 15 (g=4), PAPER.md:13, 113-121 --
whose data set is not available.  Recipe:

  row i, slot j:  u = mix64(seed, i, j)              (SplitMix64 finaliser, counter based)
                  c_j = ((u >> 32) * q) >> 32        uniform on [0, q)
  degree bit      b = mix64(seed, i, 2g+3) >> 63     (configs 3-5: degree 2g+1 / 2g+2, 50/50)
  b = 1:  c_{2g+2} = 1 + (((u >> 32) * (q-1)) >> 32)                     (nonzero)
  b = 0:  c_{2g+2} = 0 and c_{2g+1} = 1 + (((u >> 32) * (q-1)) >> 32)    (nonzero)

Rows are coeffs[i][j] = coefficient of X^j as the standard integer encoding of F_q
(sum a_i p^i <-> sum a_i T^i mod R_q; the plain residue for prime q), dtype uint16.
Any row can be regenerated from its index alone, on any rank.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


@dataclass(frozen=True)
class Workload:
    name: str
    q: int
    p: int
    r: int
    g: int
    n: int
    seed: int
    degree_mode: str          # "exhaustive" | "even" (always 2g+2) | "mixed" (50/50)
    histogram: bool = False

    @property
    def ncoef(self) -> int:
        return 2 * self.g + 3

    @property
    def xevals_per_curve(self) -> int:
        """sum_{k=1..g} q^k -- every x in F_{q^k}, x = 0 included."""
        return sum(self.q ** k for k in range(1, self.g + 1))


CONFIGS = {
    1: Workload("c1_q3_g2_exhaustive", 3, 3, 1, 2, 1944, 0, "exhaustive"),
    2: Workload("c2_q25_g2", 25, 5, 2, 2, 1 << 20, 0x1805119910000002, "even"),
    3: Workload("c3_q49_g3", 49, 7, 2, 3, 1 << 22, 0x1805119910000003, "mixed"),
    4: Workload("c4_q13_g4", 13, 13, 1, 4, 1 << 24, 0x1805119910000004, "mixed"),
    5: Workload("c5_q293_g2", 293, 293, 1, 2, 1 << 24, 0x1805119910000005, "mixed", histogram=True),
}


def mix64(seed: int, i, j) -> np.ndarray:
    """SplitMix64-style finaliser of the counter (seed, i, j); i, j broadcastable arrays."""
    with np.errstate(over="ignore"):
        i = np.asarray(i, dtype=np.uint64)
        j = np.asarray(j, dtype=np.uint64)
        z = np.uint64(seed) ^ (i * np.uint64(0x9E3779B97F4A7C15)) ^ ((j + np.uint64(1)) * np.uint64(0xD1B54A32D192ED03))
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return z


def _scale(u: np.ndarray, m: int) -> np.ndarray:
    return ((u >> np.uint64(32)) * np.uint64(m)) >> np.uint64(32)


def _exhaustive_q3_g2() -> np.ndarray:
    """All f in F_3[x] of degree 5 (486) then degree 6 (1458), base-3 counting order."""
    rows = []
    for top in (5, 6):
        cnt = 3 ** (top + 1)
        e = np.arange(cnt, dtype=np.int64)
        digs = np.zeros((cnt, 7), dtype=np.uint16)
        v = e.copy()
        for j in range(top + 1):
            digs[:, j] = v % 3
            v //= 3
        rows.append(digs[digs[:, top] != 0])
    return np.concatenate(rows, axis=0)


def rows_by_index(cfg: Workload, idx) -> np.ndarray:
    """Coefficient rows of workload `cfg` at the given row indices (any order)."""
    idx = np.asarray(idx, dtype=np.uint64)
    if cfg.degree_mode == "exhaustive":
        return _exhaustive_q3_g2()[idx.astype(np.int64)]
    nc = cfg.ncoef
    j = np.arange(nc, dtype=np.uint64)[None, :]
    u = mix64(cfg.seed, idx[:, None], j)
    c = _scale(u, cfg.q).astype(np.uint16)
    nz = (1 + _scale(u, cfg.q - 1)).astype(np.uint16)
    if cfg.degree_mode == "even":
        c[:, nc - 1] = nz[:, nc - 1]
    else:
        b = (mix64(cfg.seed, idx, np.uint64(nc)) >> np.uint64(63)).astype(bool)
        c[:, nc - 1] = np.where(b, nz[:, nc - 1], 0)
        c[:, nc - 2] = np.where(b, c[:, nc - 2], nz[:, nc - 2])
    return c


def generate(cfg: Workload, start: int = 0, count: int | None = None, chunk: int = 1 << 20) -> np.ndarray:
    """Rows start .. start+count-1 of workload `cfg` (default: all of it)."""
    count = cfg.n - start if count is None else count
    if cfg.degree_mode == "exhaustive":
        return _exhaustive_q3_g2()[start:start + count]
    out = np.empty((count, cfg.ncoef), dtype=np.uint16)
    for s in range(0, count, chunk):
        e = min(count, s + chunk)
        out[s:e] = rows_by_index(cfg, np.arange(start + s, start + e, dtype=np.uint64))
    return out


def sample_indices(cfg: Workload, S: int, edge: int = 8) -> np.ndarray:
    """Deterministic subsample for oracle parity at full size: every (n/S)-th index plus the
    first and last `edge` rows."""
    if S >= cfg.n:
        return np.arange(cfg.n, dtype=np.int64)
    stride = np.arange(S, dtype=np.int64) * (cfg.n // S)
    head = np.arange(min(edge, cfg.n), dtype=np.int64)
    tail = np.arange(max(0, cfg.n - edge), cfg.n, dtype=np.int64)
    return np.unique(np.concatenate([head, stride, tail]))


def shard_range(n: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous curve range [lo, hi) of rank `rank` out of `world`."""
    base, rem = divmod(n, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def edge_rows(q: int, g: int) -> np.ndarray:
    """Structured rows exercising the degenerate cases (patterns only, no field arithmetic):
    x^{2g+1}; c*x^{2g+2} for every nonzero c (capped); zero-heavy rows; c_0 = 0 rows;
    both degree parities; all-(q-1) rows."""
    nc = 2 * g + 3
    rows = []
    r = np.zeros(nc, dtype=np.uint16); r[nc - 2] = 1; rows.append(r)             # x^{2g+1}
    for c in range(1, min(q, 40)):
        r = np.zeros(nc, dtype=np.uint16); r[nc - 1] = c; rows.append(r)          # c x^{2g+2}
    for c in range(1, min(q, 6)):
        r = np.zeros(nc, dtype=np.uint16); r[nc - 2] = c; r[0] = 1; rows.append(r)  # c x^{2g+1} + 1
        r = np.zeros(nc, dtype=np.uint16); r[nc - 1] = 1; r[1] = c; rows.append(r)  # x^{2g+2} + c x
        r = np.zeros(nc, dtype=np.uint16); r[nc - 1] = c; r[nc - 2] = 1; r[2] = 1; rows.append(r)
    r = np.full(nc, q - 1, dtype=np.uint16); rows.append(r)
    r = np.full(nc, q - 1, dtype=np.uint16); r[nc - 1] = 0; rows.append(r)
    r = np.full(nc, 1, dtype=np.uint16); r[0] = 0; rows.append(r)
    r = np.full(nc, 1, dtype=np.uint16); r[0] = 0; r[1] = 0; r[nc - 1] = 0; rows.append(r)
    return np.stack(rows)
