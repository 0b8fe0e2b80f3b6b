"""TEST INFRASTRUCTURE ONLY -- oracle for SURVEY.md 8(f) NEXT-1: the curve-count map of Algorithm 1 without lambda.

What it defines (eq. (1.2) with the partition dropped): for fixed q, g and d in {2g+1, 2g+2}

    N_{g,d}(t) = #{ f in P_d(F_q) : (N_1(f), .., N_g(f)) = t },   P_d = squarefree polynomials of degree d,

with N_k(f) = #C_f(F_{q^k}).  Two independent ways to get it:

  * brute_force_map(q, g, d): the definition written out -- EVERY polynomial of degree d, oracle counts,
    squarefree filter, sort + run-length.  Only for tiny q (q^(d+1) rows).
  * reduced_map(q, g, d): Algorithm 1 step by step -- enumerate the reduced polynomials
    P~'_d(F_q) of sections 1.2-1.3, count each once, add mult(f) at its tuple and at the tuple
    of its quadratic twist (lines 19-21).

Readings (the printed text is garbled here):
  * G9   "i := inf{..}, j := inf{..}" must be sup: i = largest index below d with c_i != 0, j = the next one below i.
  * G8   the twist is n f, n a non-square of F_q (not f(-X)); it maps N_k to 2 q^k + 2 - N_k for odd k and fixes
         N_k for even k (line 21 as printed, a_k -> 1 + q^k - a_k for every k, is wrong for even k).
  * G18  the printed set P~_d omits f = c_d X^d + c_1 X (support {d, 1}: squarefree for suitable c_d, c_1); it is
         added with mult q (q-1) / 2, the same count as for support {d, 0}: no ratio is normalised by X -> aX.
  * G19  only p not dividing d.  For p | d the printed set misses every polynomial with
         c_{d-1} = 0 != c_{d-2}, so it cannot be followed; reduced_map raises for p | d (and so does the library).
  * R_m, the representatives of F_q^x / F_q^{x m}: any choice gives the same map.  Here: scan c = 1, 2, .. in the
    integer encoding and keep c when it is in no earlier coset (c/r is an m-th power iff (c/r)^((q-1)/gcd(m,q-1)) = 1).
    The library uses powers of its generator instead; the two sides therefore enumerate DIFFERENT reduced sets and
    must still agree on the map.

Nothing here is imported by the product (only tests/ and bench.py's oracle legs may).
"""
from __future__ import annotations

import itertools
import math
from collections import Counter

import numpy as np

from oracle import hec_oracle as O


class Fq:
    """F_q in the integer encoding of reading G7 (sum a_i p^i <-> sum a_i T^i mod R_q), via the oracle's multiply."""

    def __init__(self, q: int):
        self.q = q
        self.p, self.r = O._factor_prime_power(q)
        self.mod = O.smallest_primitive(self.p, self.r)

    def mul(self, a: int, b: int) -> int:
        if self.r == 1:
            return a * b % self.p
        return O.mul_encoded(self.p, self.mod, a, b)

    def pow(self, a: int, e: int) -> int:
        acc = 1
        while e:
            if e & 1:
                acc = self.mul(acc, a)
            a = self.mul(a, a)
            e >>= 1
        return acc

    def inv(self, a: int) -> int:
        return self.pow(a, self.q - 2)

    def coset_representatives(self, m: int) -> list[int]:
        """R_m: one element of every coset of the m-th powers in F_q^x."""
        gam = math.gcd(m, self.q - 1)
        e = (self.q - 1) // gam
        reps: list[int] = []
        for c in range(1, self.q):
            if all(self.pow(self.mul(c, self.inv(r)), e) != 1 for r in reps):
                reps.append(c)
        assert len(reps) == gam
        return reps

    def non_square(self) -> int:
        return next(c for c in range(1, self.q) if self.pow(c, (self.q - 1) // 2) != 1)


def reduced_polynomials(q: int, d: int):
    """Yields (coefficients c_0..c_d, mult) over the set P~'_d(F_q) of PAPER.md:113-121 BEFORE the squarefree
    filter (readings G9, G18); p must not divide d (reading G19).  mult per PAPER.md:91-97."""
    F = Fq(q)
    if d % F.p == 0:
        raise ValueError("reduced polynomials: p | d is not covered (reading G19)")
    units = range(1, q)
    for support_low in (0, 1):                        # c_d X^d + X^0 and c_d X^d + X^1 (reading G18)
        for cd in units:
            c = [0] * (d + 1)
            c[d], c[support_low] = cd, 1
            yield c, q * (q - 1) // 2
    for i in range(1, d - 1):                         # 1 <= i <= d-2
        for j in range(0, i):
            reps = F.coset_representatives(i - j)     # c_i = 1, so c_j runs over c_i R_{i-j} = R_{i-j}
            m = q * (q - 1) ** 2 // (2 * math.gcd(q - 1, i - j))
            for cd in units:
                for cj in reps:
                    for low in itertools.product(range(q), repeat=j):
                        c = [0] * (d + 1)
                        c[d], c[i], c[j] = cd, 1, cj
                        c[:j] = low
                        yield c, m


def twist_tuple(q: int, t) -> tuple:
    """(N_1..N_g) of the quadratic twist n f (reading G8)."""
    return tuple((2 * q ** k + 2 - n) if k % 2 else n for k, n in enumerate(t, start=1))


def _pad(rows, g: int) -> np.ndarray:
    a = np.zeros((len(rows), 2 * g + 3), dtype=np.uint16)
    for r, c in enumerate(rows):
        a[r, :len(c)] = c
    return a


def reduced_map(q: int, g: int, d: int) -> dict:
    """Algorithm 1 for one d: {(N_1..N_g): weighted count}."""
    polys, mults = [], []
    for c, m in reduced_polynomials(q, d):
        polys.append(c)
        mults.append(m)
    cnt, sf, _ = O.count(q, g, _pad(polys, g))
    out: Counter = Counter()
    for row, flag, m in zip(cnt, sf, mults):
        if not flag:
            continue                                   # P_d holds squarefree polynomials only
        t = tuple(int(v) for v in row)
        out[t] += m                                    # Algorithm 1 line 20
        out[twist_tuple(q, t)] += m                    # line 21 (reading G8)
    return dict(out)


def brute_force_map(q: int, g: int, d: int) -> dict:
    """The definition: every polynomial of degree d over F_q."""
    rows = [list(low) + [cd] for cd in range(1, q) for low in itertools.product(range(q), repeat=d)]
    cnt, sf, _ = O.count(q, g, _pad(rows, g))
    out: Counter = Counter()
    for row, flag in zip(cnt, sf):
        if flag:
            out[tuple(int(v) for v in row)] += 1
    return dict(out)


def reduced_map_lambda(q: int, g: int, d: int) -> dict:
    """Algorithm 1 for one d with the full key of (1.2): {((N_1..N_g), lambda): weighted count}, lambda a multiplicity
    vector (oracle/hec_lambda_oracle.py).  The twist n f has the factorisation type of f."""
    from oracle import hec_lambda_oracle as LO
    polys, mults = [], []
    for c, m in reduced_polynomials(q, d):
        polys.append(c)
        mults.append(m)
    rows = _pad(polys, g)
    cnt, sf, _ = O.count(q, g, rows)
    lam = LO.lambda_by_roots(q, g, rows)
    out: Counter = Counter()
    for row, flag, m, la in zip(cnt, sf, mults, lam):
        if not flag:
            continue
        t = tuple(int(v) for v in row)
        out[(t, la)] += m
        out[(twist_tuple(q, t), la)] += m
    return dict(out)


def brute_force_map_lambda(q: int, g: int, d: int) -> dict:
    """The definition (1.2): every polynomial of degree d, keyed by ((N_1..N_g), lambda)."""
    from oracle import hec_lambda_oracle as LO
    rows = _pad([list(low) + [cd] for cd in range(1, q) for low in itertools.product(range(q), repeat=d)], g)
    cnt, sf, _ = O.count(q, g, rows)
    lam = LO.lambda_by_roots(q, g, rows)
    out: Counter = Counter()
    for row, flag, la in zip(cnt, sf, lam):
        if flag:
            out[(tuple(int(v) for v in row), la)] += 1
    return dict(out)


def map_to_arrays(m: dict, g: int):
    """Sorted (tuples[n][g] uint32, weights[n] uint64), ascending lexicographic order."""
    keys = sorted(m)
    return (np.array(keys, dtype=np.uint32).reshape(len(keys), g), np.array([m[k] for k in keys], dtype=np.uint64))
