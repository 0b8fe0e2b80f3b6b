"""TEST INFRASTRUCTURE ONLY -- oracle for SURVEY.md 8(f) NEXT-3: lambda(f), the factorisation type of f over F_q.

Definition: for squarefree f of degree 2g+2, lambda(f) is the partition deg f_1 + .. + deg f_l of the
factorisation f = prod f_i into irreducibles over F_q; for degree 2g+1 that partition amended by a summand 1.

lambda_by_roots: an irreducible of degree e over F_q has all its e roots in F_{q^k} exactly when e | k, so for
squarefree f the root counts r0_k = #{x in F_{q^k}: f(x) = 0} (the oracle's plain count) satisfy
r0_k = sum_{e | k} e n_e, n_e = number of irreducible factors of degree e.  Moebius inversion gives every n_e with
e <= floor(d/2) from r0_1 .. r0_{floor(d/2)}; what is left of the degree is one more irreducible factor (two factors
above d/2 do not fit).  This uses k up to floor(d/2) = g+1, one field MORE than the device path (which, in the one
case g fields leave open -- no factor of degree <= g, d = 2g+2 -- decides by the quadratic character of the
discriminant); the two sides share nothing.

Pinned (tests/test_lambda_oracle_pins.py) against trial division by every monic irreducible over F_3, F_5 (pure
Python) and against the closed-form number of squarefree polynomials of each type, prod_e C(I_e, n_e).
A partition is a tuple of multiplicities (n_1, .., n_{2g+2}).
"""
from __future__ import annotations

import numpy as np

from oracle import hec_oracle as O

_MU = {1: 1, 2: -1, 3: -1, 4: 0, 5: -1, 6: 1, 7: -1, 8: 0, 9: 0, 10: 1, 11: -1, 12: 0}


def lambda_by_roots(q: int, g: int, coeffs) -> list:
    """For every row: the multiplicity vector (n_1..n_{2g+2}) of lambda(f), or None if f is not squarefree."""
    c = np.ascontiguousarray(coeffs, dtype=np.uint16)
    D = 2 * g + 2
    _, sf, _ = O.count(q, g, c, k_lo=1, k_hi=0)               # squarefree flags only (Euclid)
    half = g + 1                                               # floor(d/2) for d = 2g+1 and 2g+2
    r0 = O.roots(q, g, c, k_hi=half).astype(np.int64)
    out = []
    for row, flag, roots in zip(c, sf, r0):
        if not flag:
            out.append(None)
            continue
        d = D if row[D] else D - 1
        n = [0] * (D + 1)
        for e in range(1, d // 2 + 1):
            s = sum(_MU[e // m] * int(roots[m - 1]) for m in range(1, e + 1) if e % m == 0)
            assert s >= 0 and s % e == 0
            n[e] = s // e
        rest = d - sum(e * n[e] for e in range(1, D + 1))
        assert rest == 0 or rest > d // 2
        if rest:
            n[rest] += 1
        if d == D - 1:
            n[1] += 1                                          # degree 2g+1 gets an additional summand 1
        out.append(tuple(n[1:]))
    return out


def partitions(total: int) -> list:
    """All partitions of `total` as multiplicity vectors (n_1..n_total), in ascending lexicographic order of that
    vector -- the index order of the library's lambda codes (include/hec.h)."""
    res = []

    def rec(e, left, acc):
        if e > total:
            if left == 0:
                res.append(tuple(acc))
            return
        for m in range(left // e + 1):
            rec(e + 1, left - m * e, acc + [m])

    rec(1, total, [])
    return sorted(res)
