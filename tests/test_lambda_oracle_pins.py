"""Pins of oracle/hec_lambda_oracle.py (lambda(f) of PAPER.md:61), CPU only: the root-count
oracle against (a) trial division by every monic irreducible polynomial, written here in plain Python over prime
fields, and (b) the closed-form number of squarefree polynomials of each factorisation type."""
import itertools
from collections import Counter
from math import comb

import numpy as np
import pytest

from oracle import hec_lambda_oracle as L


def _polymod(a, b, p):
    """a mod b over F_p, coefficient lists low -> high, b monic."""
    a = a[:]
    while len(a) >= len(b):
        c = a[-1]
        if c:
            s = len(a) - len(b)
            for i, bi in enumerate(b):
                a[s + i] = (a[s + i] - c * bi) % p
        a.pop()
    return a


def _polydiv_exact(a, b, p):
    a, quo = a[:], [0] * (len(a) - len(b) + 1)
    while len(a) >= len(b):
        c = a[-1]
        s = len(a) - len(b)
        quo[s] = c
        for i, bi in enumerate(b):
            a[s + i] = (a[s + i] - c * bi) % p
        a.pop()
    assert not any(a)
    return quo


def _irreducibles(p, maxdeg):
    """Monic irreducibles of degree 1..maxdeg over F_p by sieving: a monic polynomial is irreducible iff no monic
    irreducible of at most half its degree divides it."""
    irr = {e: [] for e in range(1, maxdeg + 1)}
    for e in range(1, maxdeg + 1):
        for low in itertools.product(range(p), repeat=e):
            f = list(low) + [1]
            if all(any(_polymod(f, h, p)) for k in range(1, e // 2 + 1) for h in irr[k]):
                irr[e].append(f)
    return irr


def _type_by_trial_division(c, p, irr, D):
    d = max(i for i, v in enumerate(c) if v)
    inv = pow(c[d], p - 2, p)
    f = [v * inv % p for v in c[:d + 1]]
    n = [0] * (D + 1)
    for e in sorted(irr):
        for h in irr[e]:
            while len(f) > len(h) - 1 and len(f) >= len(h) and not any(_polymod(f, h, p)):
                f = _polydiv_exact(f, h, p)
                n[e] += 1
    if len(f) > 1:
        n[len(f) - 1] += 1                       # what is left has no factor of degree <= maxdeg: irreducible
    if d == D - 1:
        n[1] += 1
    return tuple(n[1:])


@pytest.mark.parametrize("p,g", [(3, 1), (3, 2), (5, 1), (5, 2), (7, 1)])
def test_root_count_lambda_equals_trial_division(p, g):
    D = 2 * g + 2
    irr = _irreducibles(p, g + 1)
    rng = np.random.default_rng(1805)
    if p ** (D + 1) <= 20000:
        rows = np.array([r for r in itertools.product(range(p), repeat=D + 1) if r[D] or r[D - 1]], dtype=np.uint16)
    else:
        rows = rng.integers(0, p, size=(4000, D + 1)).astype(np.uint16)
        rows[rows[:, D] == 0, D - 1] = 1
    lam = L.lambda_by_roots(p, g, rows)
    checked = 0
    for c, t in zip(rows.tolist(), lam):
        if t is None:
            continue
        assert t == _type_by_trial_division(c, p, irr, D), c
        assert sum((e + 1) * m for e, m in enumerate(t)) == D
        checked += 1
    assert checked > len(rows) // 2


@pytest.mark.parametrize("q,g", [(3, 1), (3, 2), (5, 1), (9, 1)])
def test_type_counts_match_the_closed_form(q, g):
    """Exhaustive over degree 2g+2: #squarefree f with n_e irreducible factors of degree e = (q-1) prod_e C(I_e, n_e),
    I_e = (1/e) sum_{m | e} mu(e/m) q^m monic irreducibles of degree e (also exercises prime-power q)."""
    D = 2 * g + 2
    rows = np.array([r for r in itertools.product(range(q), repeat=D + 1) if r[D]], dtype=np.uint16)
    got = Counter(t for t in L.lambda_by_roots(q, g, rows) if t is not None)
    I = {e: sum(L._MU[e // m] * q ** m for m in range(1, e + 1) if e % m == 0) // e for e in range(1, D + 1)}
    for part in L.partitions(D):
        want = q - 1
        for e, m in enumerate(part, start=1):
            want *= comb(I[e], m)
        assert got.get(part, 0) == want, part
    assert sum(got.values()) == (q - 1) * (q ** D - q ** (D - 1))


def test_partition_order():
    assert L.partitions(4) == [(0, 0, 0, 1), (0, 2, 0, 0), (1, 0, 1, 0), (2, 1, 0, 0), (4, 0, 0, 0)]
    assert [len(L.partitions(n)) for n in (4, 6, 8, 10, 12)] == [5, 11, 22, 42, 77]
