"""Pins of the CPU oracle (oracle/hec_oracle.c) against things OTHER than itself.

Everything here runs without a GPU.  The paper prints no point counts (its Table 1,
PAPER.md:313-326, is run times only), so the pins are: an independent pure-Python brute
force in a different representation (F_9 = F_3[i]/(i^2+1)), hand-enumerated curves
(tests/golden/f3_hand_curves.txt), closed forms, textbook identities (g = 1 zeta function,
g = 2 Newton identities), the Weil bound, the twist relation (reading G8), the zero-sum
identity (reading G17) and special families.
"""
import itertools
from collections import Counter
from pathlib import Path

import numpy as np
import pytest

from oracle import hec_oracle as O
from paper_1805_11991_b200 import workloads as W

GOLDEN = Path(__file__).resolve().parent / "golden"


# ----------------------------------------------------------------------------------------
# independent pure-Python helpers (share nothing with the oracle's C code)
# ----------------------------------------------------------------------------------------

def _f9_mul(a, b):
    """(a0 + a1 i)(b0 + b1 i) with i^2 = -1 over F_3 -- NOT the oracle's modulus."""
    return ((a[0] * b[0] - a[1] * b[1]) % 3, (a[0] * b[1] + a[1] * b[0]) % 3)


def _f9_add(a, b):
    return ((a[0] + b[0]) % 3, (a[1] + b[1]) % 3)


_F9 = [(a, b) for a in range(3) for b in range(3)]
_F9_SQUARES = {_f9_mul(y, y) for y in _F9 if y != (0, 0)}


def _brute_counts_f3(row):
    """(N_1, N_2) of y^2 = f(x), f in F_3[x] of degree 5/6, straight from PAPER.md:41-49."""
    c = [int(v) for v in row]
    n1 = 0
    for x in range(3):
        v = sum(c[j] * x ** j for j in range(7)) % 3
        n1 += 1 if v == 0 else (2 if v == 1 else 0)          # squares of F_3^x: {1}
    n1 += 1 if c[6] == 0 else (2 if c[6] == 1 else 0)
    n2 = 0
    for x in _F9:
        acc = (0, 0)
        for j in range(6, -1, -1):
            acc = _f9_add(_f9_mul(acc, x), (c[j], 0))
        n2 += 1 if acc == (0, 0) else (2 if acc in _F9_SQUARES else 0)
    n2 += 1 if c[6] == 0 else 2                              # every element of F_3^x is a square in F_9
    return n1, n2


def _polymul_mod(a, b, p):
    out = [0] * (len(a) + len(b) - 1)
    for i, x in enumerate(a):
        for j, y in enumerate(b):
            out[i + j] = (out[i + j] + x * y) % p
    return out


def _brute_squarefree_f3(row):
    """Trial division by g^2 for every monic g of degree 1..3 over F_3."""
    f = [int(v) for v in row]
    while f and f[-1] == 0:
        f.pop()
    for dg in (1, 2, 3):
        for low in itertools.product(range(3), repeat=dg):
            g2 = _polymul_mod(list(low) + [1], list(low) + [1], 3)
            if len(g2) > len(f):
                continue
            w = f[:]
            for m in range(len(w) - 1, len(g2) - 2, -1):     # monic long division
                t = w[m]
                if t:
                    for i, gv in enumerate(g2):
                        w[m - len(g2) + 1 + i] = (w[m - len(g2) + 1 + i] - t * gv) % 3
            if not any(w[: len(g2) - 1]):
                return 0
    return 1


def _poly_powmod_t(e, mod, p):
    """t^e in F_p[t]/(mod) by square-and-multiply on coefficient lists (pure Python)."""
    n = len(mod) - 1

    def red(w):
        w = w[:]
        for m in range(len(w) - 1, n - 1, -1):
            t = w[m]
            if t:
                for i in range(n + 1):
                    w[m - n + i] = (w[m - n + i] - t * mod[i]) % p
        return (w + [0] * n)[:n]

    result = [1] + [0] * (n - 1)
    base = red([0, 1])
    while e:
        if e & 1:
            result = red(_polymul_mod(result, base, p))
        base = red(_polymul_mod(base, base, p))
        e >>= 1
    return result


def _prime_factors(m):
    out, d = set(), 2
    while d * d <= m:
        while m % d == 0:
            out.add(d)
            m //= d
        d += 1
    if m > 1:
        out.add(m)
    return out


def _is_primitive_py(mod, p):
    n = len(mod) - 1
    if mod[0] == 0:
        return False
    order = p ** n - 1
    one = [1] + [0] * (n - 1)
    if _poly_powmod_t(order, mod, p) != one:
        return False
    return all(_poly_powmod_t(order // ell, mod, p) != one for ell in _prime_factors(order))


def _rand_rows(q, g, n, seed, degree=None, squarefree_only=False):
    """Seeded uniform rows of degree 2g+1/2g+2 (test-local; not one of the five workloads)."""
    rng = np.random.default_rng(seed)
    rows = rng.integers(0, q, size=(n, 2 * g + 3)).astype(np.uint16)
    top = rng.integers(1, q, size=n).astype(np.uint16)
    even = rng.integers(0, 2, size=n).astype(bool) if degree is None else np.full(n, degree == 2 * g + 2)
    rows[:, -1] = np.where(even, top, 0)
    rows[:, -2] = np.where(even, rows[:, -2], top)
    if squarefree_only:
        _, sf, _ = O.count(q, g, rows, k_lo=1, k_hi=0)
        rows = rows[sf == 1]
    return rows


# ----------------------------------------------------------------------------------------
# moduli (reading G7)
# ----------------------------------------------------------------------------------------

def _golden_moduli():
    out = []
    for line in (GOLDEN / "moduli_g7.txt").read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        left, right = line.split("|")
        p, n = (int(v) for v in left.split())
        out.append((p, n, [int(v) for v in right.split()]))
    return out


@pytest.mark.parametrize("p,n,mod", _golden_moduli())
def test_smallest_primitive_matches_golden_and_independent_order_test(p, n, mod):
    if p ** n <= 30000:                      # the oracle's own search is a brute-force walk
        assert O.smallest_primitive(p, n) == mod
    # independent check: primitive, and nothing lexicographically smaller is
    assert _is_primitive_py(mod, p)
    idx = sum(a * p ** i for i, a in enumerate(mod[:-1]))
    smaller = 0
    for e in range(idx):
        cand = [(e // p ** i) % p for i in range(n)] + [1]
        assert not _is_primitive_py(cand, p), cand
        smaller += 1
    assert smaller == idx


def test_is_primitive_agrees_with_independent_order_test():
    for p, n in [(3, 2), (5, 2), (7, 2), (3, 3)]:
        for e in range(p ** n):
            cand = [(e // p ** i) % p for i in range(n)] + [1]
            assert O.is_primitive(p, cand) == _is_primitive_py(cand, p), (p, cand)


def test_smallest_irreducible_has_no_roots_and_is_minimal():
    # degree 2 and 3: irreducible <=> no root in F_p (textbook)
    for p, n in [(3, 2), (5, 2), (7, 2), (13, 2), (13, 3), (293, 2), (7, 3)]:
        mod = O.smallest_irreducible(p, n)
        idx = sum(a * p ** i for i, a in enumerate(mod[:-1]))

        def has_root(m):
            return any(sum(a * x ** i for i, a in enumerate(m)) % p == 0 for x in range(p))

        assert not has_root(mod)
        for e in range(idx):
            cand = [(e // p ** i) % p for i in range(n)] + [1]
            assert has_root(cand)


def test_mul_encoded_field_axioms_and_prime_field():
    for a in range(13):
        for b in range(13):
            assert O.mul_encoded(13, [0, 1], a, b) == a * b % 13
    rng = np.random.default_rng(1)
    for p, n in [(3, 2), (5, 4), (7, 6), (13, 4)]:
        mod = O.smallest_primitive(p, n) if p ** n < 30000 else [5, 1, 3, 0, 0, 0, 1]
        Q = p ** n

        def add(a, b):
            return sum((((a // p ** i) + (b // p ** i)) % p) * p ** i for i in range(n))

        for _ in range(200):
            a, b, c = (int(v) for v in rng.integers(0, Q, 3))
            assert O.mul_encoded(p, mod, a, b) == O.mul_encoded(p, mod, b, a)
            assert O.mul_encoded(p, mod, a, 1) == a
            assert O.mul_encoded(p, mod, O.mul_encoded(p, mod, a, b), c) == \
                O.mul_encoded(p, mod, a, O.mul_encoded(p, mod, b, c))
            assert O.mul_encoded(p, mod, a, add(b, c)) == add(O.mul_encoded(p, mod, a, b), O.mul_encoded(p, mod, a, c))
        # t * t^{n-1} = -(a_0 + ... + a_{n-1} t^{n-1})
        expect = sum(((-mod[i]) % p) * p ** i for i in range(n))
        assert O.mul_encoded(p, mod, p, p ** (n - 1)) == expect


# ----------------------------------------------------------------------------------------
# config 1: every f over F_3 of degree 5 or 6 (1944 polynomials)
# ----------------------------------------------------------------------------------------

@pytest.fixture(scope="module")
def config1():
    rows = W.generate(W.CONFIGS[1])
    cnt, sf, _ = O.count(3, 2, rows)
    return rows, cnt, sf


def test_hand_enumerated_curves_over_f3():
    rows, want = [], []
    for line in (GOLDEN / "f3_hand_curves.txt").read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        left, right = line.split("|")
        rows.append([int(v) for v in left.split()])
        want.append([int(v) for v in right.split()])
    cnt, sf, _ = O.count(3, 2, np.array(rows, dtype=np.uint16))
    want = np.array(want)
    assert (cnt == want[:, :2]).all()
    assert (sf == want[:, 2]).all()


def test_config1_matches_independent_brute_force(config1):
    rows, cnt, sf = config1
    assert rows.shape == (1944, 7)
    for i, row in enumerate(rows):
        assert tuple(cnt[i]) == _brute_counts_f3(row), row
        assert sf[i] == _brute_squarefree_f3(row), row


def test_config1_closed_forms(config1):
    rows, cnt, sf = config1
    deg5 = rows[:, 6] == 0
    # squarefree polynomials of degree d with nonzero leading coefficient: (q-1)(q^d - q^{d-1})
    assert sf[deg5].sum() == 2 * (3 ** 5 - 3 ** 4) == 324
    assert sf[~deg5].sum() == 2 * (3 ** 6 - 3 ** 5) == 972
    # mean affine count is q over F_q and q^2+q-1 over F_{q^2}; infinity: 1 (odd degree),
    # mean 1 (k odd) / 2 (k even) for even degree
    assert cnt[deg5, 0].sum() == 486 * (3 + 1)
    assert cnt[~deg5, 0].sum() == 1458 * (3 + 1)
    assert cnt[deg5, 1].sum() == 486 * (11 + 1)
    assert cnt[~deg5, 1].sum() == 1458 * (11 + 2)
    assert cnt[:, 0].max() <= 8 and cnt[:, 1].min() >= 5 and cnt[:, 1].max() <= 20


def test_config1_histogram_against_counter_and_symmetry(config1):
    rows, cnt, sf = config1
    tup, mult = O.histogram(cnt)
    brute = Counter(_brute_counts_f3(r) for r in rows)
    assert len(tup) == len(brute) == 60
    assert [tuple(t) for t in tup] == sorted(brute)
    assert all(brute[tuple(t)] == m for t, m in zip(tup, mult))
    assert mult.sum() == 1944
    tsf, msf = O.histogram(cnt, sf)
    assert len(tsf) == 50 and msf.sum() == 1296
    # twist symmetry (reading G8): N_1 -> 2q+2-N_1 = 8-N_1, N_2 fixed
    h = {tuple(t): m for t, m in zip(tup, mult)}
    assert all(h.get((8 - a, b), 0) == m for (a, b), m in h.items())
    # stored fixture (written from the oracle by tests/golden/make_config1_histogram.py)
    lines = [ln for ln in (GOLDEN / "config1_histogram.txt").read_text().splitlines() if not ln.startswith("#")]
    stored = {(int(a), int(b)): int(m) for a, b, m in (ln.split() for ln in lines)}
    assert stored == {k: int(v) for k, v in h.items()}


def test_histogram_empty_and_mask():
    t, m = O.histogram(np.zeros((0, 3), dtype=np.uint32))
    assert t.shape == (0, 3) and m.shape == (0,)
    c = np.array([[5, 1], [2, 9], [5, 1], [2, 8]], dtype=np.uint32)
    t, m = O.histogram(c, np.array([1, 1, 1, 0]))
    assert t.tolist() == [[2, 9], [5, 1]] and m.tolist() == [1, 2]


# ----------------------------------------------------------------------------------------
# textbook identities that exercise the extension-field pipeline and the embedding (G6)
# ----------------------------------------------------------------------------------------

@pytest.mark.parametrize("q", [3, 7, 9, 13, 25])
def test_genus1_n2_from_n1(q):
    """Elliptic curves: #E(F_{q^2}) = N_1 (2q + 2 - N_1)  (zeta function of a genus-1 curve)."""
    rows = _rand_rows(q, 1, 60, seed=100 + q, squarefree_only=True)
    assert len(rows) > 20
    cnt, _, _ = O.count(q, 1, rows, k_hi=2)
    n1, n2 = cnt[:, 0].astype(np.int64), cnt[:, 1].astype(np.int64)
    assert (n2 == n1 * (2 * q + 2 - n1)).all()


@pytest.mark.parametrize("q", [3, 5, 9])
def test_genus2_n3_from_newton_identities(q):
    """L(T) = 1 + c1 T + c2 T^2 + q c1 T^3 + q^2 T^4, s_k = q^k + 1 - N_k,
    c1 = -s1, c2 = (s1^2 - s2)/2, s3 = -(c1 s2 + c2 s1 + 3 q c1)."""
    rows = _rand_rows(q, 2, 40, seed=200 + q, squarefree_only=True)
    assert len(rows) > 10
    cnt, _, _ = O.count(q, 2, rows, k_hi=3)
    n = cnt.astype(np.int64)
    s1, s2, s3 = (q ** k + 1 - n[:, k - 1] for k in (1, 2, 3))
    c1 = -s1
    assert ((s1 * s1 - s2) % 2 == 0).all()
    c2 = (s1 * s1 - s2) // 2
    assert (s3 == -(c1 * s2 + c2 * s1 + 3 * q * c1)).all()


@pytest.mark.parametrize("q,g,kmax,n", [(25, 2, 2, 48), (49, 3, 2, 32), (49, 3, 3, 3), (13, 4, 3, 48),
                                        (13, 4, 4, 8), (293, 2, 1, 64), (293, 2, 2, 8)])
def test_weil_bound_and_parity(q, g, kmax, n):
    """|N_k - (q^k + 1)| <= 2 g q^{k/2} for squarefree f; N_k = r0 + inf-term (mod 2)."""
    rows = _rand_rows(q, g, n, seed=300 + q + kmax, squarefree_only=True)
    cnt, _, _ = O.count(q, g, rows, k_lo=kmax, k_hi=kmax)
    nk = cnt[:, kmax - 1].astype(np.float64)
    assert (np.abs(nk - (q ** kmax + 1)) <= 2 * g * q ** (kmax / 2) + 1e-9).all()
    # parity: N_k = r0 + 2 r_sq + inf-term, so N_k - r0 - inf-term is even; the infinity term decided
    # here without the oracle: 1 for odd degree; for even degree 2 or 0, hence irrelevant mod 2
    r0 = O.roots(q, g, rows, k_hi=kmax)[:, kmax - 1].astype(np.int64)
    inf = np.where(rows[:, 2 * g + 2] == 0, 1, 0)
    assert ((cnt[:, kmax - 1].astype(np.int64) - r0 - inf) % 2 == 0).all()
    assert (r0 <= 2 * g + 2).all()                                           # a nonzero polynomial has at most deg f roots


def test_zero_sum_over_constant_term_orbit():
    """sum_{c0 in F_q} chi(f(x) + c0) = 0 for every x (reading G17): the affine counts of
    f + c0, c0 running over all of F_q, add up to q * q; the infinity term does not depend on c0."""
    for q, g in [(13, 2), (25, 2), (9, 3), (49, 1)]:
        for row in _rand_rows(q, g, 3, seed=400 + q, degree=2 * g + 1):       # odd degree: infinity term 1
            orbit = np.repeat(row[None, :], q, axis=0)
            orbit[:, 0] = np.arange(q)
            cnt, _, _ = O.count(q, g, orbit, k_hi=1, want_squarefree=False)
            assert int(cnt[:, 0].sum()) == q * q + q
    q, g = 13, 2                                                              # even degree, prime q
    for row in _rand_rows(q, g, 4, seed=450, degree=2 * g + 2):
        orbit = np.repeat(row[None, :], q, axis=0)
        orbit[:, 0] = np.arange(q)
        cnt, _, _ = O.count(q, g, orbit, k_hi=1, want_squarefree=False)
        inf = 2 if pow(int(row[-1]), (q - 1) // 2, q) == 1 else 0
        assert int(cnt[:, 0].sum()) == q * q + q * inf


def test_mean_affine_count_over_low_coefficients():
    """Averaging over all (c0, c1) in F_q^2: mean affine count over F_{q^2} is q^2 + q - 1."""
    for q, g in [(5, 2), (9, 1), (7, 2)]:
        row = _rand_rows(q, g, 1, seed=500 + q, degree=2 * g + 1)[0]
        grid = np.repeat(row[None, :], q * q, axis=0)
        grid[:, 0] = np.repeat(np.arange(q), q)
        grid[:, 1] = np.tile(np.arange(q), q)
        cnt, _, _ = O.count(q, g, grid, k_hi=2, want_squarefree=False)
        assert int(cnt[:, 0].sum()) == q * q * (q + 1)                 # +1: odd degree
        assert int(cnt[:, 1].sum()) == q * q * (q * q + q - 1 + 1)


def test_twist_relation():
    """Reading G8: for a non-square n of F_q, N_k(n f) + N_k(f) = 2 q^k + 2 (k odd),
    N_k(n f) = N_k(f) (k even)."""
    # prime q = 13: 2 is a non-square (squares: 1 3 4 9 10 12)
    rows = _rand_rows(13, 2, 12, seed=600)
    tw = ((rows.astype(np.int64) * 2) % 13).astype(np.uint16)
    a, _, _ = O.count(13, 2, rows, k_hi=3, want_squarefree=False)
    b, _, _ = O.count(13, 2, tw, k_hi=3, want_squarefree=False)
    assert (a[:, 0] + b[:, 0] == 2 * 13 + 2).all()
    assert (a[:, 1] == b[:, 1]).all()
    assert (a[:, 2] + b[:, 2] == 2 * 13 ** 3 + 2).all()
    # q = 9: the generator T (encoded 3) of F_9 = F_3[T]/(T^2+T+2) is a non-square
    Rq = O.smallest_primitive(3, 2)
    rows = _rand_rows(9, 2, 12, seed=601)
    tw = np.array([[O.mul_encoded(3, Rq, int(c), 3) for c in row] for row in rows], dtype=np.uint16)
    a, _, _ = O.count(9, 2, rows, want_squarefree=False)
    b, _, _ = O.count(9, 2, tw, want_squarefree=False)
    assert (a[:, 0] + b[:, 0] == 2 * 9 + 2).all()
    assert (a[:, 1] == b[:, 1]).all()


def test_special_families():
    for q, g in [(13, 4), (25, 2), (49, 3), (293, 2), (9, 2)]:
        nc = 2 * g + 3
        kmax = min(g, 2) if q > 13 else min(g, 3)
        # f = x^{2g+1}: N_k = q^k + 1 (x -> x^{2g+1} f(x) square iff x square; one zero; one point at infinity)
        row = np.zeros((1, nc), dtype=np.uint16)
        row[0, nc - 2] = 1
        cnt, sf, _ = O.count(q, g, row, k_hi=kmax)
        assert [int(v) for v in cnt[0, :kmax]] == [q ** k + 1 for k in range(1, kmax + 1)]
        assert sf[0] == 0
        # f = c x^{2g+2}: N_k = 2 q^k + 1 if c is a square in F_{q^k} (always for even k) else 1
        rows = np.zeros((q - 1, nc), dtype=np.uint16)
        rows[:, nc - 1] = np.arange(1, q)
        cnt, sf, _ = O.count(q, g, rows, k_hi=min(kmax, 2))
        assert set(cnt[:, 0].tolist()) == {1, 2 * q + 1}
        assert (cnt[:, 0] == 2 * q + 1).sum() == (q - 1) // 2        # half of F_q^x are squares
        if kmax >= 2:
            assert (cnt[:, 1] == 2 * q * q + 1).all()
        assert (sf == 0).all()


def test_c_times_square_family_prime_q():
    """f = c h(x)^2, h split over F_q with 3 distinct roots: N_k = r0 + (2 (q^k - r0) + 2) [c square in F_{q^k}]."""
    q, g = 13, 2
    h = np.array([1], dtype=np.int64)
    for root in (1, 2, 5):
        h = np.convolve(h, np.array([(-root) % q, 1])) % q             # low -> high
    h2 = np.convolve(h, h) % q
    rows = np.zeros((2, 7), dtype=np.uint16)
    rows[0, :7] = h2                      # c = 1
    rows[1, :7] = (2 * h2) % q            # c = 2, a non-square in F_13, a square in F_169
    cnt, sf, _ = O.count(q, g, rows)
    assert cnt[0].tolist() == [3 + 2 * (13 - 3) + 2, 3 + 2 * (169 - 3) + 2]
    assert cnt[1].tolist() == [3, 3 + 2 * (169 - 3) + 2]
    assert sf.tolist() == [0, 0]


def test_squarefree_closed_form_counts_prime_power():
    """#squarefree of degree d with nonzero leading coefficient = (q-1)(q^d - q^{d-1}); q = 9, g = 1."""
    q, g = 9, 1
    for d in (3, 4):
        digs = np.array(list(itertools.product(range(q), repeat=d)), dtype=np.uint16)   # c_0..c_{d-1}
        tot = 0
        for lead in range(1, q):
            rows = np.zeros((len(digs), 5), dtype=np.uint16)
            rows[:, :d] = digs[:, ::-1]
            rows[:, d] = lead
            _, sf, _ = O.count(q, g, rows, k_lo=1, k_hi=0)
            tot += int(sf.sum())
        assert tot == (q - 1) * (q ** d - q ** (d - 1))


def test_derivative_identically_zero_is_not_squarefree():
    # reading G14: x^6 + x^3 + 1 over F_3 and x^5 + 2 over F_5 (f' = 5 x^4 = 0)
    _, sf, _ = O.count(3, 2, np.array([[1, 0, 0, 1, 0, 0, 1]], dtype=np.uint16), k_lo=1, k_hi=0)
    assert sf[0] == 0
    _, sf, _ = O.count(5, 2, np.array([[2, 0, 0, 0, 0, 1, 0]], dtype=np.uint16), k_lo=1, k_hi=0)
    assert sf[0] == 0


def test_error_codes():
    with pytest.raises(ValueError, match="coefficient"):
        O.count(3, 2, np.array([[3, 0, 0, 0, 0, 1, 0]], dtype=np.uint16))
    with pytest.raises(ValueError, match="degree"):
        O.count(3, 2, np.array([[1, 1, 1, 1, 1, 0, 0]], dtype=np.uint16))
    with pytest.raises(ValueError):
        O.count(15, 2, np.zeros((1, 7), dtype=np.uint16))
    cnt, sf, _ = O.count(3, 2, np.zeros((0, 7), dtype=np.uint16))
    assert cnt.shape == (0, 2) and sf.shape == (0,)
