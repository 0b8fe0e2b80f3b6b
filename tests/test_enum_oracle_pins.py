"""Pins of oracle/hec_enum_oracle.py (Algorithm 1 without lambda), CPU only.

reduced_map follows Algorithm 1 over the reduced polynomials of sections 1.2-1.3; it is pinned
to the DEFINITION of the map (eq. (1.2), lambda dropped) computed by brute force over every
polynomial of degree d, to the textbook count of squarefree polynomials, and to the twist symmetry.  Each reading
(G8, G9, G18) is shown to matter: undoing it breaks a pin."""
import math

import pytest

from oracle import hec_enum_oracle as E

SMALL = [(3, 2, 5), (3, 1, 4), (5, 1, 3), (5, 1, 4), (7, 1, 3), (7, 1, 4), (5, 2, 6), (7, 2, 5),
         (3, 1, 3), (3, 2, 6), (5, 2, 5), (9, 1, 3)]               # the last four: p | d (reading G19)


@pytest.mark.parametrize("q,g,d", SMALL)
def test_reduced_map_equals_brute_force(q, g, d):
    assert E.reduced_map(q, g, d) == E.brute_force_map(q, g, d)


@pytest.mark.parametrize("q,g,d", SMALL + [(13, 2, 5), (11, 2, 6), (9, 1, 4)])
def test_total_weight_is_the_number_of_squarefree_polynomials(q, g, d):
    # textbook: q^d - q^(d-1) monic squarefree polynomials of degree d >= 2, times q-1 leading coefficients
    m = E.reduced_map(q, g, d)
    assert sum(m.values()) == (q - 1) * (q ** d - q ** (d - 1))


@pytest.mark.parametrize("q,g,d", [(5, 2, 6), (7, 2, 5), (13, 2, 5)])
def test_map_is_symmetric_under_the_twist(q, g, d):
    m = E.reduced_map(q, g, d)
    for t, w in m.items():
        assert m[E.twist_tuple(q, t)] == w
        assert E.twist_tuple(q, E.twist_tuple(q, t)) == t


def test_multiplicities_and_family_sizes():
    # PAPER.md:91-97 with q = 7, d = 5: mult q(q-1)/2 = 21 for the two-term families, q(q-1)^2/(2 gcd(q-1, i-j)) else
    q, d = 7, 5
    seen = {}
    n = 0
    for c, m in E.reduced_polynomials(q, d):
        n += 1
        assert c[d] != 0 and c[d - 1] == 0
        supp = [l for l in range(d) if c[l]]
        i = supp[-1]
        assert c[i] == 1                                   # P~': the coefficient in R_2 is fixed to 1
        if len(supp) == 1:
            assert i in (0, 1) and m == q * (q - 1) // 2
        else:
            j = supp[-2]
            assert m == q * (q - 1) ** 2 // (2 * math.gcd(q - 1, i - j))
        seen[tuple(c)] = m
    assert len(seen) == n                                  # no polynomial twice
    want = 2 * (q - 1) + sum((q - 1) * math.gcd(q - 1, i - j) * q ** j for i in range(1, d - 1) for j in range(i))
    assert n == want


def test_reading_g18_is_needed():
    """Without the family c_d X^d + X (omitted in the printed set) the map misses curves."""
    q, g, d = 5, 1, 3
    from collections import Counter
    import numpy as np
    from oracle import hec_oracle as O
    polys = [(c, m) for c, m in E.reduced_polynomials(q, d) if not (c[1] == 1 and sum(1 for v in c[:d] if v) == 1)]
    cnt, sf, _ = O.count(q, g, E._pad([c for c, _ in polys], g))
    out = Counter()
    for row, flag, (_, m) in zip(cnt, sf, polys):
        if flag:
            t = tuple(int(v) for v in row)
            out[t] += m
            out[E.twist_tuple(q, t)] += m
    assert dict(out) != E.brute_force_map(q, g, d)
    assert sum(out.values()) < (q - 1) * (q ** d - q ** (d - 1))


def test_reading_g8_is_needed():
    """Line 21 as printed (a_k -> 1 + q^k - a_k, i.e. N_k -> 2 q^k + 2 - N_k, for EVERY k) gives a wrong map."""
    q, g, d = 5, 2, 6
    good = E.brute_force_map(q, g, d)
    printed = lambda t: tuple(2 * q ** k + 2 - n for k, n in enumerate(t, start=1))
    assert any(printed(t) not in good for t in good)
    assert all(E.twist_tuple(q, t) in good for t in good)


def test_coset_representatives():
    F = E.Fq(25)
    for m in (1, 2, 3, 4, 6, 8):
        reps = F.coset_representatives(m)
        gam = math.gcd(m, 24)
        assert len(reps) == gam
        e = 24 // gam
        for a in range(len(reps)):
            for b in range(a):
                assert F.pow(F.mul(reps[a], F.inv(reps[b])), e) != 1


def test_reading_g19_is_needed():
    """p | d: the set as printed (i <= d-3 whatever c_{d-1} is) has no polynomial with
    c_{d-1} = 0 != c_{d-2}; without those rows the map falls short of the definition."""
    from collections import Counter
    from oracle import hec_oracle as O
    q, g, d = 3, 2, 6
    polys = [(c, m) for c, m in E.reduced_polynomials(q, d) if not (c[d - 1] == 0 and c[d - 2] != 0)]
    cnt, sf, _ = O.count(q, g, E._pad([c for c, _ in polys], g))
    out = Counter()
    for row, flag, (_, m) in zip(cnt, sf, polys):
        if flag:
            t = tuple(int(v) for v in row)
            out[t] += m
            out[E.twist_tuple(q, t)] += m
    assert sum(out.values()) < (q - 1) * (q ** d - q ** (d - 1))
    assert E.reduced_map(q, g, d) == E.brute_force_map(q, g, d)


@pytest.mark.parametrize("q,g,d", [(3, 2, 5), (5, 1, 3), (5, 1, 4), (7, 1, 4), (5, 2, 6),
                                   (3, 1, 3), (3, 2, 6), (5, 2, 5)])         # the last three: p | d (reading G19)
def test_reduced_map_with_lambda_equals_brute_force(q, g, d):
    """Full key of (1.2): Algorithm 1 with lambda (lines 18-21) over the reduced
    polynomials equals the definition over EVERY polynomial of degree d -- the reduction (shift, scaling: PAPER.md:73-121)
    and the twist n f (reading G8) preserve the factorisation type, in both strata of p | d."""
    assert E.reduced_map_lambda(q, g, d) == E.brute_force_map_lambda(q, g, d)


@pytest.mark.parametrize("q,g,d", [(5, 2, 6), (3, 2, 6), (7, 1, 4)])
def test_lambda_map_projects_onto_the_map_without_lambda(q, g, d):
    """Summing the full-key map over lambda gives the map without it (two functions, one Algorithm 1)."""
    from collections import Counter
    proj = Counter()
    for (t, lam), w in E.reduced_map_lambda(q, g, d).items():
        proj[t] += w
    assert dict(proj) == E.reduced_map(q, g, d)
