"""hec_build_field (host code, no GPU needed): the library's tables against polynomial arithmetic done by
the ORACLE's schoolbook multiply (a different code path: the library never multiplies two elements), against
the invariants of reading G16, and the moduli of reading G7.  Also: libhec.so exports every declared symbol."""
import ctypes
import re
from pathlib import Path

import numpy as np
import pytest

from oracle import hec_oracle as O
from paper_1805_11991_b200 import hec

ROOT = Path(__file__).resolve().parent.parent
FIELDS = [(3, 1, 1), (3, 1, 2), (5, 2, 1), (5, 2, 2), (7, 2, 1), (7, 2, 2), (7, 2, 3), (13, 1, 1), (13, 1, 2),
          (13, 1, 3), (13, 1, 4), (293, 1, 1), (293, 1, 2), (3, 2, 3), (3, 1, 5)]


def test_library_exports_every_declared_symbol():
    header = (ROOT / "include" / "hec.h").read_text()
    declared = set(re.findall(r"\b(hec_[a-z_A-Z0-9]+)\s*\(", header))
    declared -= {"hec_status", "hec_regime"}
    assert declared == set(hec.SYMBOLS)
    L = hec.lib()
    for name in declared:
        assert hasattr(L, name), name


def test_no_compute_without_gpu_is_loud():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(hec.HecError) as e:
        hec.count(3, 2, np.array([[1, 0, 0, 0, 0, 1, 0]], dtype=np.uint16))
    assert e.value.code == hec.HEC_ERR_CUDA


def test_invalid_fields():
    for p, r, k in [(2, 1, 1), (9, 1, 1), (15, 1, 1), (3, 0, 1), (3, 1, 0), (293, 1, 4), (3, 1, 17)]:
        with pytest.raises(hec.HecError):
            hec.build_field(p, r, k)


# every invariant below runs on the host-built tables (-m "not gpu") and on the tables built by the CUDA kernels of
# hec_build_field_device (-m gpu)
_PARAMS = [pytest.param((f, False), id=f"p{f[0]}r{f[1]}k{f[2]}") for f in FIELDS] + \
          [pytest.param((f, True), id=f"p{f[0]}r{f[1]}k{f[2]}-device", marks=pytest.mark.gpu) for f in FIELDS]


@pytest.fixture(scope="module", params=_PARAMS)
def field(request):
    f, device = request.param
    return hec.build_field_device(*f) if device else hec.build_field(*f)


@pytest.mark.gpu
@pytest.mark.parametrize("f", FIELDS + [(1009, 1, 2), (3, 1, 13), (5, 1, 9), (11, 3, 2), (3001, 1, 2)],
                         ids=lambda f: f"p{f[0]}r{f[1]}k{f[2]}")
def test_device_build_equals_host_build(f):
    """hec_build_field_device (order-test modulus search + antilog / log / Zech kernels) against hec_build_field (one
    walk through the powers of t on the host): same modulus, same tables, entry for entry."""
    H, D = hec.build_field(*f), hec.build_field_device(*f)
    assert H.modulus == D.modulus and H.Q == D.Q and H.embed_unit == D.embed_unit
    for name in ("antilog", "log", "zech", "embed"):
        assert np.array_equal(getattr(H, name), getattr(D, name)), name


def test_modulus_is_smallest_primitive(field):
    # golden list (reading G7) where present, else the oracle's own brute-force search for small fields
    golden = {}
    for line in (ROOT / "tests" / "golden" / "moduli_g7.txt").read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        left, right = line.split("|")
        golden[tuple(int(v) for v in left.split())] = [int(v) for v in right.split()]
    key = (field.p, field.n)
    if key in golden:
        assert field.modulus == golden[key]
    elif field.Q <= 30000:
        assert field.modulus == O.smallest_primitive(field.p, field.n)
    assert O.is_primitive(field.p, field.modulus) or field.Q > 200000


def test_antilog_log_are_inverse_bijections(field):
    Q, a, lg = field.Q, field.antilog, field.log
    assert a[0] == 1 and lg[0] == Q - 1                     # encoding (3.1): zero <-> Q-1
    assert sorted(a.tolist()) == list(range(1, Q))
    assert (lg[a] == np.arange(Q - 1)).all()


def test_antilog_is_multiplicative(field):
    """antilog[i] * antilog[j] = antilog[i + j mod Q-1] with the oracle's schoolbook product."""
    p, mod, a, M = field.p, field.modulus, field.antilog, field.Q - 1
    if field.n == 1:
        mod = [0, 1]          # prime field: elements are residues; oracle ring F_p[t]/(t)
    rng = np.random.default_rng(field.Q)
    pairs = [(i, 1) for i in range(min(M, 50))] + [tuple(int(v) for v in rng.integers(0, M, 2)) for _ in range(300)]
    for i, j in pairs:
        assert O.mul_encoded(p, mod, int(a[i]), int(a[j % M])) == int(a[(i + j) % M]), (i, j)


def test_zech_addition_law(field):
    """alpha^i + alpha^j = alpha^{i + Z(j - i)} (reading G5) against digit-wise addition of encodings."""
    p, n, Q = field.p, field.n, field.Q
    M, a, lg, Z = Q - 1, field.antilog.astype(np.int64), field.log, field.zech.astype(np.int64)

    def add(x, y):
        out = np.zeros_like(x)
        for d in range(n):
            out += (((x // p ** d) + (y // p ** d)) % p) * p ** d
        return out

    if M <= 700:
        i, j = np.meshgrid(np.arange(M), np.arange(M), indexing="ij")
        i, j = i.ravel(), j.ravel()
    else:
        rng = np.random.default_rng(field.Q + 1)
        i, j = rng.integers(0, M, 20000), rng.integers(0, M, 20000)
    s = add(a[i], a[j])
    z = Z[(j - i) % M]
    want = np.where(z == M, 0, a[(i + np.where(z == M, 0, z)) % M])
    assert (s == want).all()


def test_zech_invariants_g16(field):
    p, Q = field.p, field.Q
    M, Z = Q - 1, field.zech.astype(np.int64)
    e = M // 2
    assert Z[e] == M and (Z == M).sum() == 1                     # 1 + alpha^e = 0 only at e = (Q-1)/2
    ok = Z != M
    assert sorted(Z[ok].tolist()) == list(range(1, M))           # injective, image = all logs but log 1 = 0
    n = np.arange(M)
    # Z(-n) = Z(n) - n
    assert ((Z[(-n) % M][ok] - (Z[n][ok] - n[ok])) % M == 0).all()
    # Z(p n) = p Z(n)
    assert ((Z[(p * n) % M][ok] - p * Z[n][ok]) % M == 0).all()
    # W(n) = Z(n) + e is an involution on the non-sentinel entries
    W = np.where(ok, (Z + e) % M, -1)
    idx = n[ok & (W != e)]
    assert (W[W[idx]] == idx).all()
    # p-fold iterate of Z is the identity where no intermediate is the sentinel (adding 1 p times)
    cur, alive = n.copy(), np.ones(M, dtype=bool)
    for _ in range(p):
        alive &= Z[cur] != M
        cur = np.where(alive, Z[cur], 0)
    assert (cur[alive] == n[alive]).all() and alive.sum() == M - p + 1 if M >= p else True


def test_embedding_is_a_ring_homomorphism(field):
    """embed values are logs of a copy of F_q: multiples of (Q-1)/(q-1), multiplicative w.r.t. R_q and
    additive (reading G6)."""
    p, r, q, Q = field.p, field.r, field.q, field.Q
    M, emb, a, lg = Q - 1, field.embed.astype(np.int64), field.antilog.astype(np.int64), field.log.astype(np.int64)
    step = M // (q - 1)
    assert emb[0] == M and (emb[1:] % step == 0).all()
    assert emb[1] == 0                                           # 1 -> 1
    assert len(set(emb[1:].tolist())) == q - 1
    Rq = O.smallest_primitive(p, r) if r > 1 else [0, 1]
    rng = np.random.default_rng(q)
    cs = rng.integers(1, q, size=(200, 2))
    n = field.n
    for c1, c2 in cs:
        c1, c2 = int(c1), int(c2)
        prod = O.mul_encoded(p, Rq, c1, c2) if r > 1 else c1 * c2 % p
        assert (emb[c1] + emb[c2]) % M == emb[prod]
        ssum = sum((((c1 // p ** d) + (c2 // p ** d)) % p) * p ** d for d in range(r))
        x, y = int(a[emb[c1]]), int(a[emb[c2]])
        enc = sum((((x // p ** d) + (y // p ** d)) % p) * p ** d for d in range(n))
        assert int(lg[enc]) == int(emb[ssum])
    if r > 1 and field.k > 1:
        assert np.gcd(field.embed_unit, q - 1) == 1
