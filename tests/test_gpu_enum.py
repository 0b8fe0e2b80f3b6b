"""GPU parity for SURVEY.md 8(f) NEXT-1 (hec_reduced_rows, hec_curve_map) against oracle/hec_enum_oracle.py.

The two sides choose DIFFERENT coset representatives R_m (library: powers of its generator; oracle: smallest
encodings), so they enumerate different reduced sets; what is unique -- the weighted map N_{g,d} -- must agree
bit for bit, and the library's rows are checked for validity (reduced form, distinct cosets, multiplicities)."""
import math

import numpy as np
import pytest

from oracle import hec_enum_oracle as E
from paper_1805_11991_b200 import hec

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def cuda():
    import torch
    from paper_1805_11991_b200 import build as hb
    hb.build_lib()
    assert torch.cuda.is_available()
    torch.cuda.set_device(0)
    hec.set_stream(torch.cuda.current_stream().cuda_stream)
    hec.set_regime(hec.REGIME_AUTO)
    hec.set_eval(hec.EVAL_AUTO)
    return torch


@pytest.mark.parametrize("q,g,d", [(3, 2, 5), (5, 2, 6), (7, 2, 5), (9, 2, 5), (25, 2, 6), (13, 4, 9), (49, 3, 8),
                                   (3, 2, 6), (3, 1, 3), (5, 2, 5), (25, 2, 5), (49, 3, 7), (9, 1, 3)])
def test_reduced_rows_are_valid(cuda, q, g, d):
    total = hec.reduced_total(q, g, d)
    assert total == sum(1 for _ in E.reduced_polynomials(q, d)) if total < 300000 else total > 0
    n = min(total, 200000)
    first = 0 if total == n else total - n                 # the tail holds the large families
    rows, mult = hec.reduced_rows(q, g, d, first, n)
    drows, dmult = hec.reduced_rows(q, g, d, first, n, device="cuda")
    assert (drows.cpu().numpy().view(np.uint16) == rows).all() and (dmult.cpu().numpy().view(np.uint64) == mult).all()
    # ragged sub-range addressed by index
    off = min(17, n // 2)
    sub, smult = hec.reduced_rows(q, g, d, first + off, min(n - off, 1001))
    assert (sub == rows[off:off + len(sub)]).all() and (smult == mult[off:off + len(sub)]).all()
    p = E.Fq(q).p
    assert (rows[:, d] != 0).all() and (rows[:, d + 1:] == 0).all() and (rows < q).all()
    if d % p:
        assert (rows[:, d - 1] == 0).all()
    else:
        assert ((rows[:, d - 1] == 0) | (rows[:, d - 2] == 0)).all()           # reading G19: c_{d-2} = 0 where c_{d-1} != 0
    assert len(np.unique(rows, axis=0)) == n
    F = E.Fq(q)
    cosets = {}
    for c, m in zip(rows[:: max(1, n // 4000)], mult[:: max(1, n // 4000)]):
        shifted = d % p != 0 or c[d - 1] != 0                    # stratum reduced with the shift: group of order q (q-1)^2
        top = d - 1 if (d % p != 0 or c[d - 1] == 0) else d - 2
        group = q * (q - 1) ** 2 if shifted else (q - 1) ** 2
        supp = np.flatnonzero(c[:top])
        i = supp[-1]
        assert c[i] == 1
        if len(supp) == 1:
            assert i in (0, 1) and m == group // (2 * (q - 1))
        else:
            j = supp[-2]
            assert m == group // (2 * math.gcd(q - 1, i - j))
            cosets.setdefault((int(i), int(j)), set()).add(int(c[j]))
    for (i, j), reps in cosets.items():                      # the c_j seen lie in pairwise different cosets of (i-j)-th powers
        gam = math.gcd(q - 1, i - j)
        assert len(reps) <= gam
        reps = sorted(reps)
        for a in range(len(reps)):
            for b in range(a):
                assert F.pow(F.mul(reps[a], F.inv(reps[b])), (q - 1) // gam) != 1


@pytest.mark.parametrize("q,g,d", [(3, 2, 5), (3, 1, 4), (5, 1, 3), (5, 1, 4), (7, 1, 3), (7, 1, 4), (5, 2, 6), (7, 2, 5),
                                   (3, 1, 3), (3, 2, 6), (5, 2, 5), (9, 1, 3)])               # the last four: p | d
def test_curve_map_equals_the_definition(cuda, q, g, d):
    tup, w = hec.curve_map(q, g, d)
    otup, ow = E.map_to_arrays(E.brute_force_map(q, g, d), g)
    assert tup.shape == otup.shape and (tup == otup).all() and (w == ow).all()


@pytest.mark.parametrize("q,g,d", [(9, 2, 5), (11, 2, 6), (13, 2, 5), (13, 2, 6), (25, 1, 4), (27, 1, 4), (7, 3, 8),
                                   (9, 2, 6), (7, 3, 7), (27, 1, 3)])                     # the last three: p | d
def test_curve_map_equals_algorithm1_oracle(cuda, q, g, d):
    tup, w = hec.curve_map(q, g, d)
    otup, ow = E.map_to_arrays(E.reduced_map(q, g, d), g)
    assert tup.shape == otup.shape and (tup == otup).all() and (w == ow).all()
    assert int(w.sum()) == (q - 1) * (q ** d - q ** (d - 1))


def test_curve_map_multichunk(cuda):
    """More than one chunk of reduced polynomials (q = 13, g = 3, d = 8: 5.66e6 rows in chunks of 2^21): the map against the same
    pipeline assembled by hand with another chunking (hec_reduced_rows -> hec_count -> numpy), the closed-form total
    and the twist symmetry."""
    q, g, d = 13, 3, 8
    total = hec.reduced_total(q, g, d)
    assert total > 2 * (1 << 21)
    hec.set_map_chunk_rows(1 << 21)
    try:
        tup, w = hec.curve_map(q, g, d)
    finally:
        hec.set_map_chunk_rows(1 << 24)
    assert int(w.sum()) == (q - 1) * (q ** d - q ** (d - 1))
    acc = {}
    step = 1_500_001
    for first in range(0, total, step):
        n = min(step, total - first)
        rows, mult = hec.reduced_rows(q, g, d, first, n, device="cuda")
        cnt, sf = hec.count(q, g, rows)
        cnt = cnt.cpu().numpy().view(np.uint32).astype(np.uint64)
        keep = sf.cpu().numpy() != 0
        key = (cnt[:, 0] << np.uint64(44)) | (cnt[:, 1] << np.uint64(22)) | cnt[:, 2]
        m = mult.cpu().numpy().view(np.uint64)
        u, inv = np.unique(key[keep], return_inverse=True)
        s = np.zeros(len(u), dtype=np.uint64)
        np.add.at(s, inv, m[keep])
        for k, v in zip(u.tolist(), s.tolist()):
            acc[k] = acc.get(k, 0) + v
    full = {}
    for k, v in acc.items():
        t = (k >> 44, (k >> 22) & ((1 << 22) - 1), k & ((1 << 22) - 1))
        for tt in (t, E.twist_tuple(q, t)):
            full[tt] = full.get(tt, 0) + v
    otup, ow = E.map_to_arrays(full, g)
    assert tup.shape == otup.shape and (tup == otup).all() and (w == ow).all()


@pytest.mark.parametrize("q,g,d,lam", [(13, 2, 5, False), (7, 3, 7, True), (5, 2, 5, True)])
def test_curve_map_ranges_merge_to_the_map(cuda, q, g, d, lam):
    """The multi-GPU form: the ranks' hec_curve_map_range outputs over a partition of the index range, merged with
    hec_histogram_merge (the one exchange step), equal hec_curve_map."""
    from paper_1805_11991_b200 import workloads as W
    total = hec.reduced_total(q, g, d)
    parts_t, parts_w = [], []
    for r in range(3):
        lo, hi = W.shard_range(total, r, 3)
        t, w = hec.curve_map(q, g, d, with_lambda=lam, index_range=(lo, hi - lo))
        parts_t.append(t)
        parts_w.append(w)
    mt, mw = hec.histogram_merge(np.concatenate(parts_t), np.concatenate(parts_w))
    ft, fw = hec.curve_map(q, g, d, with_lambda=lam)
    assert mt.shape == ft.shape and (mt == ft).all() and (mw == fw).all()
    et, ew = hec.curve_map(q, g, d, with_lambda=lam, index_range=(5, 0))
    assert len(et) == 0 and len(ew) == 0


@pytest.mark.parametrize("q,g", [(3, 1), (5, 1), (7, 1), (3, 2), (5, 2)])
def test_curve_map_all_is_the_union_of_both_degrees(cuda, q, g):
    """Algorithm 1 line 2: N_{g,q} over d = 2g+1 and 2g+2, against the definition (brute force over both degrees)."""
    want = {}
    for d in (2 * g + 1, 2 * g + 2):
        for t, x in E.brute_force_map(q, g, d).items():
            want[t] = want.get(t, 0) + x
    tup, w = hec.curve_map_all(q, g)
    otup, ow = E.map_to_arrays(want, g)
    assert tup.shape == otup.shape and (tup == otup).all() and (w == ow).all()
    keys, wl = hec.curve_map_all(q, g, with_lambda=True)
    parts = hec.lambda_partitions(g)
    got = {(tuple(int(v) for v in k[:g]), parts[int(k[g])]): int(x) for k, x in zip(keys, wl)}
    wantl = {}
    for d in (2 * g + 1, 2 * g + 2):
        for key, x in E.brute_force_map_lambda(q, g, d).items():
            wantl[key] = wantl.get(key, 0) + x
    assert got == wantl


@pytest.mark.parametrize("q,g,d,lam", [(13, 2, 5, False), (7, 3, 7, True)])
def test_device_resident_curve_map_and_exchange_merge(cuda, q, g, d, lam):
    """The device flow of distributed.global_curve_map on ONE GPU: hec_curve_map_range with device=True (outputs written
    into CUDA tensors) equals the host-output call, and the gathered partial maps -- here simply concatenated, as the
    all-gather would deliver them -- go through distributed._to_device / distributed._merge (hec_histogram_merge on the
    device, ordered on torch's stream) to the full map."""
    from paper_1805_11991_b200 import distributed as D, workloads as W
    torch = cuda
    total = hec.reduced_total(q, g, d)
    parts_t, parts_w = [], []
    for r in range(2):
        lo, hi = W.shard_range(total, r, 2)
        ht, hw = hec.curve_map(q, g, d, with_lambda=lam, index_range=(lo, hi - lo))
        dt, dw = hec.curve_map(q, g, d, with_lambda=lam, index_range=(lo, hi - lo), device=True)
        assert dt.is_cuda and dw.is_cuda
        assert (dt.cpu().numpy().view(np.uint32) == ht).all() and (dw.cpu().numpy().view(np.uint64) == hw).all()
        parts_t.append(D._to_device(dt, torch.int32))
        parts_w.append(D._to_device(hw, torch.int64))                          # numpy input: the host-to-device branch
    mt, mw = D._merge(torch.cat(parts_t), torch.cat(parts_w))
    ft, fw = hec.curve_map(q, g, d, with_lambda=lam)
    assert mt.is_cuda and (mt.cpu().numpy().view(np.uint32) == ft).all() and (mw.cpu().numpy().view(np.uint64) == fw).all()


def test_global_curve_map_single_rank(cuda):
    """distributed.global_curve_map without a process group is hec_curve_map (the N > 1 exchange is all-gather +
    hec_histogram_merge, covered by test_curve_map_ranges_merge_to_the_map and the gloo tests)."""
    from paper_1805_11991_b200 import distributed as D
    a = D.global_curve_map(5, 2, 6, with_lambda=True)
    b = hec.curve_map(5, 2, 6, with_lambda=True)
    assert (a[0] == b[0]).all() and (a[1] == b[1]).all()


def test_errors(cuda):
    with pytest.raises(hec.HecError) as e:
        hec.reduced_total(7, 2, 4)
    assert e.value.code == hec.HEC_ERR_INVALID_ARG
    with pytest.raises(hec.HecError):
        hec.reduced_rows(7, 2, 5, hec.reduced_total(7, 2, 5) - 3, 4)
