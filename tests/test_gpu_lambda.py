"""GPU parity for SURVEY.md 8(f) NEXT-3: r0_k and lambda(f) from hec_count_ex, and the map with the full key (1.2),
against oracle/hec_lambda_oracle.py (root counts up to F_{q^(g+1)}, one field more than the device uses; the device
settles the remaining case by the discriminant's quadratic character, the oracle by counting roots)."""
import numpy as np
import pytest

from oracle import hec_enum_oracle as E
from oracle import hec_lambda_oracle as LO
from oracle import hec_oracle as O
from paper_1805_11991_b200 import hec, workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", params=["auto", "horner"])
def cuda(request):
    import torch
    from paper_1805_11991_b200 import build as hb
    hb.build_lib()
    assert torch.cuda.is_available()
    torch.cuda.set_device(0)
    hec.set_stream(torch.cuda.current_stream().cuda_stream)
    hec.set_regime(hec.REGIME_AUTO)
    hec.set_eval(hec.EVAL_AUTO if request.param == "auto" else hec.EVAL_HORNER)
    yield torch
    hec.set_eval(hec.EVAL_AUTO)


def _check(torch, q, g, rows, device=True):
    parts = hec.lambda_partitions(g)
    assert parts == LO.partitions(2 * g + 2)
    src = torch.from_numpy(np.ascontiguousarray(rows).view(np.int16)).cuda() if device else rows
    cnt, sf, r0, lam = hec.count_ex(q, g, src)
    if device:
        cnt, sf, r0, lam = (t.cpu().numpy() for t in (cnt, sf, r0, lam))
        cnt, r0 = cnt.view(np.uint32), r0.view(np.uint32)
    ocnt, osf, _ = O.count(q, g, rows)
    assert (cnt == ocnt).all() and (sf == osf).all()
    assert (r0 == O.roots(q, g, rows)).all()
    want = LO.lambda_by_roots(q, g, rows)
    got = [None if v == 0xFF else parts[v] for v in lam.tolist()]
    assert got == want, [(i, a, b) for i, (a, b) in enumerate(zip(got, want)) if a != b][:5]
    return got


def test_config1_exhaustive(cuda):
    rows = W.generate(W.CONFIGS[1])
    got = _check(cuda, 3, 2, rows)
    _check(cuda, 3, 2, rows[:777], device=False)                      # host pointers
    # both outcomes of the case the g fields leave open (irreducible sextic / two irreducible cubics) occur
    assert (0, 0, 0, 0, 0, 1) in got and (0, 0, 2, 0, 0, 0) in got


@pytest.mark.parametrize("q,g,n", [(5, 1, 3000), (7, 1, 3000), (9, 1, 2000), (5, 2, 3000), (7, 2, 3000), (13, 2, 1500),
                                   (25, 2, 300), (7, 3, 300), (13, 3, 120), (13, 4, 48)])
def test_random_rows(cuda, q, g, n):
    rng = np.random.default_rng(1805 + q * 10 + g)
    rows = rng.integers(0, q, size=(n, 2 * g + 3)).astype(np.uint16)
    rows[::2, 2 * g + 2] = 0
    rows[rows[:, 2 * g + 2] == 0, 2 * g + 1] = 1 + rng.integers(0, q - 1)
    got = [t for t in _check(cuda, q, g, rows) if t is not None]
    if n >= 1500:
        irreducible = tuple([0] * (2 * g + 1) + [1])
        two_halves = tuple([0] * g + [2] + [0] * (g + 1))
        assert irreducible in got and two_halves in got


@pytest.mark.parametrize("cid,n", [(5, 16), (3, 8), (4, 5)])
def test_small_batches_split_mode(cuda, cid, n):
    """Few curves of a large field: r0 is accumulated with atomics over the parts (hec_count_stats.splits > 1)."""
    cfg = W.CONFIGS[cid]
    _check(cuda, cfg.q, cfg.g, W.generate(cfg, 0, n))


@pytest.mark.parametrize("q,g,d", [(3, 2, 5), (5, 1, 3), (5, 1, 4), (7, 1, 4), (5, 2, 6), (7, 2, 5), (13, 2, 5), (7, 3, 8)])
def test_curve_map_with_lambda(cuda, q, g, d):
    keys, w = hec.curve_map(q, g, d, with_lambda=True)
    parts = hec.lambda_partitions(g)
    got = {(tuple(int(v) for v in k[:g]), parts[int(k[g])]): int(x) for k, x in zip(keys, w)}
    assert got == E.reduced_map_lambda(q, g, d)
    # marginal over lambda = the map without lambda
    tup, w0 = hec.curve_map(q, g, d)
    marg = {}
    for (t, _), x in got.items():
        marg[t] = marg.get(t, 0) + x
    assert marg == {tuple(int(v) for v in t): int(x) for t, x in zip(tup, w0)}
