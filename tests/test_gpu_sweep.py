"""Sweep over every field the paper's ranges contain (q < 300 for g = 2, q < 50 for g = 3, q < 15 for g = 4; here
also g = 1 up to 300, g = 4 up to 17, g = 5 up to 9): for each (q, g) a small seeded batch -- dense rows, zero-heavy rows, both
degrees, edge rows -- is counted by the oracle and, tiled to a batch large enough for one warp per curve, by all three evaluation
schemes of the library (radix split with whatever table layout, fast tables and specialised loops the field gets; the paper's
one-Horner-chain-per-x kernel; the Frobenius-orbit scheme), and once more as a small batch (split mode).  Bit-exact."""
import numpy as np
import pytest

from oracle import hec_oracle as O
from paper_1805_11991_b200 import hec, workloads as W

pytestmark = pytest.mark.gpu


def _prime_powers(lim):
    out = []
    for q in range(3, lim + 1, 2):
        p = next(d for d in range(3, q + 1, 2) if q % d == 0)
        v = q
        while v % p == 0:
            v //= p
        if v == 1 and all(p % e for e in range(2, int(p ** 0.5) + 1)):
            out.append(q)
    return out


CASES = ([(q, 1) for q in _prime_powers(300)] + [(q, 2) for q in _prime_powers(300)] + [(q, 3) for q in _prime_powers(49)] +
         [(q, 4) for q in _prime_powers(17)] + [(q, 5) for q in _prime_powers(9)])


@pytest.fixture(scope="module")
def cuda():
    import torch
    from paper_1805_11991_b200 import build as hb
    hb.build_lib()
    assert torch.cuda.is_available()
    torch.cuda.set_device(0)
    hec.set_stream(torch.cuda.current_stream().cuda_stream)
    hec.set_regime(hec.REGIME_AUTO)
    yield torch
    hec.set_eval(hec.EVAL_AUTO)


@pytest.mark.parametrize("part", range(8))
def test_every_field_every_scheme_against_oracle(cuda, part):
    rng = np.random.default_rng(1805 + part)
    for q, g in CASES[part::8]:
        nc, Q = 2 * g + 3, q ** g
        n_or = max(4, min(60, int(3e6 / Q)))
        rows = rng.integers(0, q, size=(n_or, nc)).astype(np.uint16)
        rows[: n_or // 3][rng.random((n_or // 3, nc)) < 0.3] = 0
        rows[:, -1] = np.where(rng.random(n_or) < 0.5, rng.integers(1, q, n_or), 0)
        rows[:, -2] = np.where(rows[:, -1] == 0, rng.integers(1, q, n_or), rows[:, -2])
        rows = np.concatenate([rows, W.edge_rows(q, g)[:8]])
        ocnt, osf, _ = O.count(q, g, rows)
        m = len(rows)
        reps = max(1, min(12000 // m + 1, int(4e9 / (Q * m)) + 1))
        d = cuda.from_numpy(np.tile(rows, (reps, 1)).view(np.int16)).cuda()
        try:
            for name, ev in (("auto", hec.EVAL_AUTO), ("horner", hec.EVAL_HORNER), ("orbit", hec.EVAL_ORBIT)):
                hec.set_eval(ev)
                c, s = hec.count(q, g, d)
                c, s = c.cpu().numpy().view(np.uint32), s.cpu().numpy()
                assert (c.reshape(-1, m, g) == ocnt).all() and (s.reshape(-1, m) == osf).all(), (q, g, name, hec.last_count_stats())
        finally:
            hec.set_eval(hec.EVAL_AUTO)
        c, s = hec.count(q, g, rows)                                         # small batch: split mode where the field is large
        assert (c == ocnt).all() and (s == osf).all(), (q, g, "small batch")
    hec.shutdown()                                                           # plans of ~20 fields: release them
