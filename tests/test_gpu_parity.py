"""Parity of the CUDA path (through the C ABI, paper_1805_11991_b200.hec) against the CPU oracle.

Integer work: the bar is bit-exact.  Small cases are compared element by element; at BASELINE.json's
full sizes (in the launch configuration bench.py times) the oracle checks a deterministic sample and every
row is checked against properties that hold at any size (Weil bound on squarefree rows, parity, histogram
totals, regime independence).
"""
import numpy as np
import pytest

from oracle import hec_oracle as O
from paper_1805_11991_b200 import hec, workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", params=["auto", "horner", "orbit"])
def torch_cuda(request):
    """Every test runs under all evaluation schemes of hec_count: the default (radix-R split over the cosets of
    the R-th roots of unity), the paper's one-Horner-chain-per-x scheme, and the radix split over one representative
    per Frobenius orbit (HEC_EVAL_ORBIT); the oracle is the same for all."""
    import torch
    from paper_1805_11991_b200 import build as hb
    hb.build_lib()
    assert torch.cuda.is_available()
    torch.cuda.set_device(0)
    hec.set_stream(torch.cuda.current_stream().cuda_stream)
    hec.set_regime(hec.REGIME_AUTO)
    hec.set_eval({"auto": hec.EVAL_AUTO, "horner": hec.EVAL_HORNER, "orbit": hec.EVAL_ORBIT}[request.param])
    torch.eval_scheme = request.param
    yield torch
    hec.set_eval(hec.EVAL_AUTO)


def _dev(torch, rows):
    return torch.from_numpy(np.ascontiguousarray(rows).view(np.int16)).cuda()


def _gpu_count(torch, q, g, rows):
    cnt, sf = hec.count(q, g, _dev(torch, rows))
    return cnt.cpu().numpy().view(np.uint32), sf.cpu().numpy()


def _assert_parity(torch, q, g, rows, k_hi=None):
    cnt, sf = _gpu_count(torch, q, g, rows)
    ocnt, osf, _ = O.count(q, g, rows, k_hi=k_hi)
    kk = g if k_hi is None else k_hi
    assert (cnt[:, :kk] == ocnt[:, :kk]).all(), np.argwhere(cnt[:, :kk] != ocnt[:, :kk])[:5]
    assert (sf == osf).all(), np.argwhere(sf != osf)[:5]
    return cnt, sf


# ------------------------------------------------------------------------------------------ small, element by element

def test_config1_exhaustive_device_and_host_pointers(torch_cuda):
    rows = W.generate(W.CONFIGS[1])
    cnt, sf = _assert_parity(torch_cuda, 3, 2, rows)
    # host pointers (the library stages H2D/D2H itself)
    hcnt, hsf = hec.count(3, 2, rows)
    assert (hcnt == cnt).all() and (hsf == sf).all()
    # histogram, all rows and squarefree rows only
    for mask in (None, sf):
        otup, omult = O.histogram(cnt, mask)
        tup, mult = hec.histogram(cnt, mask)
        assert (tup == otup).all() and (mult == omult).all()
        dt, dm = hec.histogram(torch_cuda.from_numpy(cnt.view(np.int32)).cuda(),
                               None if mask is None else torch_cuda.from_numpy(mask).cuda())
        assert (dt.cpu().numpy().view(np.uint32) == otup).all() and (dm.cpu().numpy().view(np.uint64) == omult).all()


@pytest.mark.parametrize("cid,n_all,n_top", [(2, 1500, 1500), (3, 160, 10), (4, 260, 70), (5, 300, 40)])
def test_config_slices_against_oracle(torch_cuda, cid, n_all, n_top):
    """First rows of each seeded workload: all N_k for n_top rows, N_k (k < g) for n_all rows.
    Sizes span several CTAs' worth of warps and a ragged tail."""
    cfg = W.CONFIGS[cid]
    rows = W.generate(cfg, 0, n_all)
    cnt, sf = _gpu_count(torch_cuda, cfg.q, cfg.g, rows)
    ocnt, osf, _ = O.count(cfg.q, cfg.g, rows, k_hi=cfg.g - 1)
    assert (cnt[:, : cfg.g - 1] == ocnt[:, : cfg.g - 1]).all()
    assert (sf == osf).all()
    otop, _, _ = O.count(cfg.q, cfg.g, rows[:n_top], k_lo=cfg.g, k_hi=cfg.g, want_squarefree=False)
    assert (cnt[:n_top, cfg.g - 1] == otop[:, cfg.g - 1]).all()


@pytest.mark.parametrize("q,g,k_hi", [(3, 2, 2), (13, 4, 3), (25, 2, 2), (49, 3, 2), (293, 2, 1), (9, 1, 1), (5, 3, 3), (27, 2, 2), (7, 5, 3)])
def test_edge_rows(torch_cuda, q, g, k_hi):
    """Degenerate inputs: monomials, c x^{2g+2} for every c, sparse rows (gaps > 1), c_0 = 0, all-(q-1)."""
    rows = W.edge_rows(q, g)
    _assert_parity(torch_cuda, q, g, rows, k_hi=k_hi)


def test_edge_rows_top_field_q13_g4(torch_cuda):
    rows = W.edge_rows(13, 4)[::3]
    _assert_parity(torch_cuda, 13, 4, rows)


@pytest.mark.parametrize("n", [1, 2, 31, 32, 33, 4735, 4737])
def test_ragged_batch_sizes(torch_cuda, n):
    cfg = W.CONFIGS[2]
    rows = W.generate(cfg, 1000, n)
    cnt, sf = _gpu_count(torch_cuda, cfg.q, cfg.g, rows)
    idx = np.unique(np.concatenate([np.arange(min(n, 40)), np.arange(max(0, n - 40), n)]))
    ocnt, osf, _ = O.count(cfg.q, cfg.g, rows[idx])
    assert (cnt[idx] == ocnt).all() and (sf[idx] == osf).all()


def test_sparse_and_zero_heavy_rows(torch_cuda):
    """Random rows with many zero coefficients (exercises every gap m_j and trailing zeros)."""
    rng = np.random.default_rng(7)
    for q, g in [(13, 2), (25, 2), (7, 3)]:
        rows = rng.integers(0, q, size=(400, 2 * g + 3)).astype(np.uint16)
        rows[rng.random(rows.shape) < 0.6] = 0
        rows[:, -1] = np.where(rng.random(400) < 0.5, rng.integers(1, q, 400), 0)
        rows[:, -2] = np.where(rows[:, -1] == 0, rng.integers(1, q, 400), rows[:, -2])
        _assert_parity(torch_cuda, q, g, rows)


def test_regimes_agree(torch_cuda):
    """Every table layout gives identical counts: full shared-memory table (extended 16-bit / 2x16-bit pairs),
    L2-resident table, shared-memory half table (32-bit for q=13^4 and 293^2, 16+8-bit or 16+1-bit planes for 49^3)."""
    radix = torch_cuda.eval_scheme in ("auto", "orbit")
    modes = {hec.REGIME_SMEM: 4, hec.REGIME_L2: 7} if radix else {hec.REGIME_SMEM: 1, hec.REGIME_L2: 0}
    h32, h24 = (5, 6) if radix else (2, 3)
    try:
        for cid, n, regimes, half_mode in [(2, 3000, (hec.REGIME_SMEM, hec.REGIME_L2), None),
                                           (4, 600, (hec.REGIME_SMEM, hec.REGIME_L2, hec.REGIME_SMEM_HALF), h32),
                                           (5, 300, (hec.REGIME_L2, hec.REGIME_SMEM_HALF, hec.REGIME_AUTO), h32),
                                           (3, 200, (hec.REGIME_L2, hec.REGIME_SMEM_HALF, hec.REGIME_AUTO), h24)]:
            cfg = W.CONFIGS[cid]
            rows = np.concatenate([W.generate(cfg, 5000, n), W.edge_rows(cfg.q, cfg.g)])
            ref = None
            for regime in regimes:
                hec.set_regime(regime)
                a, sa = _gpu_count(torch_cuda, cfg.q, cfg.g, rows)
                st = hec.last_count_stats()
                if regime == hec.REGIME_AUTO:
                    assert st["regime"] == hec.REGIME_SMEM_HALF and st["table_mode"] == half_mode
                else:
                    assert st["regime"] == regime
                    assert st["table_mode"] == (half_mode if regime == hec.REGIME_SMEM_HALF else modes[regime])
                if ref is None:
                    ref = (a, sa)
                assert (a == ref[0]).all() and (sa == ref[1]).all(), (cid, regime)
        for regime, cid in [(hec.REGIME_SMEM, 5), (hec.REGIME_SMEM_HALF, 2)]:
            hec.set_regime(regime)
            with pytest.raises(hec.HecError):
                _gpu_count(torch_cuda, W.CONFIGS[cid].q, W.CONFIGS[cid].g, W.generate(W.CONFIGS[cid], 0, 8))
    finally:
        hec.set_regime(hec.REGIME_AUTO)


@pytest.mark.parametrize("q,g,mode,min_launches", [(17, 4, 2, 2), (19, 4, 3, 3), (9, 5, 2, 2), (11, 5, 0, 2)])
def test_mixed_layout_launch_groups(torch_cuda, q, g, mode, min_launches):
    """Fields that need different layouts in one call (17^4 = 83521 and 9^5 = 59049: 32-bit half table next
    to the lower fields' extended tables; 19^4 = 130321: 16+8-bit half table in a launch of its own;
    11^5 = 161051: nothing fits, L2-resident).  Oracle on the fields k <= 3 and on a few rows of k = 4; the
    forced L2 regime must agree on everything."""
    if torch_cuda.eval_scheme in ("auto", "orbit"):        # radix tables: pairs / 32-bit half / 16+1-bit half / global pairs
        mode, min_launches = {(17, 4): (5, 2), (19, 4): (6, 3), (9, 5): (5, 2), (11, 5): (7, 2)}[(q, g)]
    rng = np.random.default_rng(q)
    rows = rng.integers(0, q, size=(70, 2 * g + 3)).astype(np.uint16)
    rows[:, -1] = np.where(rng.random(70) < 0.5, rng.integers(1, q, 70), 0)
    rows[:, -2] = np.where(rows[:, -1] == 0, rng.integers(1, q, 70), rows[:, -2])
    rows = np.concatenate([rows, W.edge_rows(q, g)[:12]])
    try:
        hec.set_regime(hec.REGIME_AUTO)
        a, sa = _gpu_count(torch_cuda, q, g, rows)
        st = hec.last_count_stats()
        assert st["launches"] >= min_launches and st["table_mode"] == mode, st
        hec.set_regime(hec.REGIME_L2)
        b, sb = _gpu_count(torch_cuda, q, g, rows)
        assert (a == b).all() and (sa == sb).all()
    finally:
        hec.set_regime(hec.REGIME_AUTO)
    ocnt, osf, _ = O.count(q, g, rows, k_hi=3)
    assert (a[:, :3] == ocnt[:, :3]).all() and (sa == osf).all()
    otop, _, _ = O.count(q, g, rows[:3], k_lo=4, k_hi=4, want_squarefree=False)
    assert (a[:3, 3] == otop[:, 3]).all()


# ------------------------------------------------------------------------------------------ boundary behaviour

def test_error_codes(torch_cuda):
    good = W.generate(W.CONFIGS[2], 0, 100)
    bad = good.copy(); bad[37, 3] = 25
    with pytest.raises(hec.HecError) as e:
        hec.count(25, 2, _dev(torch_cuda, bad))
    assert e.value.code == hec.HEC_ERR_COEFF_RANGE and e.value.index == 37
    bad = good.copy(); bad[61, 5] = 0; bad[61, 6] = 0; bad[80, 5] = 0; bad[80, 6] = 0
    with pytest.raises(hec.HecError) as e:
        hec.count(25, 2, bad)
    assert e.value.code == hec.HEC_ERR_DEGREE and e.value.index == 61
    for q, g in [(15, 2), (4, 2), (1, 2), (13, 0), (13, 6), (293, 4)]:
        with pytest.raises(hec.HecError):
            hec.count(q, g, np.zeros((1, 2 * g + 3), dtype=np.uint16))
    # mixed host / device pointers
    with pytest.raises(hec.HecError) as e:
        hec.count(25, 2, _dev(torch_cuda, good), out_counts=np.empty((100, 2), dtype=np.uint32))
    assert e.value.code == hec.HEC_ERR_INVALID_ARG
    # empty batch is a no-op
    cnt, sf = hec.count(25, 2, np.zeros((0, 7), dtype=np.uint16))
    assert cnt.shape == (0, 2)
    # the library still works after errors
    cnt, _ = hec.count(25, 2, good[:10])
    assert (cnt == O.count(25, 2, good[:10])[0]).all()


def test_histogram_random_tuples_and_capacity(torch_cuda):
    rng = np.random.default_rng(11)
    cases = [
        rng.integers(0, 50, size=(100000, 2)),                       # few distinct, heavy multiplicities
        rng.integers(0, 2 ** 20, size=(300000, 3)),                  # almost all distinct
        np.stack([rng.integers(5, 9, 50000), rng.integers(2 ** 31, 2 ** 31 + 1000, 50000)], axis=1),
        np.full((1000, 4), 7),                                       # single tuple, zero-width key
        rng.integers(0, 3, size=(5, 1)),
    ]
    for c in cases:
        c = c.astype(np.uint32)
        mask = (rng.random(len(c)) < 0.7).astype(np.uint8)
        for m in (None, mask):
            otup, omult = O.histogram(c, m)
            tup, mult = hec.histogram(c, m)
            assert tup.shape == otup.shape and (tup == otup).all() and (mult == omult).all()
            assert int(mult.sum()) == (len(c) if m is None else int(m.sum()))
    # all rows masked out
    tup, mult = hec.histogram(cases[0].astype(np.uint32), np.zeros(len(cases[0]), dtype=np.uint8))
    assert tup.shape[0] == 0
    # capacity error keeps *out_m
    import ctypes
    c = cases[0].astype(np.uint32)
    m = ctypes.c_size_t(0)
    tup = np.empty((3, 2), dtype=np.uint32); mult = np.empty(3, dtype=np.uint64)
    rc = hec.lib().hec_histogram(c.ctypes.data, None, len(c), 2, tup.ctypes.data, mult.ctypes.data, 3, ctypes.byref(m))
    assert rc == hec.HEC_ERR_CAPACITY and m.value == len(O.histogram(c)[0])
    # more than 63 bits of key
    wide = rng.integers(0, 2 ** 32, size=(100, 3), dtype=np.uint64).astype(np.uint32)
    with pytest.raises(hec.HecError) as e:
        hec.histogram(wide)
    assert e.value.code == hec.HEC_ERR_UNSUPPORTED


# ------------------------------------------------------------------------------------------ full sizes

def _full_size_checks(torch, cid, S):
    cfg = W.CONFIGS[cid]
    rows = W.generate(cfg)
    d_rows = _dev(torch, rows)
    cnt_d, sf_d = hec.count(cfg.q, cfg.g, d_rows)
    stats = hec.last_count_stats()
    cnt, sf = cnt_d.cpu().numpy().view(np.uint32), sf_d.cpu().numpy()
    # oracle on a deterministic sample
    idx = W.sample_indices(cfg, S)
    ocnt, osf, _ = O.count(cfg.q, cfg.g, rows[idx])
    assert (cnt[idx] == ocnt).all() and (sf[idx] == osf).all()
    # properties on every row
    q, g = cfg.q, cfg.g
    sq = sf == 1
    for k in range(1, g + 1):
        nk = cnt[:, k - 1].astype(np.int64)
        assert (np.abs(nk[sq] - (q ** k + 1)) <= np.floor(2 * g * q ** (k / 2))).all(), f"Weil bound, k={k}"
        assert (nk <= 2 * q ** k + 2).all()
    # squarefree density ~ 1 - 1/q
    assert abs(sq.mean() - (1 - 1 / q)) < 0.01
    # histogram of the device counts against sort + run-length
    tup_d, mult_d = hec.histogram(cnt_d, sf_d)
    otup, omult = O.histogram(cnt, sf)
    assert (tup_d.cpu().numpy().view(np.uint32) == otup).all()
    assert (mult_d.cpu().numpy().view(np.uint64) == omult).all()
    return stats


def test_full_config2(torch_cuda):
    _full_size_checks(torch_cuda, 2, 2048)


def test_full_config4_headline(torch_cuda):
    stats = _full_size_checks(torch_cuda, 4, 96)
    assert stats["regime"] == hec.REGIME_SMEM
    # 13^k - 1 = 12, 168, 2196, 28560: R = 4, 8, 4, 8
    assert stats["radix_fields"] == (0x8484 if torch_cuda.eval_scheme in ("auto", "orbit") else 0)


@pytest.mark.parametrize("cid", [2, 3, 4, 5])
def test_eval_schemes_agree_full_config(torch_cuda, cid):
    """ALL rows of every seeded workload at full size (SURVEY.md 8(c) "whole GPU path at full size, where the oracle is
    too slow"): the radix split (default) and the paper's one-Horner-chain-per-x kernel (Algorithm 1 lines 7-8,
    PAPER.md:141-143) are two independent evaluations of f at every x -- different kernels, different table layouts
    (pair / half tables against extended / half tables) -- and must give identical N_k on every row."""
    if torch_cuda.eval_scheme != "auto":
        pytest.skip("compares both schemes in one run")
    cfg = W.CONFIGS[cid]
    d_rows = _dev(torch_cuda, W.generate(cfg))
    try:
        a, _ = hec.count(cfg.q, cfg.g, d_rows, want_squarefree=False)
        assert hec.last_count_stats()["radix_fields"] != 0
        hec.set_eval(hec.EVAL_HORNER)
        b, _ = hec.count(cfg.q, cfg.g, d_rows, want_squarefree=False)
        assert hec.last_count_stats()["radix_fields"] == 0
    finally:
        hec.set_eval(hec.EVAL_AUTO)
    assert bool((a == b).all())


def test_full_config5_half_table(torch_cuda):
    stats = _full_size_checks(torch_cuda, 5, 256)
    assert stats["regime"] == hec.REGIME_SMEM_HALF and stats["table_mode"] == (5 if torch_cuda.eval_scheme in ("auto", "orbit") else 2)


def test_full_config3_half_planes(torch_cuda):
    stats = _full_size_checks(torch_cuda, 3, 64)
    assert stats["regime"] == hec.REGIME_SMEM_HALF and stats["table_mode"] == (6 if torch_cuda.eval_scheme in ("auto", "orbit") else 3)


# ------------------------------------------------------------------------------------------ radix split

@pytest.mark.parametrize("cap", [hec.EVAL_RADIX2, hec.EVAL_RADIX4, hec.EVAL_RADIX8])
def test_every_radix_against_oracle(torch_cuda, cap):
    """R = 2, 4, 8 (capped; the field decides what divides q^k - 1) on fields of every residue of q^k - 1 mod 8,
    dense and sparse rows, in every table layout the field admits: all against the oracle."""
    if torch_cuda.eval_scheme != "auto":
        pytest.skip("radix caps are set explicitly")
    rng = np.random.default_rng(cap)
    try:
        hec.set_eval(cap)
        for q, g, n in [(3, 2, 200), (7, 3, 120), (5, 3, 120), (9, 2, 300), (13, 3, 60), (27, 2, 200), (11, 1, 100), (3, 5, 60)]:
            rows = rng.integers(0, q, size=(n, 2 * g + 3)).astype(np.uint16)
            rows[rng.random(rows.shape) < 0.35] = 0
            rows[:, -1] = np.where(rng.random(n) < 0.5, rng.integers(1, q, n), 0)
            rows[:, -2] = np.where(rows[:, -1] == 0, rng.integers(1, q, n), rows[:, -2])
            rows = np.concatenate([rows, W.edge_rows(q, g)[:40]])
            ocnt, osf, _ = O.count(q, g, rows)
            for regime in (hec.REGIME_AUTO, hec.REGIME_L2):
                hec.set_regime(regime)
                cnt, sf = _gpu_count(torch_cuda, q, g, rows)
                st = hec.last_count_stats()
                assert (cnt == ocnt).all(), (q, g, cap, regime, np.argwhere(cnt != ocnt)[:5])
                assert (sf == osf).all()
                for k in range(1, g + 1):
                    R = (st["radix_fields"] >> (4 * (k - 1))) & 15
                    assert R in (2, 4, 8) and R <= cap and (q ** k - 1) % R == 0
                    assert R == cap or (q ** k - 1) % (2 * R) != 0
        # the half-table layouts on fields that admit them, against the pair layout
        for cid, n in [(4, 300), (5, 100), (3, 60)]:
            cfg = W.CONFIGS[cid]
            rows = np.concatenate([W.generate(cfg, 777, n), W.edge_rows(cfg.q, cfg.g)[:30]])
            hec.set_regime(hec.REGIME_L2)
            ref, _ = _gpu_count(torch_cuda, cfg.q, cfg.g, rows)
            hec.set_regime(hec.REGIME_SMEM_HALF)
            a, _ = _gpu_count(torch_cuda, cfg.q, cfg.g, rows)
            assert (a == ref).all(), (cid, cap)
            hec.set_eval(hec.EVAL_HORNER)
            hec.set_regime(hec.REGIME_AUTO)
            b, _ = _gpu_count(torch_cuda, cfg.q, cfg.g, rows)
            hec.set_eval(cap)
            assert (b == ref).all(), (cid, cap)
    finally:
        hec.set_regime(hec.REGIME_AUTO)
        hec.set_eval(hec.EVAL_AUTO)


# ------------------------------------------------------------------------------------------ small batches / single curve
# the workload of the paper's Table 1 is ONE genus-2 curve over F_p and
# F_{p^2}; hec_count then spreads the curve over the whole GPU (stats["splits"] warps per curve, atomics into the
# pre-zeroed counts) and, above 2^16 elements, builds the field tables with the kernels of hec_build_field_device.

TABLE1_CURVE = [17, 12, 16, 11, 10, 13, 12]     # Y^2 = 12X^6 + 13X^5 + 10X^4 + 11X^3 + 16X^2 + 12X + 17, c_0 first


@pytest.mark.parametrize("p", [101, 211, 503, 1009])
def test_table1_single_curve(torch_cuda, p):
    rows = np.array([[c % p for c in TABLE1_CURVE]], dtype=np.uint16)
    cnt, sf = _assert_parity(torch_cuda, p, 2, rows)
    st = hec.last_count_stats()
    if torch_cuda.eval_scheme in ("auto", "orbit"):
        assert st["splits"] > 1, st
    # Weil bound for a squarefree genus-2 curve
    if sf[0]:
        for k in (1, 2):
            assert abs(int(cnt[0, k - 1]) - (p ** k + 1)) <= 4 * p ** (k / 2)


def test_table1_single_curve_p3001(torch_cuda):
    if torch_cuda.eval_scheme != "auto":
        pytest.skip("one warp for 9e6 points: the split mode exists for the radix scheme only")
    p = 3001
    rows = np.array([[c % p for c in TABLE1_CURVE]], dtype=np.uint16)
    _assert_parity(torch_cuda, p, 2, rows)
    assert hec.last_count_stats()["splits"] > 1


@pytest.mark.parametrize("cid", [3, 4, 5])
@pytest.mark.parametrize("n", [1, 2, 7, 33, 300])
def test_small_batches_use_split_mode_and_agree_with_big_batches(torch_cuda, cid, n):
    cfg = W.CONFIGS[cid]
    big = W.generate(cfg, 0, 12000)             # above 2 * 148 * 32 rows: one warp per curve, no atomics
    cnt_big, sf_big = _gpu_count(torch_cuda, cfg.q, cfg.g, big)
    if torch_cuda.eval_scheme in ("auto", "orbit"):
        assert hec.last_count_stats()["splits"] == 1
    cnt, sf = _gpu_count(torch_cuda, cfg.q, cfg.g, big[:n])
    if torch_cuda.eval_scheme in ("auto", "orbit"):
        assert hec.last_count_stats()["splits"] > 1
    assert (cnt == cnt_big[:n]).all() and (sf == sf_big[:n]).all()
    m = min(n, 4 if cid == 3 else 16)
    ocnt, osf, _ = O.count(cfg.q, cfg.g, big[:m])
    assert (cnt[:m] == ocnt).all() and (sf[:m] == osf).all()


def test_split_mode_edge_rows(torch_cuda):
    """Degenerate rows (monomials, empty residue classes, zero-heavy) in split mode: few rows of a large field."""
    q, g = 293, 2
    rows = W.edge_rows(q, g)
    for lo in range(0, len(rows), 9):
        _assert_parity(torch_cuda, q, g, rows[lo:lo + 9])


# ------------------------------------------------------------------------------------------ shift pre-pass

def _poly_shift_mod_p(c, t, p):
    """Coefficients of f(X + t) over F_p (plain Horner-style Taylor shift on Python ints)."""
    b = [int(v) for v in c]
    d = len(b) - 1
    for lo in range(d):
        for j in range(d - 1, lo - 1, -1):
            b[j] = (b[j] + t * b[j + 1]) % p
    return b


def test_shift_prepass_rows_are_shifts_and_counts_do_not_change(torch_cuda):
    """hec_count evaluates f(X + t) instead of f when f has an empty residue class mod R (hec.h: hec_set_shift).
    The rows it evaluates (hec_shift_rows) must be genuine shifts with every class non-empty, and N_k, r0_k, the flag
    and lambda must equal those without the pre-pass and the oracle's."""
    if torch_cuda.eval_scheme == "horner":
        pytest.skip("the pre-pass belongs to the radix evaluation")
    cfg = W.CONFIGS[4]
    q, g = cfg.q, cfg.g
    rows = np.concatenate([W.generate(cfg, 0, 3000), W.edge_rows(q, g)])
    out = hec.shift_rows(q, g, rows)
    dev_out = hec.shift_rows(q, g, _dev(torch_cuda, rows)).cpu().numpy().view(np.uint16)
    assert (out == dev_out).all()
    changed = (out != rows).any(axis=1)
    assert 0.2 < changed[:3000].mean() < 0.45               # about a third of the uniform rows have an empty class mod 8
    nzm = out != 0
    present = np.stack([nzm[:, r::8].any(axis=1) for r in range(8)], axis=1).all(axis=1)
    assert present[:3000].mean() > 0.99
    for c, o in zip(rows[changed][:400], out[changed][:400]):
        d = int(np.flatnonzero(c)[-1])
        assert any(_poly_shift_mod_p(c[:d + 1], t, q) == [int(v) for v in o[:d + 1]] for t in range(1, q)), (c, o)
        assert (o[d + 1:] == 0).all() and o[d] == c[d]
    try:
        hec.set_shift(True)
        on = [t.cpu().numpy() for t in hec.count_ex(q, g, _dev(torch_cuda, rows))]
        hec.set_shift(False)
        off = [t.cpu().numpy() for t in hec.count_ex(q, g, _dev(torch_cuda, rows))]
    finally:
        hec.set_shift(True)
    for a, b in zip(on, off):
        assert (a == b).all()
    ocnt, osf, _ = O.count(q, g, rows[:64])
    assert (on[0].view(np.uint32)[:64] == ocnt).all() and (on[1][:64] == osf).all()


@pytest.mark.parametrize("cid", [2, 3, 5])
def test_shift_prepass_off_agrees(torch_cuda, cid):
    cfg = W.CONFIGS[cid]
    rows = W.generate(cfg, 0, 2000)
    try:
        hec.set_shift(False)
        off = _gpu_count(torch_cuda, cfg.q, cfg.g, rows)
    finally:
        hec.set_shift(True)
    on = _gpu_count(torch_cuda, cfg.q, cfg.g, rows)
    assert (on[0] == off[0]).all() and (on[1] == off[1]).all()


# ------------------------------------------------------------------------------------------ host-buffer pipeline, fused call

def test_host_pointer_pipeline_large_batch(torch_cuda):
    """Host buffers from 2^20 rows on go through the library's chunked copy/compute pipeline (hec.h: hec_count): the
    outputs must equal those of the device-pointer call on the same rows, row for row, for 2^22 rows of config 4 and all of
    config 2 -- with pinned and with pageable host memory -- and an invalid row must be reported at its index in the batch."""
    if torch_cuda.eval_scheme != "auto":
        pytest.skip("one scheme is enough: the pipeline is host-side")
    torch = torch_cuda
    for cid, n in [(4, 1 << 22), (2, 1 << 20)]:
        cfg = W.CONFIGS[cid]
        rows = W.generate(cfg, 0, n)
        d_cnt, d_sf = hec.count(cfg.q, cfg.g, _dev(torch, rows))
        assert hec.last_count_stats()["chunks"] == 1
        ref_cnt, ref_sf = d_cnt.cpu().numpy().view(np.uint32), d_sf.cpu().numpy()
        h_cnt, h_sf = hec.count(cfg.q, cfg.g, rows)                          # pageable
        assert hec.last_count_stats()["chunks"] == 4
        assert (h_cnt == ref_cnt).all() and (h_sf == ref_sf).all()
        p_rows = torch.from_numpy(rows.view(np.int16)).pin_memory()
        p_cnt = torch.empty((n, cfg.g), dtype=torch.int32).pin_memory()
        p_sf = torch.empty((n,), dtype=torch.uint8).pin_memory()
        hec.count(cfg.q, cfg.g, p_rows.numpy().view(np.uint16), p_cnt.numpy().view(np.uint32), p_sf.numpy())
        assert (p_cnt.numpy().view(np.uint32) == ref_cnt).all() and (p_sf.numpy() == ref_sf).all()
    bad = rows.copy()
    bad[3 * (n // 4) + 17, 2] = cfg.q                                        # in the last chunk
    with pytest.raises(hec.HecError) as e:
        hec.count(cfg.q, cfg.g, bad)
    assert e.value.code == hec.HEC_ERR_COEFF_RANGE and e.value.index == 3 * (n // 4) + 17
    cnt, _ = hec.count(cfg.q, cfg.g, rows[:100])                             # still works
    assert (cnt == ref_cnt[:100]).all()


@pytest.mark.parametrize("cid,n", [(1, None), (2, 70000), (2, 1 << 20), (5, 3000)])
def test_count_histogram_fused_call(torch_cuda, cid, n):
    """hec_count_histogram = hec_count + hec_histogram of the squarefree rows, host and device pointers, incl. the
    capacity retry of the binding and the pipelined host path (2^20 rows)."""
    torch = torch_cuda
    cfg = W.CONFIGS[cid]
    rows = W.generate(cfg, 0, n)
    cnt, sf = _gpu_count(torch, cfg.q, cfg.g, rows)
    otup, omult = O.histogram(cnt, sf)
    hec._cap_hint.clear()
    for kind in ("host", "device", "host"):                                  # the second host call uses the capacity hint
        if kind == "host":
            c, s, t, m = hec.count_histogram(cfg.q, cfg.g, rows)
        else:
            c, s, t, m = (x.cpu().numpy() for x in hec.count_histogram(cfg.q, cfg.g, _dev(torch, rows)))
        assert (c.view(np.uint32) == cnt).all() and (s == sf).all()
        assert t.shape == otup.shape and (t.view(np.uint32) == otup).all() and (m.view(np.uint64) == omult).all()
    # every row (no flag wanted)
    c, s, t, m = hec.count_histogram(cfg.q, cfg.g, rows, want_squarefree=False)
    atup, amult = O.histogram(cnt, None)
    assert s is None and (t == atup).all() and (m == amult).all()


@pytest.mark.parametrize("cid,n", [(2, 12000), (4, 12000), (5, 12000), (3, 10000)])
def test_fast_tables_off_agrees(torch_cuda, cid, n):
    """hec_set_fast_tables: the transposed chain-start table and the tabulated set-up change no count."""
    cfg = W.CONFIGS[cid]
    rows = np.concatenate([W.generate(cfg, 12345, n), W.edge_rows(cfg.q, cfg.g)])
    on = _gpu_count(torch_cuda, cfg.q, cfg.g, rows)
    st = hec.last_count_stats()
    if torch_cuda.eval_scheme == "auto":
        assert st["fast_fields"] != 0
    else:
        assert st["fast_fields"] == 0
    try:
        hec.set_fast_tables(False)
        off = _gpu_count(torch_cuda, cfg.q, cfg.g, rows)
        assert hec.last_count_stats()["fast_fields"] == 0
    finally:
        hec.set_fast_tables(True)
    assert (on[0] == off[0]).all() and (on[1] == off[1]).all()


@pytest.mark.parametrize("q,g,n", [(73, 1, 200), (97, 1, 200), (31, 2, 300), (49, 2, 200), (181, 2, 60), (191, 2, 60), (293, 1, 300), (17, 2, 300),
                                   (49, 3, 24), (17, 4, 16), (19, 4, 10)])
def test_monomial_class_loops_against_oracle(torch_cuda, q, g, n):
    """Genus <= 2 on fields with 8 | M (hec_radix.cuh: radix_mono_x at R = 8 for the 32-bit half table + parity table of q = 191,
    radix_mono8_packed_x for pair tables) and genus 3, 4 on half-table fields with 16 | M (radix_mono_x at R = 16: 49^3, 17^4 with
    32-bit entries, 19^4 with 16+1-bit planes): dense rows take the monomial-class loop, rows with zero coefficients are shifted
    or fall back to the general loops; both degrees; batches large enough for one warp per curve.  All against the oracle."""
    rng = np.random.default_rng(1000 * q + g)
    nc = 2 * g + 3
    rows = rng.integers(0, q, size=(n, nc)).astype(np.uint16)
    rows[: n // 4][rng.random((n // 4, nc)) < 0.3] = 0                      # some sparse rows
    rows[:, -1] = np.where(rng.random(n) < 0.5, rng.integers(1, q, n), 0)
    rows[:, -2] = np.where(rows[:, -1] == 0, rng.integers(1, q, n), rows[:, -2])
    rows = np.concatenate([rows, W.edge_rows(q, g)[:30 if g <= 2 else 6]])
    ocnt, osf, _ = O.count(q, g, rows)
    big = np.tile(rows, (12000 // len(rows) + 1, 1))                        # above 2 * 148 * 32 rows: no split mode
    cnt, sf = _gpu_count(torch_cuda, q, g, big)
    assert hec.last_count_stats()["splits"] == 1
    m = len(rows)
    assert (cnt[:m] == ocnt).all(), np.argwhere(cnt[:m] != ocnt)[:5]
    assert (sf[:m] == osf).all()
    assert (cnt.reshape(-1, m, g) == ocnt).all() and (sf.reshape(-1, m) == osf).all()          # every copy of the rows
    cnt2, sf2 = _gpu_count(torch_cuda, q, g, rows)                          # the same rows in split mode
    assert (cnt2 == ocnt).all() and (sf2 == osf).all()


@pytest.mark.parametrize("cid,n", [(2, None), (3, None), (4, None), (5, None), (1, None)])
def test_other_primitive_polynomial_full_size(torch_cuda, cid, n):
    """SURVEY.md 8(c) "whole GPU path at full size": rerun on ANOTHER primitive polynomial (hec_set_field_variant: another
    generator of every F_{q^k}, k >= 2, hence other log / Zech / embedding tables and other table indices throughout) --
    every N_k and every flag of every row must be identical.  Together with test_eval_schemes_agree_full_config (another
    kernel and table layout) this is the representation independence of the counts at full size."""
    if torch_cuda.eval_scheme != "auto":
        pytest.skip("one scheme is enough: the field build is shared")
    cfg = W.CONFIGS[cid]
    d_rows = _dev(torch_cuda, W.generate(cfg))
    a, sa = hec.count(cfg.q, cfg.g, d_rows)
    try:
        for v in ((1,) if cid == 1 else (1, 2)):                         # F_9 has only two primitive quadratics
            hec.set_field_variant(v)
            b, sb = hec.count(cfg.q, cfg.g, d_rows)
            assert bool((a == b).all()) and bool((sa == sb).all()), (cid, v)
    finally:
        hec.set_field_variant(0)


def test_other_primitive_polynomial_changes_the_tables_not_the_map(torch_cuda):
    """Algorithm 1's map (lambda included) and hec_count_ex's root counts and lambda do not notice the other representation."""
    if torch_cuda.eval_scheme != "auto":
        pytest.skip("one scheme is enough")
    ref = hec.curve_map(7, 2, 6, True)
    rows = W.generate(W.CONFIGS[3], 0, 6000)
    r0 = hec.count_ex(49, 3, _dev(torch_cuda, rows))
    try:
        hec.set_field_variant(1)
        got = hec.curve_map(7, 2, 6, True)
        r1 = hec.count_ex(49, 3, _dev(torch_cuda, rows))
    finally:
        hec.set_field_variant(0)
    assert (ref[0] == got[0]).all() and (ref[1] == got[1]).all()
    for x, y in zip(r0, r1):
        assert bool((x == y).all())


def test_field_variant_beyond_the_fields_polynomials_and_shutdown_resets(torch_cuda):
    """F_9 has two primitive quadratics: variant 2 cannot be built and the error says so (not "no primitive polynomial
    found"); hec_shutdown puts the variant and the stream setting back to their defaults (hec.h)."""
    if torch_cuda.eval_scheme != "auto":
        pytest.skip("one scheme is enough")
    rows = W.generate(W.CONFIGS[1])
    ref, _ = hec.count(3, 2, _dev(torch_cuda, rows))
    try:
        hec.set_field_variant(2)
        with pytest.raises(hec.HecError) as e:
            hec.count(3, 2, _dev(torch_cuda, rows))
        assert e.value.code == hec.HEC_ERR_INVALID_FIELD and "variant 2" in str(e.value)
        hec.set_field_variant(1)
        hec.shutdown()                                                   # variant back to 0, stream back to the default
        got, _ = hec.count(3, 2, _dev(torch_cuda, rows))
        assert bool((got == ref).all())
        assert hec.last_count_stats()["launches"] >= 1
    finally:
        hec.set_field_variant(0)
        hec.set_stream(torch_cuda.cuda.current_stream().cuda_stream)
