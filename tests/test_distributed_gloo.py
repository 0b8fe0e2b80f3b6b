"""N > 1 host logic on CPU (gloo, world_size 2): the curve sharding and the histogram exchange step.
The merge kernel itself (hec_histogram_merge) is CUDA and is covered by the -m gpu tests."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1805_11991_b200 import distributed as D, workloads as W


def test_shard_range_partitions_every_size():
    for n in [0, 1, 2, 7, 1944, 1 << 20, (1 << 24) + 3]:
        for world in [1, 2, 3, 4, 8]:
            spans = [W.shard_range(n, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
            sizes = [hi - lo for lo, hi in spans]
            assert max(sizes) - min(sizes) <= 1


def test_rows_are_index_addressable_across_ranks():
    """Any rank regenerates exactly the rows of its shard: generate(start, count) == rows_by_index(range)."""
    for cid in (2, 3, 4, 5):
        cfg = W.CONFIGS[cid]
        whole = W.generate(cfg, 1000, 64)
        parts = [W.generate(cfg, 1000 + lo, hi - lo) for lo, hi in (W.shard_range(64, r, 2) for r in range(2))]
        assert (np.concatenate(parts) == whole).all()
        assert (W.rows_by_index(cfg, np.arange(1000, 1064)) == whole).all()
        assert whole.max() < cfg.q
        assert ((whole[:, -1] != 0) | (whole[:, -2] != 0)).all()


def _worker(rank, world, port, ret):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        rng = np.random.default_rng(5)
        counts = rng.integers(0, 6, size=(1001, 2)).astype(np.int32)          # same on every rank
        lo, hi = W.shard_range(len(counts), rank, world)
        tup, mult = np.unique(counts[lo:hi], axis=0, return_counts=True)      # stand-in for hec_histogram
        all_t, all_m = D.allgather_histograms(torch.from_numpy(tup), torch.from_numpy(mult.astype(np.int64)))
        # merge on the host (test only) and compare with the histogram of all rows
        mt, inv = np.unique(all_t.numpy(), axis=0, return_inverse=True)
        mm = np.bincount(inv.ravel(), weights=all_m.numpy()).astype(np.int64)
        wt, wm = np.unique(counts, axis=0, return_counts=True)
        ok = mt.shape == wt.shape and (mt == wt).all() and (mm == wm).all() and int(all_m.sum()) == len(counts)
        # ragged: rank 1 contributes nothing
        e_t = torch.from_numpy(tup if rank == 0 else tup[:0])
        e_m = torch.from_numpy((mult if rank == 0 else mult[:0]).astype(np.int64))
        g_t, g_m = D.allgather_histograms(e_t, e_m)
        t0, m0 = np.unique(counts[: W.shard_range(len(counts), 0, world)[1]], axis=0, return_counts=True)
        ok = ok and g_t.shape[0] == len(t0) and (g_t.numpy() == t0).all() and (g_m.numpy() == m0).all()
        ret[rank] = bool(ok)
    finally:
        dist.destroy_process_group()


def _np_merge(all_t, all_m):
    """numpy stand-in for hec_histogram_merge (a CUDA kernel): sorted distinct tuples, summed multiplicities."""
    t, m = all_t.numpy(), all_m.numpy()
    if len(t) == 0:
        return torch.from_numpy(t), torch.from_numpy(m)
    ut, inv = np.unique(t, axis=0, return_inverse=True)
    um = np.zeros(len(ut), dtype=np.int64)
    np.add.at(um, inv.ravel(), m)
    return torch.from_numpy(ut), torch.from_numpy(um)


def _fake_partial_map(lo, n, cols):
    """Stand-in for hec_curve_map_range: a deterministic 'map' of the index range [lo, lo + n) whose merge over any
    partition of [0, total) is the same."""
    i = np.arange(lo, lo + n, dtype=np.int64)
    keys = np.stack([(i * 7) % 11] + [(i // 3) % 5] * (cols - 1), axis=1).astype(np.uint32)
    ut, inv = np.unique(keys, axis=0, return_inverse=True)
    w = np.zeros(len(ut), dtype=np.uint64)
    np.add.at(w, inv.ravel(), (i % 13 + 1).astype(np.uint64))
    return ut, w


def _worker_global(rank, world, port, ret):
    """Control flow of global_histogram / global_curve_map with world = 2: library calls replaced by numpy stand-ins,
    exchange on CPU tensors over gloo."""
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from paper_1805_11991_b200 import hec
        D._exchange_device = lambda: torch.device("cpu")
        D._merge = _np_merge
        total = 1001

        def fake_histogram(counts, mask=None, _weights=None):
            c = np.asarray(counts)
            if mask is not None:
                c = c[np.asarray(mask) != 0]
            t, m = np.unique(c, axis=0, return_counts=True)
            return t.astype(np.uint32), m.astype(np.uint64)

        def fake_curve_map(q, g, d, with_lambda=False, index_range=None, device=False):
            lo, n = index_range if index_range is not None else (0, total)
            return _fake_partial_map(lo, n, g + 1 if with_lambda else g)

        hec.histogram, hec.curve_map, hec.reduced_total = fake_histogram, fake_curve_map, lambda q, g, d: total
        rng = np.random.default_rng(9)
        counts = rng.integers(0, 5, size=(777, 3)).astype(np.uint32)          # same on every rank
        mask = (rng.random(777) < 0.8).astype(np.uint8)
        lo, hi = W.shard_range(len(counts), rank, world)
        ok = True
        for msk in (None, mask):                                              # numpy inputs, world > 1
            t, m = D.global_histogram(counts[lo:hi], None if msk is None else msk[lo:hi])
            wt, wm = fake_histogram(counts, msk)
            ok = ok and (t.numpy().view(np.uint32) == wt).all() and (m.numpy().view(np.uint64) == wm).all()
        for lam in (False, True):
            keys, w = D.global_curve_map(13, 2, 6, with_lambda=lam)
            wk, ww = _fake_partial_map(0, total, 3 if lam else 2)
            ok = ok and keys.shape == wk.shape and (keys == wk).all() and (w == ww).all()
        ret[rank] = bool(ok)
    finally:
        dist.destroy_process_group()


def test_global_histogram_and_curve_map_control_flow_world2_gloo():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ret = mp.Manager().dict()
    mp.spawn(_worker_global, args=(2, port, ret), nprocs=2, join=True)
    assert dict(ret) == {0: True, 1: True}


def test_allgather_histograms_world2_gloo():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ret = mp.Manager().dict()
    mp.spawn(_worker, args=(2, port, ret), nprocs=2, join=True)
    assert dict(ret) == {0: True, 1: True}
