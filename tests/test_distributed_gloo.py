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


def test_allgather_histograms_world2_gloo():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ret = mp.Manager().dict()
    mp.spawn(_worker, args=(2, port, ret), nprocs=2, join=True)
    assert dict(ret) == {0: True, 1: True}
