"""N > 1 on hardware: two ranks over NCCL, one GPU each.  Skipped on boxes with fewer than two GPUs
(this build only ever saw one: row 8(e) is unmeasured on hardware)."""
import os
import socket

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _worker(rank, world, port, ret):
    import torch
    import torch.distributed as dist
    from paper_1805_11991_b200 import distributed as D, hec, workloads as W
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", rank))
    try:
        hec.set_stream(torch.cuda.current_stream().cuda_stream)
        cfg = W.CONFIGS[2]
        n = 20001
        rows = W.generate(cfg, 0, n)
        lo, hi = W.shard_range(n, rank, world)
        d_rows = torch.from_numpy(rows[lo:hi].view(np.int16)).cuda()
        cnt, sf = hec.count(cfg.q, cfg.g, d_rows)
        tup, mult = D.global_histogram(cnt, sf)                               # device tensors
        ht, hm = D.global_histogram(cnt.cpu().numpy().view(np.uint32), sf.cpu().numpy())      # numpy inputs, world > 1
        wcnt, wsf = hec.count(cfg.q, cfg.g, torch.from_numpy(rows.view(np.int16)).cuda())
        wt, wm = hec.histogram(wcnt, wsf)
        ok = bool((tup == wt).all() and (mult == wm).all() and (ht == wt).all() and (hm == wm).all())
        keys, w = D.global_curve_map(5, 2, 6, with_lambda=True)
        k1, w1 = hec.curve_map(5, 2, 6, True)
        ok = ok and keys.shape == k1.shape and bool((keys == k1).all() and (w == w1).all())
        ret[rank] = ok
    finally:
        dist.destroy_process_group()


def test_global_histogram_and_curve_map_world2_nccl():
    import torch
    import torch.multiprocessing as mp
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ret = mp.Manager().dict()
    mp.spawn(_worker, args=(2, port, ret), nprocs=2, join=True)
    assert dict(ret) == {0: True, 1: True}
