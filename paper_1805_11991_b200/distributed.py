"""Multi-GPU plumbing: curves are independent, so `hec_count` shards by contiguous curve
range with NO data-path collective; only the tuple histogram has an exchange step -- an all-gather of the
ranks' sparse (tuple, multiplicity) lists followed by `hec_histogram_merge` on every rank.

One process per GPU, `torch.distributed` for the plumbing (NCCL over NVLink on GPUs; the same code runs on
gloo/CPU tensors in the tests, where only the gather is exercised -- the merge itself is a CUDA kernel).
"""
from __future__ import annotations

import os


def init_from_env():
    """(rank, local_rank, world) from torchrun's environment; initialises NCCL when world > 1."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch
        import torch.distributed as dist
        torch.cuda.set_device(local_rank)
        if not dist.is_initialized():
            dist.init_process_group(backend="nccl", device_id=torch.device("cuda", local_rank))
    return rank, local_rank, world


def allgather_histograms(tuples, mult, group=None):
    """All-gather variable-length partial histograms.

    tuples: [m][g] integer tensor, mult: [m] int64 tensor (both on the backend's device).
    Returns (all_tuples [sum m_r][g], all_mult [sum m_r]) -- the concatenation over ranks in rank
    order, tuples possibly repeated across ranks.  Lists are padded to the longest rank for the collective
    and trimmed afterwards.
    """
    import torch
    import torch.distributed as dist

    world = dist.get_world_size(group)
    m = torch.tensor([tuples.shape[0]], dtype=torch.int64, device=tuples.device)
    sizes = [torch.zeros_like(m) for _ in range(world)]
    dist.all_gather(sizes, m, group=group)
    sizes = [int(s.item()) for s in sizes]
    mmax = max(sizes)
    g = tuples.shape[1]
    pad_t = torch.zeros((mmax, g), dtype=tuples.dtype, device=tuples.device)
    pad_m = torch.zeros((mmax,), dtype=mult.dtype, device=mult.device)
    pad_t[: tuples.shape[0]] = tuples
    pad_m[: mult.shape[0]] = mult
    out_t = [torch.empty_like(pad_t) for _ in range(world)]
    out_m = [torch.empty_like(pad_m) for _ in range(world)]
    dist.all_gather(out_t, pad_t, group=group)
    dist.all_gather(out_m, pad_m, group=group)
    all_t = torch.cat([t[:s] for t, s in zip(out_t, sizes)], dim=0)
    all_m = torch.cat([x[:s] for x, s in zip(out_m, sizes)], dim=0)
    return all_t, all_m


def global_histogram(counts, mask, group=None):
    """Per-rank `hec_histogram` + all-gather + `hec_histogram_merge`: every rank returns the histogram of
    the union of all ranks' rows.  With one rank this is just `hec_histogram`."""
    import torch.distributed as dist
    from . import hec

    tup, mult = hec.histogram(counts, mask)
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return tup, mult
    all_t, all_m = allgather_histograms(tup, mult, group)
    return hec.histogram_merge(all_t.contiguous(), all_m.contiguous())


def global_curve_map(q: int, g: int, d: int, with_lambda: bool = False, group=None):
    """Algorithm 1 on all ranks: rank r takes the reduced polynomials with index in shard_range(total, r, world)
    (`hec_curve_map_range`: enumeration, counts, weighted histogram and twists, no collective), then ONE exchange:
    all-gather of the partial maps + `hec_histogram_merge`.  Returns (keys, weights) as numpy arrays on every rank."""
    import numpy as np
    import torch
    import torch.distributed as dist
    from . import hec, workloads as W

    multi = dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1
    if not multi:
        return hec.curve_map(q, g, d, with_lambda)
    rank, world = dist.get_rank(group), dist.get_world_size(group)
    lo, hi = W.shard_range(hec.reduced_total(q, g, d), rank, world)
    keys, w = hec.curve_map(q, g, d, with_lambda, index_range=(lo, hi - lo))
    dev = torch.device("cuda", torch.cuda.current_device())
    t = torch.from_numpy(keys.view(np.int32)).to(dev)
    m = torch.from_numpy(w.view(np.int64)).to(dev)
    all_t, all_m = allgather_histograms(t, m, group)
    mt, mm = hec.histogram_merge(all_t.contiguous(), all_m.contiguous())
    return mt.cpu().numpy().view(np.uint32), mm.cpu().numpy().view(np.uint64)
