"""Multi-GPU plumbing: curves are independent, so `hec_count` shards by contiguous curve
range with NO data-path collective; only the tuple histogram has an exchange step -- an all-gather of the
ranks' sparse (tuple, multiplicity) lists followed by `hec_histogram_merge` on every rank.

One process per GPU, `torch.distributed` for the plumbing (NCCL over NVLink on GPUs; the same code runs on
gloo/CPU tensors in the tests, where the merge -- a CUDA kernel -- is replaced by a stand-in).
Unmeasured on hardware: no multi-GPU box was available to this build.
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
    """All-gather variable-length partial histograms with TWO collectives: the lengths, then one packed buffer.

    tuples: [m][g] int32 tensor, mult: [m] int64 tensor (both on the backend's device; the bits may be unsigned).
    Returns (all_tuples [sum m_r][g], all_mult [sum m_r]) -- the concatenation over ranks in rank order, tuples
    possibly repeated across ranks.  Every rank sends ONE int32 buffer of mmax rows x (g + 2) words (tuple, then the
    two halves of the multiplicity), padded to the longest rank, into one [world * mmax][g + 2] receive buffer.
    """
    import torch
    import torch.distributed as dist

    world = dist.get_world_size(group)
    dev = tuples.device
    g = tuples.shape[1]
    m = torch.tensor([tuples.shape[0]], dtype=torch.int64, device=dev)
    sizes_t = torch.empty((world,), dtype=torch.int64, device=dev)
    dist.all_gather_into_tensor(sizes_t, m, group=group)
    sizes = [int(v) for v in sizes_t.tolist()]
    mmax = max(max(sizes), 1)
    send = torch.zeros((mmax, g + 2), dtype=torch.int32, device=dev)
    if tuples.shape[0]:
        send[: tuples.shape[0], :g] = tuples.to(torch.int32)
        send[: mult.shape[0], g:] = mult.to(torch.int64).contiguous().view(torch.int32).view(-1, 2)
    recv = torch.empty((world * mmax, g + 2), dtype=torch.int32, device=dev)
    dist.all_gather_into_tensor(recv, send, group=group)
    keep = torch.cat([torch.arange(r * mmax, r * mmax + s, device=dev) for r, s in enumerate(sizes)]) if sum(sizes) else \
        torch.empty((0,), dtype=torch.int64, device=dev)
    rows = recv.index_select(0, keep)
    all_t = rows[:, :g].contiguous()
    if rows.shape[0] == 0:
        return all_t, torch.empty((0,), dtype=torch.int64, device=dev)
    all_m = rows[:, g:].contiguous().view(torch.int64).view(-1)
    return all_t, all_m


def _exchange_device():
    """Device the exchange runs on: the current CUDA device (the CPU tests replace this and _merge)."""
    import torch
    return torch.device("cuda", torch.cuda.current_device())


def _to_device(x, dtype):
    """numpy array or tensor -> tensor of `dtype` (same bits) on the exchange device."""
    import numpy as np
    import torch
    if isinstance(x, np.ndarray):
        np_dtype = {torch.int32: np.int32, torch.int64: np.int64}[dtype]
        x = torch.from_numpy(np.ascontiguousarray(x).view(np_dtype))
    return x.to(_exchange_device())


def _merge(all_t, all_m):
    """hec_histogram_merge on the gathered lists.  The collectives ran on torch's current stream: the library is pointed
    at that stream first, so that the merge is ordered after them."""
    import torch
    from . import hec
    hec.set_stream(torch.cuda.current_stream().cuda_stream)
    return hec.histogram_merge(all_t.contiguous(), all_m.contiguous())


def global_histogram(counts, mask, group=None):
    """Per-rank `hec_histogram` + all-gather + `hec_histogram_merge`: every rank returns the histogram of
    the union of all ranks' rows.  With one rank this is just `hec_histogram`.  Host (numpy) inputs give host outputs
    with one rank and device tensors otherwise (the exchange runs on the device)."""
    import torch.distributed as dist
    from . import hec

    tup, mult = hec.histogram(counts, mask)
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return tup, mult
    import torch
    all_t, all_m = allgather_histograms(_to_device(tup, torch.int32), _to_device(mult, torch.int64), group)
    return _merge(all_t, all_m)


def global_curve_map(q: int, g: int, d: int, with_lambda: bool = False, group=None):
    """Algorithm 1 on all ranks: rank r takes the reduced polynomials with index in shard_range(total, r, world)
    (`hec_curve_map_range`: enumeration, counts, weighted histogram and twists, no collective), then ONE exchange:
    all-gather of the partial maps + `hec_histogram_merge`, all on the device.  Returns (keys, weights) as numpy arrays
    on every rank."""
    import numpy as np
    import torch
    import torch.distributed as dist
    from . import hec, workloads as W

    multi = dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1
    if not multi:
        return hec.curve_map(q, g, d, with_lambda)
    rank, world = dist.get_rank(group), dist.get_world_size(group)
    lo, hi = W.shard_range(hec.reduced_total(q, g, d), rank, world)
    keys, w = hec.curve_map(q, g, d, with_lambda, index_range=(lo, hi - lo), device=True)
    all_t, all_m = allgather_histograms(_to_device(keys, torch.int32), _to_device(w, torch.int64), group)
    mt, mm = _merge(all_t, all_m)
    return mt.cpu().numpy().view(np.uint32), mm.cpu().numpy().view(np.uint64)
