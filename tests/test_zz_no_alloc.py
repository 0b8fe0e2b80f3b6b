"""hec_histogram_static: the histogram entry point for callers that cannot allocate device memory.

Who that is: code running inside a process whose GPU memory has already been handed out (a tensor framework's caching
allocator or a serving engine holding nearly all of HBM, so that the ~hundreds of MB hec_histogram's pool may ask
cudaMalloc for are not there or are not ours to take), and code that cannot afford the device-wide synchronisation a
cudaMalloc / cudaFree brings while other streams are busy.  The entry point keeps its hash table and sort buffers in a
fixed 8 MiB array inside the library's device image instead, limited to HEC_HISTOGRAM_STATIC_MAX_ROWS = 2^17 rows.

What is checked: its output equals hec_histogram's (the pooled path), bit for bit -- tuples, order, multiplicities --
on two calls in a row with different inputs.  The second batch is smaller and has other values, so anything the first
call left in the shared array (hash slots, sort buffers, counters) would show up as a wrong result.  The file sorts last
on purpose (pytest -x stops at the first failure), and the test stands alone: it needs no other libhec call before it.
"""
import ctypes

import numpy as np
import pytest
import torch

from paper_1805_11991_b200 import hec


def _batch(seed: int, n: int, g: int, spread: int):
    """Seeded synthetic count rows shaped like hec_count's output: column k scattered around a centre that grows with
    k (as N_k does around q^k + 1), narrow enough that tuples repeat."""
    rng = np.random.default_rng(seed)
    cols = [(10 ** (k + 3) + rng.integers(-spread * (k + 1), spread * (k + 1) + 1, size=n)).astype(np.int64) for k in range(g)]
    counts = np.stack(cols, axis=1).astype(np.uint32)
    mask = (rng.random(n) < 0.9).astype(np.uint8)
    return counts, mask


def _reference(counts_d, mask_d):
    tup, mult = hec.histogram(counts_d, mask_d)           # existing path: pooled scratch, may call cudaMalloc
    return tup.cpu().numpy().view(np.uint32), mult.cpu().numpy().view(np.uint64)


def _static(counts_d, mask_d, out_t, out_m):
    m = hec.histogram_static(counts_d, mask_d, out_t, out_m)
    return out_t[:m].cpu().numpy().view(np.uint32), out_m[:m].cpu().numpy().view(np.uint64)


@pytest.mark.gpu
def test_static_scratch_histogram_matches_pooled_path_twice_in_a_row():
    torch.cuda.set_device(0)
    hec.set_stream(torch.cuda.current_stream().cuda_stream)
    g = 3
    # caller-owned buffers, made once up front: from here on the entry point itself allocates nothing
    cap = hec.HISTOGRAM_STATIC_MAX_ROWS
    out_t = torch.empty((cap, g), dtype=torch.int32, device="cuda")
    out_m = torch.empty((cap,), dtype=torch.int64, device="cuda")
    batches = [_batch(1805, hec.HISTOGRAM_STATIC_MAX_ROWS, g, 40),      # the maximum size: 64 sort tiles, every hash slot range
               _batch(11991, 70001, g, 3)]                              # then a smaller, ragged one with other values
    for counts, mask in batches:
        counts_d = torch.from_numpy(counts.view(np.int32)).cuda()
        mask_d = torch.from_numpy(mask).cuda()
        torch.cuda.synchronize()
        got_t, got_m = _static(counts_d, mask_d, out_t, out_m)
        ref_t, ref_m = _reference(counts_d, mask_d)
        assert got_t.shape == ref_t.shape and (got_t == ref_t).all()    # integer work: bit-exact, same order
        assert (got_m == ref_m).all()
        assert int(got_m.sum()) == int(mask.sum())
        # and without a mask
        got_t, got_m = _static(counts_d, None, out_t, out_m)
        ref_t, ref_m = _reference(counts_d, None)
        assert got_t.shape == ref_t.shape and (got_t == ref_t).all() and (got_m == ref_m).all()
        assert int(got_m.sum()) == counts.shape[0]


@pytest.mark.gpu
def test_static_scratch_histogram_limits_and_errors():
    torch.cuda.set_device(0)
    hec.set_stream(torch.cuda.current_stream().cuda_stream)
    g = 2
    n = hec.HISTOGRAM_STATIC_MAX_ROWS + 1
    counts_d = torch.zeros((n, g), dtype=torch.int32, device="cuda")
    out_t = torch.empty((16, g), dtype=torch.int32, device="cuda")
    out_m = torch.empty((16,), dtype=torch.int64, device="cuda")
    with pytest.raises(hec.HecError) as e:                               # one row too many: refused, the limit is named
        hec.histogram_static(counts_d, None, out_t, out_m)
    assert e.value.code == hec.HEC_ERR_CAPACITY and str(hec.HISTOGRAM_STATIC_MAX_ROWS) in str(e.value)
    # capacity protocol: too small a result buffer reports m and writes nothing
    counts, _ = _batch(7, 5000, g, 6)
    counts_d = torch.from_numpy(counts.view(np.int32)).cuda()
    m = ctypes.c_size_t(0)
    rc = hec.lib().hec_histogram_static(counts_d.data_ptr(), None, 5000, g, out_t.data_ptr(), out_m.data_ptr(), 16, ctypes.byref(m))
    assert rc == hec.HEC_ERR_CAPACITY and m.value == len(np.unique(counts, axis=0))
    # host arrays are refused (staging them would allocate)
    with pytest.raises(hec.HecError) as e:
        mm = ctypes.c_size_t(0)
        hec._check(hec.lib().hec_histogram_static(counts.ctypes.data, None, 5000, g, out_t.data_ptr(), out_m.data_ptr(), 16, ctypes.byref(mm)))
    assert e.value.code == hec.HEC_ERR_INVALID_ARG
    # n = 0 is a no-op
    assert hec.histogram_static(counts_d[:0], None, out_t, out_m) == 0
