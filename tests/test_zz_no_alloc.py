"""spt_peak_filter_static: the peak filter for callers that cannot allocate device memory -- a real-time
loop that must not take the device-wide stall of a cudaMalloc / cudaFree, or a process whose device memory another
allocator already owns.  Its working memory is a fixed block inside libspt.so instead of buffers grown on demand.

What is checked: on the same candidate list it keeps exactly the records spt_peak_filter keeps (the two run the same
kernels, so the survivor sets must be identical, as test_gpu_peaks.py asks of the existing path), on two calls in a row
with different lists -- the second call finds the first one's hash table and flags in the shared block and must not be
misled by them -- and a list beyond the fixed limit is refused with a message instead of being filtered wrongly.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here should not hide the
parity tests.  It does not depend on what ran before it (own plan, own buffers; the shared block is cleared per call)."""
import numpy as np
import pytest

from test_gpu_parity import mini3, run_gpu

pytestmark = pytest.mark.gpu


def as_set(c):
    return {(int(r["beam"]), int(r["trial"]), int(r["t"]), int(r["width"]), float(r["snr"])) for r in c}


def static_filter(cuda, api, plan, cands, windows):
    """The call a no-allocation user makes; the tensors here stand for buffers such a caller set aside at start-up."""
    n = int(cands.size)
    d_cand = cuda.from_numpy(np.ascontiguousarray(cands).view(np.uint8).copy()).cuda()
    d_peaks = cuda.zeros(max(n, 1) * api.CAND_DTYPE.itemsize, dtype=cuda.uint8, device="cuda")
    d_count = cuda.full((1,), -1, dtype=cuda.int64, device="cuda")
    plan.peak_filter_static(d_cand, n, windows, d_peaks, d_count)
    cuda.cuda.synchronize()
    k = int(d_count.item())
    assert 0 <= k <= n
    return d_peaks.cpu().numpy().view(api.CAND_DTYPE)[:k]


def test_static_filter_matches_the_allocating_filter_twice_in_a_row(cuda, api, synth):
    w = mini3(synth, 12)
    fb = synth.generate(w)
    plan, dmt, cands = run_gpu(cuda, api, w, fb[None], cand_capacity=1 << 20)
    assert 1000 < cands.size <= api.PEAKS_STATIC_MAX
    windows = (3, 11)
    plan.set_option("peaks_lookup", 1)                       # the existing path through its own (allocated) hash table
    expect = plan.peak_filter(windows)
    assert 0 < expect.size < cands.size

    got1 = static_filter(cuda, api, plan, cands, windows)    # first call: also the one-time address look-up
    assert as_set(got1) == as_set(expect)

    # second call, at once, with other windows; then a different, shorter list (the survivors of the first call: a
    # sparser plane hashed into slots that still hold the longer list's keys)
    got2 = static_filter(cuda, api, plan, cands, (5, 3, 7))
    assert as_set(got2) == as_set(plan.peak_filter((5, 3, 7)))
    got3 = static_filter(cuda, api, plan, got1, (11,))
    # filtering survivors again with the larger of the two windows removes nothing: every survivor already won its 11x11
    assert as_set(got3) == as_set(got1)
    got4 = static_filter(cuda, api, plan, cands, windows)    # and the first list again after a shorter one
    assert as_set(got4) == as_set(expect)

    assert as_set(plan.candidates_read()) == as_set(cands)   # the plan's own lists are left alone
    assert as_set(plan.peak_filter(windows)) == as_set(expect)


def test_static_filter_empty_list_and_limit(cuda, api, synth):
    w = synth.workload(1)
    fb = synth.generate(w)
    plan, dmt, cands = run_gpu(cuda, api, w, fb[None])
    got = static_filter(cuda, api, plan, cands[:0], (3,))
    assert got.size == 0
    n = api.PEAKS_STATIC_MAX + 1
    d_big = cuda.zeros(n * api.CAND_DTYPE.itemsize, dtype=cuda.uint8, device="cuda")
    d_count = cuda.full((1,), -1, dtype=cuda.int64, device="cuda")
    with pytest.raises(api.SptError) as e:
        plan.peak_filter_static(d_big, n, (3,), d_big, d_count)
    assert e.value.code == api.SPT_ERR_UNSUPPORTED and str(api.PEAKS_STATIC_MAX) in str(e.value)
    cuda.cuda.synchronize()
    assert int(d_count.item()) == -1                         # refused: nothing was enqueued
    fresh = api.Plan(w.fch1, w.foff, w.nchan, w.tsamp, w.nsamp, w.ranges, w.widths, max_beams=1, cand_capacity=1024)
    with pytest.raises(api.SptError) as e:                   # a plan that never ran has no device tables, and none are made here
        fresh.peak_filter_static(d_big, 1, (3,), d_big, d_count)
    assert e.value.code == api.SPT_ERR_STATE
    fresh.close()
