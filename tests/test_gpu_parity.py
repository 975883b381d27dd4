"""Parity of the CUDA path (through the C ABI) with the oracle, element by element, on seeded synthetic inputs.

Bar (BASELINE.json north_star): bit-exact delay tables, decimated series, int32 DM transform and integer statistics;
|dSNR| <= 1e-3; identical candidate lists except for events within 1e-3 of the threshold.
"""
import numpy as np
import pytest

from helpers import (check_candidates_against_oracle, check_dmt_against_oracle, check_plan_against_oracle,
                     check_stats_against_oracle, make_plan)

pytestmark = pytest.mark.gpu

TSAMP = 1.31072e-3


class Shape:
    """A free-form workload (same attribute names as synth.Workload) for the odd-shape cases."""

    def __init__(self, fch1, foff, nchan, nsamp, ranges, widths, threshold, nbeam=1, tsamp=TSAMP):
        self.fch1, self.foff, self.nchan, self.nsamp, self.ranges = fch1, foff, nchan, nsamp, ranges
        self.widths, self.threshold, self.nbeam, self.tsamp = widths, threshold, nbeam, tsamp


def run_gpu(cuda, api, w, fb_host, options=None, search=True, cand_capacity=1 << 22):
    """fb_host: uint8 [nbeam][nchan][nsamp].  Returns (plan, dmt host array [nbeam][elems], candidates or None)."""
    plan = make_plan(api, w, nbeam=fb_host.shape[0], cand_capacity=cand_capacity, options=options)
    d_fb = cuda.from_numpy(fb_host).cuda()
    d_dmt = cuda.full((fb_host.shape[0], plan.dmt_elems_per_beam), -7, dtype=cuda.int32, device="cuda")
    plan.dedisperse(d_fb, d_dmt)
    cands = None
    if search:
        plan.single_pulse_search(d_dmt, w.threshold)
        total, ovf = plan.candidates_count()
        assert not ovf, f"candidate list overflowed ({total})"
        cands = plan.candidates_read()
        assert cands.size == total
    cuda.cuda.synchronize()
    return plan, d_dmt.cpu().numpy(), cands


def oracle_path(orc, w, fb, search=True):
    return orc.run_path(fb, w.fch1, w.foff, w.tsamp, w.ranges, w.widths, w.threshold, do_search=search)


# ---- config 1 (Tiny), every kernel variant --------------------------------------------------------------------
@pytest.mark.parametrize("options", [
    {"dedisp_kernel": 1},
    {"group": 1}, {"group": 2}, {"group": 4}, {"group": 8}, {"group": 4, "dm_tile": 32}, {"group": 8, "dm_tile": 32},
    {"group": 8, "skew": 0}, {"group": 12, "max_entries": 12}, {"group": 16, "max_entries": 12}, {"group": 16, "max_entries": 16},
    {"tile_words": 224}, {"tile_words": 224, "max_entries": 12}, {"tile_words": 224, "max_entries": 16, "skew": 0},
])
def test_cfg1_dm_transform_bit_exact(cuda, api, orc, synth, options):
    w = synth.workload(1)
    fb = synth.generate(w)
    ref = oracle_path(orc, w, fb, search=False)
    plan, dmt, _ = run_gpu(cuda, api, w, fb[None], options=options, search=False)
    check_plan_against_oracle(orc, plan, w)
    check_dmt_against_oracle(plan, dmt, ref)
    # row padding is never written
    _, _, _, nout, off = plan.trial_table()
    for d in range(plan.ntrials - 1):
        assert np.all(dmt[0][off[d] + nout[d]: off[d + 1]] == -7)


def test_cfg1_search_and_recovery(cuda, api, orc, synth):
    w = synth.workload(1)
    fb = synth.generate(w)
    ref = oracle_path(orc, w, fb)
    plan, dmt, cands = run_gpu(cuda, api, w, fb[None])
    check_dmt_against_oracle(plan, dmt, ref)
    check_stats_against_oracle(plan, ref)
    st = check_candidates_against_oracle(orc, plan, cands, ref, w.widths, w.threshold)
    assert st["oracle"] > 0 and st["matched"] >= st["oracle"] - st["near_threshold_only_oracle"]
    # the injected burst (DM 50 = trial 50, t 1000, width 4, S/N 24) is the top candidate of the CUDA path too
    top = cands[np.argmax(cands["snr"])]
    assert abs(int(top["trial"]) - 50) <= 1 and abs(int(top["t"]) - 1000) <= 2 and top["width"] in (2, 4, 8)
    assert abs(float(top["snr"]) - 24.0) <= 3.0
    n, s, q = plan.trial_stats(0, 50)
    assert (n, s, q) == (int(ref[0].nout[50]), int(ref[0].search.sum[50]), int(ref[0].search.sumsq[50]))


# ---- several ranges with decimation, several tiles and a ragged tail ---------------------------------------------
def mini3(synth, seed, nsamp=65536, nchan=1024):
    """Config-3-like: three ranges (decimation 1, 2, 4), one dispersed burst inside each, a zero-DM spike."""
    import math
    w = synth.Workload("mini3", 0, 1, nchan, nsamp, 500.0, -200.0 / nchan, TSAMP, 128.0, 10.0,
                       [(0.0, 0.2, 150, 1), (480.0, 0.5, 70, 2), (1900.0, 1.0, 101, 4)],
                       [1, 2, 4, 8, 16, 32, 64, 128, 256, 512], 6.0, seed)
    amp = lambda snr, wid: snr * w.std / math.sqrt(nchan * wid)
    w.bursts = [[synth.Burst(dm=15.1, t0=20000, width=4, snr=30.0, amp=amp(30.0, 4)),
                 synth.Burst(dm=497.3, t0=9000, width=8, snr=40.0, amp=amp(40.0, 8)),
                 synth.Burst(dm=1950.0, t0=3000, width=16, snr=50.0, amp=amp(50.0, 16))]]
    w.spikes = [(30000, 3, 4.0)]
    return w


@pytest.mark.parametrize("options", [{"group": 4}, {"group": 8}, {"group": 2, "dm_tile": 32}, {"dedisp_kernel": 1},
                                     {"group": 8, "skew": 0}, {"group": 16, "max_entries": 12},
                                     {"group": 16, "max_entries": 16}, {"compact": 0}, {"compact": 0, "max_entries": 12},
                                     {"tile_words": 224, "max_entries": 12}, {"tile_words": 224, "compact": 0}])
def test_multirange_decimated_bit_exact(cuda, api, orc, synth, options):
    w = mini3(synth, 11)
    fb = synth.generate(w)
    ref = oracle_path(orc, w, fb, search=False)
    plan, dmt, _ = run_gpu(cuda, api, w, fb[None], options=options, search=False)
    check_plan_against_oracle(orc, plan, w, stride=7)
    check_dmt_against_oracle(plan, dmt, ref)
    for ri, rr in enumerate(ref):                      # decimated series, bit-exact
        got = plan.decimated_read(ri)
        if rr.decim == 1:
            assert got is None
        else:
            assert got.dtype == np.uint16 and np.array_equal(got, rr.series)


def test_multirange_search(cuda, api, orc, synth):
    w = mini3(synth, 12)
    fb = synth.generate(w)
    ref = oracle_path(orc, w, fb)
    per_range = [int(r.search.candoff[-1]) for r in ref]
    assert all(n > 0 for n in per_range), per_range     # every range (decimation 1, 2, 4) has detections
    plan, dmt, cands = run_gpu(cuda, api, w, fb[None], cand_capacity=sum(per_range) + 4096)
    check_dmt_against_oracle(plan, dmt, ref)
    check_stats_against_oracle(plan, ref)
    st = check_candidates_against_oracle(orc, plan, cands, ref, w.widths, w.threshold)
    assert st["oracle"] > 1000, st            # the append path is exercised
    assert st["near_threshold_only_oracle"] + st["near_threshold_only_gpu"] <= max(5, st["oracle"] // 1000)


# ---- odd shapes and degenerate inputs -------------------------------------------------------------------------
@pytest.mark.parametrize("fill", ["uniform", "all255", "zero"])
@pytest.mark.parametrize("options", [{"group": 4}, {"group": 8}, {"dedisp_kernel": 1}, {"group": 16, "max_entries": 12},
                                     {"group": 16, "max_entries": 16}, {"tile_words": 224}, {"tile_words": 224, "max_entries": 12}])
def test_odd_shapes(cuda, api, orc, fill, options):
    # 71 channels (not a multiple of any group size), 5003 samples (rows not 16-byte multiples), trial counts that
    # are not multiples of the DM tile, decimation 8, a range whose last trials have no valid output at all
    w = Shape(420.0, -1.0, 71, 5003, [(3.0, 0.7, 77, 1), (60.0, 1.1, 41, 2), (100.0, 2.0, 5, 8), (600.0, 150.0, 4, 1)],
              [1, 3, 7, 20], 5.0)
    rs = np.random.default_rng(5)
    if fill == "uniform":
        fb = rs.integers(0, 256, size=(w.nchan, w.nsamp), dtype=np.uint8)
    elif fill == "all255":
        fb = np.full((w.nchan, w.nsamp), 255, dtype=np.uint8)      # every 16-bit lane at its maximum
    else:
        fb = np.zeros((w.nchan, w.nsamp), dtype=np.uint8)          # sigma == 0: no candidates
    ref = oracle_path(orc, w, fb)
    plan, dmt, cands = run_gpu(cuda, api, w, fb[None], options=options)
    check_plan_against_oracle(orc, plan, w)
    _, _, _, nout, _ = plan.trial_table()
    assert (nout == 0).any() and (nout > 0).any()
    check_dmt_against_oracle(plan, dmt, ref)
    check_stats_against_oracle(plan, ref)
    st = check_candidates_against_oracle(orc, plan, cands, ref, w.widths, w.threshold)
    if fill != "uniform":
        assert st["gpu"] == 0 and st["oracle"] == 0
    for ri, rr in enumerate(ref):
        if rr.decim > 1:
            assert np.array_equal(plan.decimated_read(ri), rr.series)


def test_rows_that_are_not_16_sample_multiples_keep_the_8bit_copy(cuda, api, orc):
    """5003 samples: the input rows, and the decimated rows (2501 and 625 samples), all end in padding.  The padding must
    not count in the bounds of a series: with Gaussian bytes the decimated ranges still take their 8-bit copy (floor > 0).
    Run on a non-blocking stream: the padded input copy and its one-time zero fill are ordered on the caller's stream."""
    w = Shape(420.0, -1.0, 71, 5003, [(3.0, 0.7, 77, 1), (60.0, 1.1, 41, 2), (100.0, 2.0, 5, 8)], [1, 3, 7, 20], 4.5)
    rs = np.random.default_rng(6)
    fb = rs.normal(128, 10, size=(w.nchan, w.nsamp)).round().clip(0, 255).astype(np.uint8)
    ref = oracle_path(orc, w, fb)
    with cuda.cuda.stream(cuda.cuda.Stream()):
        plan, dmt, cands = run_gpu(cuda, api, w, fb[None])
        for ri, rr in enumerate(ref):
            if rr.decim > 1:
                assert rr.series.shape[1] % 16 != 0
                in_use, floor, span = plan.decimated_compact(ri)
                assert in_use and floor == int(rr.series.min()) and span == int(rr.series.max()) - floor, (ri, in_use, floor, span)
                assert np.array_equal(plan.decimated_read(ri), rr.series)
            else:
                assert plan.decimated_compact(ri) == (False, 0, 0)
    check_dmt_against_oracle(plan, dmt, ref)
    check_stats_against_oracle(plan, ref)
    st = check_candidates_against_oracle(orc, plan, cands, ref, w.widths, w.threshold)
    assert st["oracle"] > 0


def test_all255_wide_band_lane_limits(cuda, api, orc):
    """4096 channels of 255 at decimation 4: int32 outputs reach 4096*255*4 and every packed lane flush is needed."""
    w = Shape(500.0, -0.048828125, 4096, 4096, [(0.0, 0.2, 70, 1), (0.0, 1.0, 70, 4)], [1, 2, 1024], 6.0)
    fb = np.full((w.nchan, w.nsamp), 255, dtype=np.uint8)
    ref = oracle_path(orc, w, fb, search=False)
    plan, dmt, _ = run_gpu(cuda, api, w, fb[None], search=False)
    check_dmt_against_oracle(plan, dmt, ref)
    assert dmt.max() == 4096 * 255 * 4


def test_square_wave_takes_the_exact_search_path(cuda, api, orc):
    """Rows whose samples sit 2e6 counts from their mean with a 1024-wide boxcar: boxcar sums of x - mean do not fit
    the fast path's int32 test (wmax * max|x - m| >= 2^30), so the search kernel must take its exact path."""
    w = Shape(500.0, -0.048828125, 4096, 8192, [(0.0, 0.2, 12, 1), (0.0, 1.0, 12, 4)], [1, 4, 64, 1024], 1.5)
    t = np.arange(w.nsamp)
    fb = np.where((t // 96) % 2 == 0, 255, 0).astype(np.uint8)[None, :].repeat(w.nchan, axis=0)
    fb[::7, 5000:5003] = 17
    ref = oracle_path(orc, w, fb)
    ncand = sum(int(r.search.candoff[-1]) for r in ref)
    assert ncand > 1000
    plan, dmt, cands = run_gpu(cuda, api, w, fb[None], cand_capacity=ncand + 4096)
    check_dmt_against_oracle(plan, dmt, ref)
    check_stats_against_oracle(plan, ref)
    st = check_candidates_against_oracle(orc, plan, cands, ref, w.widths, w.threshold)
    assert st["matched"] >= st["oracle"] - st["near_threshold_only_oracle"]
    _, _, _, nout, off = plan.trial_table()
    row = dmt[0][off[12]: off[12] + nout[12]]                   # the DM 0 row at decimation 4: samples 0 or 4*4096*255
    assert int(row.max()) - int(row.min()) > (1 << 21)          # the premise: 1024 * max|x - m| >= 2^30


@pytest.mark.parametrize("lo,hi", [(200, 203), (0, 3), (250, 255), (17, 17)])
def test_narrow_value_ranges_bit_exact(cuda, api, orc, lo, hi):
    """The packed lanes sum (sample - smallest sample of the launch) and may then go floor(65535 / (largest - smallest))
    channels without widening: data confined to a narrow band of values far from zero, at both ends of the uint8 range,
    constant data, decimated ranges, and tiles whose skewed windows start before the rows."""
    w = Shape(500.0, -0.048828125, 4096, 6000, [(0.0, 0.2, 70, 1), (300.0, 0.5, 70, 2), (900.0, 1.0, 40, 4)], [1, 2, 8], 6.0)
    rs = np.random.default_rng(lo)
    fb = rs.integers(lo, hi + 1, size=(w.nchan, w.nsamp), dtype=np.uint8)
    ref = oracle_path(orc, w, fb, search=False)
    for options in ({}, {"skew": 0}):
        plan, dmt, _ = run_gpu(cuda, api, w, fb[None], options=options, search=False)
        check_dmt_against_oracle(plan, dmt, ref)


# ---- config 2 at reduced length -----------------------------------------------------------------------------------
def test_cfg2_reduced(cuda, api, orc, synth):
    w = synth.workload(2, nsamp=16384)
    fb = synth.generate(w)
    ref = oracle_path(orc, w, fb)
    plan, dmt, cands = run_gpu(cuda, api, w, fb[None])
    check_plan_against_oracle(orc, plan, w, stride=41)
    check_dmt_against_oracle(plan, dmt, ref)
    check_stats_against_oracle(plan, ref)
    check_candidates_against_oracle(orc, plan, cands, ref, w.widths, w.threshold)


# ---- multibeam batch (config 4 shape, reduced) -----------------------------------------------------------------------
def test_multibeam_batch(cuda, api, orc, synth):
    w = synth.workload(4, nsamp=1 << 14, nbeam=3)
    w.ranges = [(0.0, 0.2, 130, 1), (500.0, 0.5, 66, 2), (1000.0, 1.0, 40, 4)]
    w.threshold = 6.0
    fb = np.stack([synth.generate(w, beam=b) for b in range(w.nbeam)])
    fb[1, :, 5000:5004] += 30
    plan, dmt, cands = run_gpu(cuda, api, w, fb)
    assert set(np.unique(cands["beam"])) <= {0, 1, 2}
    for b in range(w.nbeam):
        ref = oracle_path(orc, w, fb[b])
        check_dmt_against_oracle(plan, dmt, ref, beam=b)
        check_stats_against_oracle(plan, ref, beam=b, nbeam=w.nbeam)
        check_candidates_against_oracle(orc, plan, cands, ref, w.widths, w.threshold, beam=b)


# ---- the host-buffer entry point ---------------------------------------------------------------------------------------
def test_search_host_matches_device_path(cuda, api, orc, synth):
    w = synth.workload(1)
    fb = synth.generate(w)
    ref = oracle_path(orc, w, fb)
    plan = make_plan(api, w)
    h_dmt = np.full((1, plan.dmt_elems_per_beam), -7, dtype=np.int32)
    ncand, ovf = plan.search_host(fb[None], w.threshold, h_dmt)
    assert not ovf
    check_dmt_against_oracle(plan, h_dmt, ref)
    cands = plan.candidates_read()
    assert cands.size == ncand
    check_candidates_against_oracle(orc, plan, cands, ref, w.widths, w.threshold)
    assert plan.launches() >= 2


# ---- spt_search inside a CUDA graph: the call only enqueues (memsets, kernels, event fork/join of its side streams), so a
# caller can capture it once and replay it -- what a launch-bound small plan wants ------------------------------------
def test_search_can_be_captured_in_a_cuda_graph(cuda, api, orc, synth):
    w = mini3(synth, 12)
    fbs = [synth.generate(w, beam=b) for b in range(2)]           # two different inputs through the same graph
    plan = make_plan(api, w, cand_capacity=1 << 20)
    d_fb = cuda.from_numpy(fbs[0][None]).cuda()
    d_dmt = cuda.zeros((1, plan.dmt_elems_per_beam), dtype=cuda.int32, device="cuda")
    plan.search(d_fb, w.threshold, d_dmt)                          # first call outside the capture: it allocates and uploads
    cuda.cuda.synchronize()
    side = cuda.cuda.Stream()
    graph = cuda.cuda.CUDAGraph()
    with cuda.cuda.graph(graph, stream=side):
        plan.search(d_fb, w.threshold, d_dmt, side)
    for fb in fbs[::-1] + fbs:
        d_fb.copy_(cuda.from_numpy(fb[None]))
        d_dmt.fill_(-3)
        graph.replay()
        total, ovf = plan.candidates_count()
        cands = plan.candidates_read()
        assert not ovf and cands.size == total
        ref = oracle_path(orc, w, fb)
        check_dmt_against_oracle(plan, d_dmt.cpu().numpy(), ref)
        check_stats_against_oracle(plan, ref)
        st = check_candidates_against_oracle(orc, plan, cands, ref, w.widths, w.threshold)
        assert st["oracle"] > 100, st


# ---- spt_search: both steps in one call, every range searched behind its own dedispersion --------------------------
@pytest.mark.parametrize("profile", [0, 1])
def test_fused_search_call_matches_oracle_and_two_call_path(cuda, api, orc, synth, profile):
    w = mini3(synth, 12)
    w.nbeam = 2
    fb = np.stack([synth.generate(w, beam=b) for b in range(2)])
    plan = make_plan(api, w, nbeam=2, options={"profile": profile})
    d_fb = cuda.from_numpy(fb).cuda()
    d_dmt = cuda.full((2, plan.dmt_elems_per_beam), -7, dtype=cuda.int32, device="cuda")
    for _ in range(2):                                   # twice: the second pass reuses side streams and events
        plan.search(d_fb, w.threshold, d_dmt)
    total, ovf = plan.candidates_count()
    assert not ovf
    cands = plan.candidates_read()
    assert cands.size == total
    dmt = d_dmt.cpu().numpy()
    for b in range(2):
        ref = oracle_path(orc, w, fb[b])
        check_dmt_against_oracle(plan, dmt, ref, beam=b)
        check_stats_against_oracle(plan, ref, beam=b, nbeam=2)
        st = check_candidates_against_oracle(orc, plan, cands, ref, w.widths, w.threshold, beam=b)
        assert st["oracle"] > 100, st
    # the two separate calls give the same list (up to its order)
    plan.dedisperse(d_fb, d_dmt)
    plan.single_pulse_search(d_dmt, w.threshold)
    two = plan.candidates_read()
    key = lambda c: np.lexsort((c["t"], c["trial"], c["beam"]))
    a, b2 = cands[key(cands)], two[key(two)]
    assert a.size == b2.size
    for f in ("beam", "trial", "t", "width", "snr"):
        assert np.array_equal(a[f], b2[f]), f


def test_search_host_multirange(cuda, api, orc, synth):
    w = mini3(synth, 13)
    fb = synth.generate(w)
    ref = oracle_path(orc, w, fb)
    plan = make_plan(api, w)
    h_dmt = np.full((1, plan.dmt_elems_per_beam), -7, dtype=np.int32)
    ncand, ovf = plan.search_host(fb[None], w.threshold, h_dmt)
    assert not ovf
    check_dmt_against_oracle(plan, h_dmt, ref)
    check_stats_against_oracle(plan, ref)
    cands = plan.candidates_read()
    assert cands.size == ncand
    check_candidates_against_oracle(orc, plan, cands, ref, w.widths, w.threshold)


def test_stream_pipeline_matches_search_host(cuda, api, synth):
    """Two batches in flight (H2D of one overlapping the kernels of the other): every pop gives what the synchronous call
    gives for that batch, and the read-out calls follow the popped batch."""
    w = synth.workload(4, nsamp=1 << 13, nbeam=2)
    w.ranges = [(0.0, 0.2, 70, 1), (500.0, 0.5, 40, 2)]
    w.threshold = 5.0
    batches = []
    for i in range(4):
        fb = np.stack([synth.generate(w, beam=2 * i + b) for b in range(2)])
        fb[0, :, 3000 + 100 * i: 3004 + 100 * i] += 25             # a different zero-DM spike per batch
        batches.append(cuda.from_numpy(fb).pin_memory())
    ref_plan = make_plan(api, w, nbeam=2)
    expect = []
    for hb in batches:
        n, ovf = ref_plan.search_host(hb, w.threshold)
        c = ref_plan.candidates_read()
        s, q = ref_plan.trial_stats_all(2)
        expect.append((n, np.sort(c, order=["beam", "trial", "t"]), s.copy(), q.copy()))
    assert len({e[0] for e in expect}) > 1 and all(e[0] > 0 for e in expect)
    plan = make_plan(api, w, nbeam=2)
    with pytest.raises(api.SptError) as e:
        plan.stream_pop()                                            # nothing in flight
    assert e.value.code == api.SPT_ERR_STATE
    plan.stream_push(batches[0], w.threshold)
    plan.stream_push(batches[1], w.threshold)
    with pytest.raises(api.SptError) as e:
        plan.stream_push(batches[2], w.threshold)                    # a third batch must wait for a pop
    assert e.value.code == api.SPT_ERR_STATE
    for i in range(4):
        n, ovf = plan.stream_pop()                                   # batch i + 1 is still in flight
        assert (n, ovf) == (expect[i][0], False)
        c = np.sort(plan.candidates_read(), order=["beam", "trial", "t"])
        assert np.array_equal(c, expect[i][1])
        s, q = plan.trial_stats_all(2)
        assert np.array_equal(s, expect[i][2]) and np.array_equal(q, expect[i][3])
        if i + 2 < 4:
            plan.stream_push(batches[i + 2], w.threshold)            # reuses the buffers of the batch just read out


def test_plan_with_no_valid_output_at_all(cuda, api):
    """Every sweep longer than the data: nothing to compute, nothing found, no error."""
    w = Shape(500.0, -400.0 / 17, 17, 2314, [(32.6, 0.05, 93, 8), (37.3, 1.0, 88, 8)], [1, 3, 100], 5.0)
    plan = api.Plan(w.fch1, w.foff, w.nchan, w.tsamp, w.nsamp, w.ranges, w.widths)
    assert plan.dmt_elems_per_beam == 0
    fb = cuda.zeros((1, w.nchan, w.nsamp), dtype=cuda.uint8, device="cuda")
    d_dmt = plan.dedisperse(fb)
    plan.single_pulse_search(d_dmt, w.threshold)
    assert plan.candidates_count() == (0, False)


def test_wide_delay_spread_is_refused_not_miscomputed(cuda, api, orc):
    """DM steps of 3 pc cm^-3 over a band that reaches down to 100 MHz: the 64-trial tile does not fit shared memory ->
    UNSUPPORTED; the cross-check kernel takes the same plan."""
    w = Shape(500.0, -400.0 / 1024, 1024, 17003, [(4.4, 0.5, 125, 1), (66.9, 3.0, 139, 1)], [2, 100], 5.0)
    fb = np.random.default_rng(0).integers(0, 256, size=(1, w.nchan, w.nsamp), dtype=np.uint8)
    with pytest.raises(api.SptError) as e:
        run_gpu(cuda, api, w, fb, search=False)
    assert e.value.code == api.SPT_ERR_UNSUPPORTED
    plan, dmt, _ = run_gpu(cuda, api, w, fb, options={"dedisp_kernel": 1}, search=False)
    check_dmt_against_oracle(plan, dmt, oracle_path(orc, w, fb[0], search=False))


def test_candidate_overflow_is_reported(cuda, api, synth):
    w = synth.workload(1)
    fb = synth.generate(w)
    plan = make_plan(api, w, cand_capacity=3)
    ncand, ovf = plan.search_host(fb[None], 2.0)
    assert ovf and ncand > 3
    assert plan.candidates_read().size == 3


# ---- the degenerate corners of the plan space ------------------------------------------------------------------
@pytest.mark.parametrize("case", [
    dict(nchan=1, nsamp=64, ranges=[(0.0, 1.0, 1, 1)], widths=[1, 2], thr=-1e9),            # one channel, one trial: out = in
    dict(nchan=3, nsamp=16, ranges=[(0.0, 5.0, 2, 1)], widths=[1, 64], thr=0.5),             # a width longer than the rows
    dict(nchan=5, nsamp=200, ranges=[(0.0, 1.0, 3, 64)], widths=[1, 2], thr=-1e9),           # decimation 64: rows of 3 samples
    dict(nchan=64, nsamp=515, ranges=[(0.0, 0.5, 130, 1), (65.0, 1.0, 2, 2)], widths=[1, 3, 9], thr=-1e9),   # every start a candidate
    dict(nchan=4096, nsamp=600, ranges=[(0.0, 0.05, 65, 1)], widths=[1], thr=3.0),           # rows shorter than two tiles, 65 trials
])
def test_degenerate_plans(cuda, api, orc, case):
    nchan = case["nchan"]
    w = Shape(500.0, -200.0 / nchan, nchan, case["nsamp"], case["ranges"], case["widths"], case["thr"])
    rs = np.random.default_rng(nchan + case["nsamp"])
    fb = rs.integers(0, 256, size=(nchan, w.nsamp), dtype=np.uint8)
    ref = oracle_path(orc, w, fb)
    plan, dmt, cands = run_gpu(cuda, api, w, fb[None])
    check_plan_against_oracle(orc, plan, w)
    check_dmt_against_oracle(plan, dmt, ref)
    check_stats_against_oracle(plan, ref)
    st = check_candidates_against_oracle(orc, plan, cands, ref, w.widths, w.threshold)
    if case["thr"] < -1e8:                      # every start position of every row with a non-zero variance is a candidate, once
        assert st["gpu"] == st["oracle"] == st["matched"] > 0
    if nchan == 1:
        assert np.array_equal(dmt[0][: w.nsamp], fb[0].astype(np.int32))
