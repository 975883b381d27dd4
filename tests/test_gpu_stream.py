"""NEXT-2 (reading F): corner turn of time-major blocks and overlap-save segments.  The DM transform after
every push must be, bit for bit, the oracle's batch dedispersion of the last nsamp samples of the stream, so that the
last nnew/decim outputs of every trial continue the previous push's."""
import numpy as np
import pytest

from helpers import check_dmt_against_oracle, check_segment_against_oracle, make_plan
from test_gpu_parity import Shape, oracle_path

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("shape,flip", [((1, 1000, 71), False), ((2, 513, 256), True), ((1, 64, 4096), True), ((3, 7, 5), False)])
def test_corner_turn(cuda, api, orc, shape, flip):
    rs = np.random.default_rng(sum(shape))
    x = rs.integers(0, 256, size=shape, dtype=np.uint8)
    got = api.corner_turn(cuda.from_numpy(x).cuda(), flip).cpu().numpy()
    for b in range(shape[0]):
        assert np.array_equal(got[b], orc.corner_turn(x[b], flip))


@pytest.mark.parametrize("shape,flip", [((1000, 3, 71), True), ((64, 2, 4096), False), ((7, 5, 5), False)])
def test_corner_turn_time_spliced(cuda, api, orc, shape, flip):
    """The rings' layout: [t][beam][chan], the beams of a host interleaved sample by sample."""
    rs = np.random.default_rng(sum(shape) + 1)
    x = rs.integers(0, 256, size=shape, dtype=np.uint8)
    got = api.corner_turn(cuda.from_numpy(x).cuda(), flip, spliced=True).cpu().numpy()
    for b, exp in enumerate(orc.corner_turn_spliced(x, flip)):
        assert np.array_equal(got[b], exp)


def test_incremental_push_computes_only_the_new_tail(cuda, api, orc):
    """whole_rows = 0 with time-spliced input: after every push the last nnew/k + wmax - 1 outputs of every row equal the
    oracle's dedispersion of the stream buffer, and nothing else in the DM transform buffer is touched."""
    nchan, nnew, nbeam = 256, 2048, 2
    widths = [1, 2, 4, 16]
    w = Shape(500.0, -200.0 / nchan, nchan, 0, [(0.0, 0.2, 70, 1), (10.0, 0.5, 40, 2), (30.0, 1.0, 33, 4)], widths, 6.0, nbeam=nbeam)
    probe = api.Plan(w.fch1, w.foff, nchan, w.tsamp, 1 << 16, w.ranges, w.widths)
    _, hsearch, _ = probe.segment_info()
    w.nsamp = hsearch + nnew + 1024                                 # rows longer than the tail: there is something to leave alone
    rs = np.random.default_rng(10)
    blocks = [rs.integers(0, 256, size=(nnew, nbeam, nchan), dtype=np.uint8) for _ in range(3)]   # [t][beam][chan]
    plan = make_plan(api, w, nbeam=nbeam)
    refs = [orc.overlap_save_buffers([blk[:, b, :] for blk in blocks], w.nsamp, flip=True) for b in range(nbeam)]
    _, _, dec, nout, off = plan.trial_table()
    SENT = -123456789
    for i, blk in enumerate(blocks):
        d_dmt = cuda.full((nbeam, plan.dmt_elems_per_beam), SENT, dtype=cuda.int32, device="cuda")
        plan.segment_push(cuda.from_numpy(blk).cuda(), flip=True, d_dmt=d_dmt, spliced=True, whole_rows=False)
        dmt = d_dmt.cpu().numpy()
        untouched = 0
        for b in range(nbeam):
            ref = oracle_path(orc, w, refs[b][i], search=False)
            d = 0
            for rr in ref:
                for j in range(len(rr.nout)):
                    n, k = int(nout[d]), int(dec[d])
                    tail = min(n, nnew // k + max(widths) - 1)
                    got = dmt[b][off[d]: off[d] + n]
                    exp = rr.dmt[rr.rowoff[j]: rr.rowoff[j + 1]]
                    assert np.array_equal(got[n - tail:], exp[n - tail:]), (i, b, d)
                    assert np.all(got[: n - tail] == SENT), (i, b, d)          # not a single output before the tail
                    untouched += n - tail
                    d += 1
        assert untouched > 100000


def test_overlap_save_segments(cuda, api, orc):
    nchan, nnew = 256, 2048
    w = Shape(500.0, -200.0 / nchan, nchan, 0, [(0.0, 0.2, 70, 1), (10.0, 0.5, 40, 2), (30.0, 1.0, 33, 4)], [1, 2, 4], 6.0, nbeam=2)
    probe = api.Plan(w.fch1, w.foff, nchan, w.tsamp, 1 << 16, w.ranges, w.widths)
    hmin, _, gran = probe.segment_info()
    assert gran == 16 and hmin % 16 == 0 and hmin > 0
    w.nsamp = hmin + nnew                                          # exactly the shortest legal history
    rs = np.random.default_rng(9)
    blocks = [rs.integers(0, 256, size=(2, nnew, nchan), dtype=np.uint8) for _ in range(4)]
    plan = make_plan(api, w, nbeam=2)
    refs = [orc.overlap_save_buffers([blk[b] for blk in blocks], w.nsamp, flip=True) for b in range(2)]
    _, _, dec, nout, off = plan.trial_table()
    prev = None
    for i, blk in enumerate(blocks):
        d_dmt = plan.segment_push(cuda.from_numpy(blk).cuda(), flip=True)
        dmt = d_dmt.cpu().numpy()
        for b in range(2):
            ref = oracle_path(orc, w, refs[b][i], search=False)
            check_dmt_against_oracle(plan, dmt, ref, beam=b)
        if prev is not None:                                       # every row slid by nnew/decim: old outputs repeat, new ones follow
            for d in (0, 69, 70, 109, 110, 142):
                k, n = int(dec[d]), int(nout[d])
                assert n >= nnew // k
                assert np.array_equal(dmt[0][off[d]: off[d] + n - nnew // k], prev[0][off[d] + nnew // k: off[d] + n])
        prev = dmt
    # a history shorter than the longest sweep, or a shift that breaks the decimation phase, is refused
    short = make_plan(api, w, nbeam=2, nsamp=hmin + nnew - 16)
    with pytest.raises(api.SptError) as e:
        short.segment_push(cuda.from_numpy(blocks[0]).cuda())
    assert e.value.code == api.SPT_ERR_SHAPE
    with pytest.raises(api.SptError) as e:
        plan.segment_push(cuda.from_numpy(blocks[0][:, : nnew - 8]).cuda())
    assert e.value.code == api.SPT_ERR_INVALID


@pytest.mark.parametrize("whole_rows", [True, False])
def test_segment_search_matches_the_oracle_window(cuda, api, orc, whole_rows):
    """spt_segment_search after every push: per trial, statistics and candidates of the window (last nnew/k + wmax - 1
    samples) restricted to its first nnew/k start positions, against the oracle's composition of C1-C5 on that window."""
    nchan, nnew = 128, 4096
    widths = [1, 2, 8, 32]
    w = Shape(500.0, -200.0 / nchan, nchan, 0, [(0.0, 0.5, 40, 1), (20.0, 1.0, 24, 2), (50.0, 2.0, 17, 4)], widths, 3.5, nbeam=1)
    probe = api.Plan(w.fch1, w.foff, nchan, w.tsamp, 1 << 16, w.ranges, w.widths)
    hmin, hsearch, gran = probe.segment_info()
    assert hsearch >= hmin + (max(widths) - 1) * 4 - gran
    w.nsamp = hsearch + nnew
    plan = make_plan(api, w, cand_capacity=1 << 22)
    with pytest.raises(api.SptError) as e:                         # a history that covers the sweeps but not the widest boxcar
        make_plan(api, w, nsamp=hmin + nnew).segment_search(cuda.zeros((1, 8), dtype=cuda.int32, device="cuda"), nnew, 5.0)
    assert e.value.code == api.SPT_ERR_SHAPE
    rs = np.random.default_rng(21)
    _, _, dec, nout, off = plan.trial_table()
    total = 0
    d_dmt = cuda.zeros((1, plan.dmt_elems_per_beam), dtype=cuda.int32, device="cuda")
    blocks = []
    for i in range(3):
        blk = rs.normal(128, 12, size=(1, nnew, nchan)).round().clip(0, 255).astype(np.uint8)
        blk[0, 1000 + 300 * i: 1003 + 300 * i, :] += 20            # a zero-DM spike per segment
        blocks.append(blk)
    bufs = orc.overlap_save_buffers([blk[0] for blk in blocks], w.nsamp, flip=False)
    for i, blk in enumerate(blocks):
        # the rows the oracle's search is given are the ORACLE's dedispersion of the stream buffer, so that the pair
        # (push, search) is checked end to end; the GPU's own rows must equal them over the window the search reads
        orows = []
        for rr in oracle_path(orc, w, bufs[i], search=False):
            orows += [rr.dmt[rr.rowoff[j]: rr.rowoff[j + 1]] for j in range(len(rr.nout))]
        d_dmt = plan.segment_push(cuda.from_numpy(blk).cuda(), d_dmt=d_dmt, whole_rows=whole_rows)
        plan.segment_search(d_dmt, nnew, w.threshold)
        n, ovf = plan.candidates_count()
        assert not ovf
        cands = plan.candidates_read()
        s_all, q_all = plan.trial_stats_all(1)
        dmt = d_dmt.cpu().numpy()[0]
        check_segment_against_oracle(orc, plan, dmt, orows, range(plan.ntrials), widths, w.threshold, nnew, cands, s_all[0], q_all[0])
        total += n
    assert total > 1000


def test_push_on_a_non_blocking_stream_takes_the_8bit_body_with_a_tail(cuda, api, orc):
    """Two things no other stream test does.  (1) The pushes run on a torch.cuda.Stream(), a non-blocking stream that does
    not wait for the legacy default stream: the library's one-time zero fill of its working buffers has to be ordered on
    the caller's stream, or it can land after the first block.  (2) Gaussian bytes, as the telescope's are: once the buffer
    holds no more start-up zeros the decimated series span fewer than 256 values, so the decimated ranges of a tail-only
    push (whole_rows = 0) run the dual kernel's 8-BIT body with tail > 0 -- asserted through spt_decimated_compact -- and
    their outputs are compared with the oracle's dedispersion of the oracle's stream buffer."""
    nchan, nnew, nbeam = 256, 2048, 2
    widths = [1, 2, 4, 16]
    w = Shape(500.0, -200.0 / nchan, nchan, 0, [(0.0, 0.2, 70, 1), (10.0, 0.5, 40, 2), (30.0, 1.0, 33, 4)], widths, 6.0, nbeam=nbeam)
    probe = api.Plan(w.fch1, w.foff, nchan, w.tsamp, 1 << 16, w.ranges, w.widths)
    _, hsearch, _ = probe.segment_info()
    w.nsamp = hsearch + nnew + 1024
    npush = (w.nsamp + nnew - 1) // nnew + 2                        # the last two pushes see a buffer without start-up zeros
    rs = np.random.default_rng(12)
    blocks = [rs.normal(128, 10, size=(nnew, nbeam, nchan)).round().clip(0, 255).astype(np.uint8) for _ in range(npush)]
    plan = make_plan(api, w, nbeam=nbeam)
    refs = [orc.overlap_save_buffers([blk[:, b, :] for blk in blocks], w.nsamp, flip=True) for b in range(nbeam)]
    _, _, dec, nout, off = plan.trial_table()
    SENT = -123456789
    s = cuda.cuda.Stream()
    took_8bit = 0
    with cuda.cuda.stream(s):
        for i, blk in enumerate(blocks):
            d_dmt = cuda.full((nbeam, plan.dmt_elems_per_beam), SENT, dtype=cuda.int32, device="cuda")
            plan.segment_push(cuda.from_numpy(blk).cuda(), flip=True, d_dmt=d_dmt, stream=s, spliced=True, whole_rows=False)
            s.synchronize()
            dmt = d_dmt.cpu().numpy()
            if i >= npush - 2:
                for ri in (1, 2):
                    in_use, floor, span = plan.decimated_compact(ri)
                    assert in_use and floor > 0 and span < 256, (i, ri, in_use, floor, span)
                    took_8bit += 1
            elif i == 0:
                assert not plan.decimated_compact(1)[0]             # zeros and noise together span more than a byte
            if 0 < i < npush - 2:
                continue                                            # the oracle's time goes to the first push and the 8-bit ones
            for b in range(nbeam):
                ref = oracle_path(orc, w, refs[b][i], search=False)
                d = 0
                for rr in ref:
                    for j in range(len(rr.nout)):
                        n, k = int(nout[d]), int(dec[d])
                        tail = min(n, nnew // k + max(widths) - 1)
                        got = dmt[b][off[d]: off[d] + n]
                        exp = rr.dmt[rr.rowoff[j]: rr.rowoff[j + 1]]
                        assert np.array_equal(got[n - tail:], exp[n - tail:]), (i, b, d)
                        assert np.all(got[: n - tail] == SENT), (i, b, d)
                        d += 1
    assert took_8bit == 4
