"""NEXT-2 (reading F): corner turn of time-major blocks and overlap-save segments.  The DM transform after
every push must be, bit for bit, the oracle's batch dedispersion of the last nsamp samples of the stream, so that the
last nnew/decim outputs of every trial continue the previous push's."""
import numpy as np
import pytest

from helpers import check_dmt_against_oracle, make_plan
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
    for i in range(3):
        blk = rs.normal(128, 12, size=(1, nnew, nchan)).round().clip(0, 255).astype(np.uint8)
        blk[0, 1000 + 300 * i: 1003 + 300 * i, :] += 20            # a zero-DM spike per segment
        d_dmt = plan.segment_push(cuda.from_numpy(blk).cuda(), d_dmt=d_dmt, whole_rows=whole_rows)
        plan.segment_search(d_dmt, nnew, w.threshold)
        n, ovf = plan.candidates_count()
        assert not ovf
        cands = plan.candidates_read()
        s_all, q_all = plan.trial_stats_all(1)
        dmt = d_dmt.cpu().numpy()[0]
        got = {}
        for c in cands:
            got.setdefault(int(c["trial"]), []).append((int(c["t"]), int(c["width"]), float(c["snr"])))
        for d in range(plan.ntrials):
            row = dmt[off[d]: off[d] + nout[d]]     # (whole_rows = False: only its tail, the window, is defined)
            sx, sxx, t, bw, snr = orc.search_segment(row, widths, w.threshold, nnew // int(dec[d]))
            assert (int(s_all[0, d]), int(q_all[0, d])) == (sx, sxx), d
            g = sorted(got.get(d, []))
            exp = sorted(zip(t.tolist(), bw.tolist(), snr.tolist()))
            near = [x for x in exp if abs(x[2] - w.threshold) <= 1e-3]
            assert abs(len(g) - len(exp)) <= len(near), (d, len(g), len(exp))
            ge = {x[0]: x for x in g}
            for (tt, ww, ss) in exp:
                if tt in ge:
                    assert ge[tt][1] == ww and abs(ge[tt][2] - ss) <= 1e-3, (d, tt)
                else:
                    assert abs(ss - w.threshold) <= 1e-3
            lo = nout[d] - (nnew // int(dec[d]) + max(widths) - 1)
            assert all(lo <= x[0] < lo + nnew // int(dec[d]) for x in g)      # only this segment's start positions
        total += n
    assert total > 1000
