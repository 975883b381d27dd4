"""Pins for oracle B (decimation + brute-force dedispersion): PAPER.md:80, 90; SURVEY.md 8(c)-B P1..P6.

The references here are written independently of oracle.cpp: pure-Python triple loops, numpy
reductions, and structural properties (one-hot, constant, shift).
"""
import numpy as np
import pytest

TSAMP = 1.31072e-3


def py_dedisperse(y, delay, nout):
    """Literal triple loop in Python ints (tiny inputs only)."""
    rows = []
    for d in range(delay.shape[0]):
        row = []
        for t in range(int(nout[d])):
            acc = 0
            for c in range(y.shape[0]):
                acc += int(y[c][t + int(delay[d][c])])
            row.append(acc)
        rows.append(row)
    return rows


def rows_of(dmt, rowoff):
    return [dmt[rowoff[i]:rowoff[i + 1]] for i in range(len(rowoff) - 1)]


@pytest.mark.parametrize("dtype,hi", [(np.uint8, 256), (np.uint16, 1021)])
def test_p2_bruteforce_triple_loop_tiny(orc, dtype, hi):
    rs = np.random.default_rng(11)
    nchan, ns, ndm = 8, 64, 5
    y = rs.integers(0, hi, size=(nchan, ns)).astype(dtype)
    delay = np.sort(rs.integers(0, 20, size=(ndm, nchan)), axis=1).astype(np.int32)
    delay[:, 0] = 0
    nout = (ns - delay[:, -1]).astype(np.int32)
    dmt, rowoff = orc.dedisperse(y, delay, nout)
    want = py_dedisperse(y, delay, nout)
    for got, w in zip(rows_of(dmt, rowoff), want):
        assert got.tolist() == w


def test_p2_all_255_hits_the_integer_range(orc):
    nchan, ns = 4096, 40
    y = np.full((nchan, ns), 255, dtype=np.uint8)
    delay = np.zeros((2, nchan), dtype=np.int32)
    delay[1] = np.minimum(np.arange(nchan) // 512, 7)
    nout = (ns - delay[:, -1]).astype(np.int32)
    dmt, rowoff = orc.dedisperse(y, delay, nout)
    assert np.all(dmt == 4096 * 255)
    y16 = np.full((nchan, ns), 1020, dtype=np.uint16)        # k = 4 decimated maximum
    dmt, _ = orc.dedisperse(y16, delay, nout)
    assert np.all(dmt == 4096 * 1020)                        # 4,177,920


def test_p1_dm0_equals_channel_sum(orc, synth):
    w = synth.workload(1)
    fb = synth.generate(w)
    dly = orc.delay_table(w.fch1, w.foff, w.nchan, w.tsamp, 0.0, 1.0, 101, 1)
    no = orc.nout(dly, w.nsamp, 1)
    dmt, rowoff = orc.dedisperse(fb, dly, no)
    assert no[0] == w.nsamp
    assert np.array_equal(dmt[rowoff[0]:rowoff[1]], fb.astype(np.int64).sum(axis=0))


def test_p3_one_hot_pins_direction_and_offsets(orc):
    # x[c*][t*] = v  =>  out[d][t* - delay[d][c*]] = v and zero elsewhere: the read is FORWARD in time.
    nchan, ns = 16, 200
    dly = orc.delay_table(500.0, -12.5, nchan, TSAMP, 0.0, 3.0, 12, 1)
    no = orc.nout(dly, ns, 1)
    for (cs, ts, v) in [(15, 150, 7), (5, 60, 255), (0, 10, 1)]:
        y = np.zeros((nchan, ns), dtype=np.uint8)
        y[cs, ts] = v
        dmt, rowoff = orc.dedisperse(y, dly, no)
        for d, row in enumerate(rows_of(dmt, rowoff)):
            want = np.zeros(no[d], dtype=np.int32)
            tt = ts - dly[d, cs]
            if 0 <= tt < no[d]:
                want[tt] = v
            assert np.array_equal(row, want), (cs, ts, d)


def test_p4_constant_input(orc):
    nchan, ns = 64, 3000
    dly = orc.delay_table(500.0, -3.125, nchan, TSAMP, 0.0, 1.0, 101, 1)
    no = orc.nout(dly, ns, 1)
    y = np.full((nchan, ns), 37, dtype=np.uint8)
    dmt, _ = orc.dedisperse(y, dly, no)
    assert np.all(dmt == nchan * 37) and dmt.size == no.astype(np.int64).sum()
    y4 = orc.decimate(y, 4)
    dly4 = orc.delay_table(500.0, -3.125, nchan, TSAMP, 0.0, 1.0, 101, 4)
    dmt4, _ = orc.dedisperse(y4, dly4, orc.nout(dly4, ns, 4))
    assert np.all(dmt4 == nchan * 4 * 37)


def test_p5_time_shift_of_input_shifts_every_row(orc):
    rs = np.random.default_rng(5)
    nchan, ns, s = 32, 1500, 8
    base = rs.integers(0, 256, size=(nchan, ns + s)).astype(np.uint8)
    a, b = np.ascontiguousarray(base[:, :ns]), np.ascontiguousarray(base[:, s:])
    for k in (1, 2, 4):
        dly = orc.delay_table(500.0, -6.25, nchan, TSAMP, 0.0, 2.0, 40, k)
        no = orc.nout(dly, ns, k)
        ya, yb = (a, b) if k == 1 else (orc.decimate(a, k), orc.decimate(b, k))
        da, off = orc.dedisperse(ya, dly, no)
        db, _ = orc.dedisperse(yb, dly, no)
        for d in range(40):
            ra, rb = da[off[d]:off[d + 1]], db[off[d]:off[d + 1]]
            assert np.array_equal(ra[s // k:], rb[:len(rb) - s // k]), (k, d)


def test_p6_decimation_sums(orc):
    rs = np.random.default_rng(3)
    x = rs.integers(0, 256, size=(7, 1003)).astype(np.uint8)
    for k in (1, 2, 3, 4, 8):
        y = orc.decimate(x, k)
        nk = 1003 // k
        assert y.shape == (7, nk) and y.dtype == np.uint16
        want = x[:, :nk * k].astype(np.int64).reshape(7, nk, k).sum(axis=2)       # numpy, independent
        assert np.array_equal(y, want)
        assert np.array_equal(y.sum(axis=1), x[:, :nk * k].astype(np.int64).sum(axis=1))
    # decimate-by-4 == decimate-by-2 twice (on the sums); k = 1 is the identity
    y2 = orc.decimate(x, 2).astype(np.int64)
    y22 = y2[:, :(y2.shape[1] // 2) * 2].reshape(7, -1, 2).sum(axis=2)
    assert np.array_equal(orc.decimate(x, 4), y22)
    assert np.array_equal(orc.decimate(x, 1), x)
    assert orc.decimate(np.full((1, 8), 255, np.uint8), 4).tolist() == [[1020, 1020]]


def test_point_evaluation_agrees_with_rows(orc, synth):
    # dedisperse_point goes from the RAW bytes (decimation folded in): a second, independent route.
    w = synth.workload(3, nsamp=16384)
    fb = synth.generate(w)
    rs = np.random.default_rng(9)
    for (lo, step, ndm, k) in [(0.0, 0.2, 40, 1), (500.0, 0.5, 30, 2), (1000.0, 1.0, 20, 4)]:
        dly = orc.delay_table(w.fch1, w.foff, w.nchan, w.tsamp, lo, step, ndm, k)
        no = orc.nout(dly, w.nsamp, k)
        y = fb if k == 1 else orc.decimate(fb, k)
        dmt, off = orc.dedisperse(y, dly, no)
        for _ in range(25):
            d = int(rs.integers(ndm))
            if no[d] == 0:
                continue
            t = int(rs.integers(no[d]))
            assert dmt[off[d] + t] == orc.dedisperse_point(fb, dly[d], k, t)
        d = ndm - 1
        if no[d] > 0:                                   # last valid sample touches the end of the data
            assert dmt[off[d] + no[d] - 1] == orc.dedisperse_point(fb, dly[d], k, int(no[d]) - 1)


def test_zero_length_trials_are_legal(orc):
    y = np.ones((4, 10), dtype=np.uint8)
    delay = np.array([[0, 1, 2, 3], [0, 4, 8, 12], [0, 3, 6, 10]], dtype=np.int32)
    no = orc.nout(delay, 10, 1)
    assert no.tolist() == [7, 0, 0]
    dmt, off = orc.dedisperse(y, delay, no)
    assert dmt.tolist() == [4] * 7 and off.tolist() == [0, 7, 7, 7]
