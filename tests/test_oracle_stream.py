"""Pins of the oracle's stream definitions (reading F): worked examples written out by hand and the
overlap-save identity -- the buffer after push i, dedispersed, continues the buffer after push i-1."""
import numpy as np


def test_corner_turn_worked_example(orc):
    x = np.array([[1, 2, 3], [4, 5, 6]], dtype=np.uint8)                 # 2 samples x 3 channels, time-major
    assert orc.corner_turn(x).tolist() == [[1, 4], [2, 5], [3, 6]]         # channel rows
    assert orc.corner_turn(x, flip=True).tolist() == [[3, 6], [2, 5], [1, 4]]   # last channel (highest frequency) first


def test_corner_turn_spliced_worked_example(orc):
    # 2 samples x 2 beams x 3 channels, time-spliced: sample 0 of beam 0, sample 0 of beam 1, sample 1 of beam 0, ...
    x = np.array([[[1, 2, 3], [11, 12, 13]], [[4, 5, 6], [14, 15, 16]]], dtype=np.uint8)
    b0, b1 = orc.corner_turn_spliced(x)
    assert b0.tolist() == [[1, 4], [2, 5], [3, 6]] and b1.tolist() == [[11, 14], [12, 15], [13, 16]]
    assert orc.corner_turn_spliced(x, flip=True)[1].tolist() == [[13, 16], [12, 15], [11, 14]]


def test_overlap_save_buffers_worked_example(orc):
    b0 = np.array([[1, 10], [2, 20]], dtype=np.uint8)                    # 2 new samples x 2 channels per push
    b1 = np.array([[3, 30], [4, 40]], dtype=np.uint8)
    bufs = orc.overlap_save_buffers([b0, b1], nsamp=3)
    assert bufs[0].tolist() == [[0, 1, 2], [0, 10, 20]]                   # one sample of zero history, then block 0
    assert bufs[1].tolist() == [[2, 3, 4], [20, 30, 40]]                  # the last sample of block 0 is the history


def test_overlap_save_continues_the_dm_transform(orc):
    """With history >= the longest sweep, the DM transform of the buffer after push i, shifted by the new samples, is
    the DM transform of one long observation: nothing is lost or doubled at segment borders."""
    rs = np.random.default_rng(1)
    nchan, nnew, npush = 16, 64, 4
    fch1, foff, tsamp = 500.0, -12.5, 1.31072e-3
    dly = orc.delay_table(fch1, foff, nchan, tsamp, 0.0, 1.0, 12, 1)
    hist = int(dly.max())
    hist += (-hist) % 16
    nsamp = hist + nnew
    blocks = [rs.integers(0, 256, size=(nnew, nchan), dtype=np.uint8) for _ in range(npush)]
    bufs = orc.overlap_save_buffers(blocks, nsamp)
    whole = np.concatenate([np.zeros((nchan, hist), dtype=np.uint8)] + [orc.corner_turn(b) for b in blocks], axis=1)
    no_w = orc.nout(dly, whole.shape[1], 1)
    full, off_w = orc.dedisperse(whole, dly, no_w)
    no = orc.nout(dly, nsamp, 1)
    for i, buf in enumerate(bufs):
        out, off = orc.dedisperse(buf, dly, no)
        for d in range(dly.shape[0]):
            row = out[off[d]: off[d + 1]]
            a = i * nnew                                                  # buffer start inside the long observation
            assert np.array_equal(row, full[off_w[d] + a: off_w[d] + a + no[d]])
            assert no[d] >= nnew                                          # every push yields nnew new outputs per trial


def test_segment_windows_report_every_start_once(orc):
    """Window arithmetic of the segment search (reading F): with row length n, segment length s and widest boxcar wmax,
    segment i reports the row-relative starts [n - s - (wmax-1), n - (wmax-1)), i.e. the stream starts
    [i*s + n - s - wmax + 1, (i+1)*s + n - s - wmax + 1): consecutive segments tile the stream, and every reported start
    has all its boxcars inside the data seen so far."""
    rs = np.random.default_rng(0)
    n, s, widths = 300, 64, [1, 4, 16]
    stream = rs.integers(0, 1000, size=n + 5 * s).astype(np.int32)
    seen = []
    for i in range(6):
        row = stream[i * s: i * s + n]                              # what the push leaves in the row (it slid by s)
        sx, sxx, t, bw, snr = orc.search_segment(row, widths, -1e9, s)      # threshold so low that every start is reported
        assert t.size == s and t[0] == n - s - (max(widths) - 1) and np.all(np.diff(t) == 1)
        assert np.all(t + max(widths) <= n)                         # the widest boxcar fits
        seen.append(t + i * s)                                      # stream positions
        win = row[n - (s + max(widths) - 1):]
        assert sx == int(win.sum())                                 # statistics are the window's
    allpos = np.concatenate(seen)
    assert np.array_equal(allpos, np.arange(allpos[0], allpos[0] + 6 * s))   # contiguous, no gap, no repeat
