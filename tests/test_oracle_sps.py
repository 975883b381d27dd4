"""Pins for oracle C-D (statistics, boxcar S/N, best width, candidates): PAPER.md:94; SURVEY.md 8(c) P7..P10.

Closed form sqrt(N - w0), exact big-integer statistics, white-noise invariants, pure-Python brute force
on hand-written series (including an exact tie between widths), injected-burst recovery.
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ---- an independent, literal Python statement of C3-C5/D1 (tiny inputs only) -------------------------
def py_search(x, widths, thr):
    n = len(x)
    sx = sum(int(v) for v in x)
    sxx = sum(int(v) * int(v) for v in x)
    var = Fraction(n * sxx - sx * sx, n * n) if n else Fraction(0)
    sigma = math.sqrt(var)
    best = []
    for t in range(max(0, n - widths[0] + 1)):
        b, bw = None, None
        for w in widths:
            if t + w > n:
                break
            S = sum(int(v) for v in x[t:t + w])
            s = 0.0 if (sigma == 0 or n < 2) else (S - w * sx / n) / (sigma * math.sqrt(w))
            if b is None or s > b:
                b, bw = s, w
        best.append((b, bw))
    cands = [(t, bw, b) for t, (b, bw) in enumerate(best) if b >= thr]
    return best, cands


def test_p7_worked_example_sqrt_n_minus_w(orc):
    row = [l.split() for l in open(os.path.join(GOLD, "boxcar_worked_example.txt")) if l.strip() and l[0] != "#"][0]
    N, w0, h = int(row[0]), int(row[1]), int(row[2])
    mu_w, sg_w, snr_w, snr_half, snr_dbl = map(float, row[3:])
    t0 = 300
    x = np.zeros(N, dtype=np.int32)
    x[t0:t0 + w0] = h
    s, q = orc.stats(x)
    mu, sg = orc.mean_sigma(N, s, q)
    assert abs(mu - mu_w) < 1e-12 and abs(sg - sg_w) < 1e-6
    b, bw = orc.best_width(x, [1, 2, 4, 8, 16])
    assert int(np.argmax(b)) == t0 and bw[t0] == w0                 # the arg-max picks the matched width
    assert abs(b[t0] - math.sqrt(N - w0)) < 1e-9 and abs(b[t0] - snr_w) < 1e-4
    assert abs(orc.boxcar_snr(x, 2)[t0] - snr_half) < 5e-3
    assert abs(orc.boxcar_snr(x, 8)[t0] - snr_dbl) < 5e-3
    for hh in (1, 1000, 4_000_000):                                  # independent of the height
        xx = np.zeros(N, dtype=np.int32)
        xx[t0:t0 + w0] = hh
        assert abs(orc.best_width(xx, [1, 2, 4, 8])[0][t0] - math.sqrt(N - w0)) < 1e-9


def test_stats_exact_against_python_bigints(orc):
    rs = np.random.default_rng(2)
    x = rs.integers(0, 4_177_921, size=262_144).astype(np.int32)        # nchan*255*k at its largest, N = 2^18
    s, q = orc.stats(x)
    assert s == sum(int(v) for v in x)
    assert q == sum(int(v) * int(v) for v in x)
    mu, sg = orc.mean_sigma(x.size, s, q)
    n = x.size
    var = Fraction(n * q - s * s, n * n)                                # exact; N*Sxx ~ 1e24 needs > 64 bits
    assert abs(mu - s / n) < 1e-6
    assert abs(sg - math.sqrt(var)) / math.sqrt(var) < 1e-14
    # the float shortcut E[x^2] - E[x]^2 would be useless here (mean^2/var ~ 1e6 for real data): not used
    big = np.full(1000, 2_000_000, dtype=np.int32)
    big[::2] += 1
    _, sgb = orc.mean_sigma(1000, *orc.stats(big))
    assert abs(sgb - 0.5) < 1e-12


def test_sigma_zero_and_short_series(orc):
    x = np.full(100, 12345, dtype=np.int32)
    b, bw = orc.best_width(x, [1, 2, 4])
    assert np.all(b == 0.0) and b.size == 100
    assert orc.best_width(np.array([5], dtype=np.int32), [1, 2])[0].tolist() == [0.0]     # N < 2
    assert orc.best_width(np.zeros(3, np.int32), [4, 8])[0].size == 0                     # every width > N
    assert orc.best_width(np.zeros(0, np.int32), [1])[0].size == 0
    sr = orc.search_plane(x, np.array([0], np.int64), np.array([100], np.int32), [1, 2, 4], 6.0)
    assert sr.count.tolist() == [0]


def test_p10_bruteforce_hand_series_and_tie(orc):
    series = [
        [3, 1, 4, 1, 5, 9, 2, 6, 5, 3],
        [0, 0, 0, 9, 9, 0, 0, 0, 0, 0],
        [10, 0, 0, 0, 0, 0, 0, 0, 0, 10],
        [1, 2, 3, 4, 5, 6, 7, 8, 9, 10],
        [0, 0, 0, 0, 0, 0, 0, 0, 0, 7],
    ]
    for widths in ([1, 2, 4, 8], [1, 3, 5], [2, 4], [1]):
        for x in series:
            best, cands = py_search(x, widths, 1.0)
            b, bw = orc.best_width(np.array(x, np.int32), widths)
            assert len(best) == b.size
            for t, (pb, pw) in enumerate(best):
                assert abs(b[t] - pb) < 1e-12 and bw[t] == pw, (x, widths, t)
            sr = orc.search_plane(np.array(x, np.int32), np.array([0], np.int64), np.array([len(x)], np.int32),
                                  widths, 1.0)
            assert sr.t.tolist() == [c[0] for c in cands]
            assert sr.w.tolist() == [c[1] for c in cands]
    # exact tie between widths: with mean exactly 0, x = [1,1,0,...] has S_1 = 1 at t=0 and S_4 = 2,
    # snr_1 = 1/sigma, snr_4 = 2/(sigma*2) = 1/sigma  -> identical doubles -> the smaller width wins.
    x = np.array([1, 1, 0, 0, -1, -1, 0, 0], dtype=np.int32)
    s1, s4 = orc.boxcar_snr(x, 1)[0], orc.boxcar_snr(x, 4)[0]
    assert s1 == s4 and s1 > 0
    b, bw = orc.best_width(x, [1, 4])
    assert bw[0] == 1 and b[0] == s1
    b, bw = orc.best_width(x, [4, 8])
    assert bw[0] == 4


def test_cumulative_sum_route_equals_literal_boxcar(orc):
    rs = np.random.default_rng(17)
    x = (rs.normal(500_000, 700, size=5000)).astype(np.int32)
    for w in (1, 2, 7, 64, 1000, 5000):
        lit = orc.boxcar_snr(x, w)                        # literal sum over the width
        b, bw = orc.best_width(x, [w])                    # via the exact cumulative sum
        assert lit.size == b.size == 5000 - w + 1
        assert np.array_equal(lit, b) and np.all(bw == w)
        for t in (0, (5000 - w) // 2, 5000 - w):
            assert orc.snr_at(x, w, t) == lit[t]
    assert orc.boxcar_snr(x, 5001).size == 0


def test_valid_widths_shrink_near_the_end(orc):
    x = np.zeros(20, dtype=np.int32)
    x[16:20] = 5
    b, bw = orc.best_width(x, [1, 2, 4, 8])
    assert b.size == 20
    assert bw[16] == 4                   # w = 8 would run off the end at t = 16: not considered
    assert bw[19] == 1 and bw[18] == 2   # only w <= N - t are valid


def test_threshold_is_inclusive(orc):
    rs = np.random.default_rng(23)
    x = rs.integers(0, 1000, size=400).astype(np.int32)
    b, _ = orc.best_width(x, [1, 2, 4])
    thr = float(np.sort(b)[-5])
    sr = orc.search_plane(x, np.array([0], np.int64), np.array([400], np.int32), [1, 2, 4], thr)
    assert sr.count[0] == int((b >= thr).sum()) >= 5
    assert thr in sr.snr.tolist()


def test_p8_white_noise_invariants(orc, synth):
    # burst-free generator output: pooled snr_w has mean 0 and unit variance for every width
    w = synth.workload(1)
    w.bursts = [[]]
    fb = synth.generate(w)
    row = fb.astype(np.int32).sum(axis=0)
    for wd in (1, 2, 4, 8, 16, 32, 64):
        s = orc.boxcar_snr(row, wd)
        n_eff = row.size / wd
        assert abs(s.mean()) < 3.0 / math.sqrt(n_eff) + 0.02, wd
        assert abs(s.std() - 1.0) < 4.0 / math.sqrt(2 * n_eff) + 0.02, wd
    b, _ = orc.best_width(row, w.widths)
    assert (b >= 6.0).sum() == 0          # Gaussian tail Q(6) ~ 1e-9: no crossing in 4096 x 7 evaluations


def test_p9_cfg1_injected_burst_recovered(orc, synth):
    w = synth.workload(1)
    fb = synth.generate(w)
    res = orc.run_path(fb, w.fch1, w.foff, w.tsamp, w.ranges, w.widths, w.threshold)[0]
    assert res.nout[50] == 4096 - 1089 and res.dm[50] == 50.0
    s = res.search
    assert s.count.sum() > 0
    i = int(np.argmax(s.snr))
    trial = int(np.searchsorted(s.candoff, i, side="right") - 1)
    # injected: DM 50 (= trial 50), t0 = 1000, width 4, +24 per channel over N(128,16) noise in 64 channels:
    # expected S/N = 24*sqrt(64*4)/16 = 24, measured scatters by ~1 sigma (+ the burst inflates sigma a little)
    assert abs(trial - 50) <= 1 and abs(int(s.t[i]) - 1000) <= 2 and int(s.w[i]) in (2, 4, 8)
    assert abs(s.snr[i] - 24.0) <= 3.0
    # every candidate lies inside its trial's valid range
    for d in range(101):
        tt = s.t[s.candoff[d]:s.candoff[d + 1]]
        assert np.all(tt >= 0) and np.all(tt <= res.nout[d] - 1)
        assert np.all(np.diff(tt) > 0)


def test_p9_reduced_cfg3_bursts_recovered_in_every_range(orc, synth):
    # one strong burst per DM range, on a short cfg-3-shaped beam; recovered within 2 DM steps / 2 widths
    w = synth.workload(3, nsamp=32768)
    w.nchan = 256
    w.foff = -200.0 / 256
    w.ranges = [(0.0, 0.2, 400, 1), (500.0, 0.5, 40, 2), (1000.0, 1.0, 21, 4)]
    mk = synth.Burst
    inj = [(60.0, 3000, 4, 30.0), (510.0, 5000, 8, 30.0), (1010.0, 2000, 16, 30.0)]
    w.bursts = [[mk(dm=dm, t0=t0, width=wd, snr=snr, amp=snr * w.std / math.sqrt(w.nchan * wd))
                 for dm, t0, wd, snr in inj]]
    fb = synth.generate(w)
    res = orc.run_path(fb, w.fch1, w.foff, w.tsamp, w.ranges, w.widths, w.threshold)
    for r, (dm, t0, wd, snr) in zip(res, inj):
        s = r.search
        assert s.count.sum() > 0
        i = int(np.argmax(s.snr))
        trial = int(np.searchsorted(s.candoff, i, side="right") - 1)
        step = r.dm[1] - r.dm[0]
        assert abs(r.dm[trial] - dm) <= 2 * step + 1e-9, (dm, r.dm[trial])
        assert abs(int(s.t[i]) * r.decim - t0) <= max(2 * wd, 2 * r.decim)
        assert s.snr[i] >= 0.6 * snr and s.snr[i] <= snr + 4.0
        assert wd // (2 * r.decim) <= int(s.w[i]) <= max(1, 2 * wd // r.decim)


def test_search_plane_matches_per_trial_calls(orc, synth):
    w = synth.workload(1)
    fb = synth.generate(w)
    res = orc.run_path(fb, w.fch1, w.foff, w.tsamp, w.ranges, w.widths, w.threshold)[0]
    s = res.search
    for d in (0, 49, 50, 51, 100):
        row = res.dmt[res.rowoff[d]:res.rowoff[d + 1]]
        assert (int(s.sum[d]), int(s.sumsq[d])) == orc.stats(row)
        b, bw = orc.best_width(row, w.widths)
        sel = np.nonzero(b >= w.threshold)[0]
        assert s.t[s.candoff[d]:s.candoff[d + 1]].tolist() == sel.tolist()
        assert s.w[s.candoff[d]:s.candoff[d + 1]].tolist() == bw[sel].tolist()
        assert np.array_equal(s.snr[s.candoff[d]:s.candoff[d + 1]], b[sel])
