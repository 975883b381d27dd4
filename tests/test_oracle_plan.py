"""Pins for oracle A (plan + delay table): PAPER.md:51-58 (Eq. 1-2), SURVEY.md 8(c)-A.

None of these re-types the oracle's double-precision formula: the closed form is evaluated in exact
rational arithmetic (fractions.Fraction), plus physical spot checks, invariants and the stored
spot values of tests/golden/delay_spot_values.txt.
"""
import os
from fractions import Fraction

import numpy as np
import pytest

TSAMP = 1.31072e-3
D = Fraction("4148.808")            # BASELINE.json north_star (2)
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def exact_delay(fch1, foff, c, tsamp, dm, k):
    """floor(x + 1/2) with x = D*DM*(f^-2 - ftop^-2)/(tsamp*k) in exact rationals (inputs = the doubles)."""
    f = Fraction(fch1) + c * Fraction(foff)
    ftop = Fraction(fch1)
    x = D * Fraction(dm) * (1 / (f * f) - 1 / (ftop * ftop)) / (Fraction(tsamp) * k)
    return (x + Fraction(1, 2)).__floor__()


def test_cfg1_whole_table_exact_rational(orc):
    dly = orc.delay_table(500.0, -3.125, 64, TSAMP, 0.0, 1.0, 101, 1)
    assert dly.shape == (101, 64) and dly.dtype == np.int32
    for i in range(101):
        for c in range(64):
            assert dly[i, c] == exact_delay(500.0, -3.125, c, TSAMP, 0.0 + i * 1.0, 1), (i, c)


@pytest.mark.parametrize("fch1,foff,nchan,rng_", [
    (750.0, -0.09765625, 2048, (0.0, 0.5, 2048, 1)),
    (500.0, -0.048828125, 4096, (0.0, 0.2, 2500, 1)),
    (500.0, -0.048828125, 4096, (500.0, 0.5, 1000, 2)),
    (500.0, -0.048828125, 4096, (1000.0, 1.0, 1001, 4)),
])
def test_sampled_entries_exact_rational(orc, fch1, foff, nchan, rng_):
    lo, step, ndm, k = rng_
    dly = orc.delay_table(fch1, foff, nchan, TSAMP, lo, step, ndm, k)
    rs = np.random.default_rng(7)
    picks = [(0, 0), (ndm - 1, nchan - 1), (ndm - 1, 0), (0, nchan - 1), (1, nchan - 1), (ndm // 2, nchan // 2)]
    picks += [(int(rs.integers(ndm)), int(rs.integers(nchan))) for _ in range(400)]
    for i, c in picks:
        dm = lo + float(i) * step            # the oracle's trial DM (reading A3: multiply, do not accumulate)
        assert dly[i, c] == exact_delay(fch1, foff, c, TSAMP, dm, k), (i, c)


def test_invariants_reference_channel_dm0_monotone(orc):
    for (fch1, foff, nchan, lo, step, ndm, k) in [(500.0, -3.125, 64, 0.0, 1.0, 101, 1),
                                                  (750.0, -0.09765625, 2048, 0.0, 0.5, 2048, 1),
                                                  (500.0, -0.048828125, 4096, 500.0, 0.5, 1000, 2)]:
        dly = orc.delay_table(fch1, foff, nchan, TSAMP, lo, step, ndm, k)
        assert np.all(dly[:, 0] == 0)                       # channel 0 = f_top is the reference
        if lo == 0.0:
            assert np.all(dly[0] == 0)                      # DM 0: no shift anywhere
        assert np.all(np.diff(dly, axis=1) >= 0)            # later at lower frequency
        assert np.all(np.diff(dly, axis=0) >= 0)            # later at higher DM
        assert dly.min() >= 0


def test_physical_scale_4p15ms_per_dm_at_1ghz(orc):
    # Against a reference at "infinite" frequency, 1 GHz lags by 4.148808 ms per unit DM (the meaning of D).
    fch1 = 1.0e9
    foff = -(1.0e9 - 1000.0)          # channel 1 sits at exactly 1000 MHz
    dly = orc.delay_table(fch1, foff, 2, 1.0e-6, 0.0, 100.0, 2, 1)
    assert dly[1, 1] == 414881        # 100 * 4148.808 us = 414880.8 samples of 1 us
    # and it scales as f^-2: 500 MHz lags 4x more
    dly2 = orc.delay_table(fch1, -(1.0e9 - 500.0), 2, 1.0e-6, 0.0, 100.0, 2, 1)
    assert dly2[1, 1] == 1659523      # 4 * 414880.8 = 1659523.2


def test_band3_dm2000_sweep_is_59s(orc):
    # the DM-2000 sweep across Band 3 (300-500 MHz); Eq. 2 gives 59.0 s = 45017 samples.
    dly = orc.delay_table(500.0, -200.0, 2, TSAMP, 2000.0, 1.0, 1, 1)
    x = D * 2000 * (Fraction(1, 300 * 300) - Fraction(1, 500 * 500))          # seconds, exact
    assert abs(float(x) - 59.0) < 0.01
    assert dly[0, 1] == (x / Fraction(TSAMP) + Fraction(1, 2)).__floor__() == 45017


def test_golden_spot_values(orc):
    rows = [l.split() for l in open(os.path.join(GOLD, "delay_spot_values.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 14
    for fch1, foff, dm, k, c, want in rows:
        c, k = int(c), int(k)
        dly = orc.delay_table(float(fch1), float(foff), c + 1, TSAMP, float(dm), 1.0, 1, k)
        assert dly[0, c] == int(want), (fch1, dm, k, c)


def test_decimated_delay_is_rounded_at_decimated_period(orc):
    # reading A4: round(x/k), not round(x)/k
    d1 = orc.delay_table(500.0, -0.048828125, 4096, TSAMP, 500.0, 0.5, 50, 1)
    d2 = orc.delay_table(500.0, -0.048828125, 4096, TSAMP, 500.0, 0.5, 50, 2)
    assert np.all(np.abs(2 * d2.astype(np.int64) - d1) <= 1)
    assert np.any(2 * d2 != d1)       # it is a different table, not d1 // 2 * 2


def test_nout_ragged_and_clamped(orc):
    dly = orc.delay_table(500.0, -0.048828125, 4096, TSAMP, 1000.0, 1.0, 1001, 4)
    no = orc.nout(dly, 1 << 17, 4)
    assert no[0] == 32768 - 5624 and no[-1] == 32768 - 11249          # 27144 ... 21519
    no4 = orc.nout(dly, 1 << 15, 4)                                   # cfg 4: sweep longer than the data
    assert no4.min() == 0 and (no4 == 0).sum() == 544
    assert np.all(no4 >= 0)


def test_bad_arguments_rejected(orc):
    out = np.zeros((1, 4), dtype=np.int32)
    L = orc.lib()
    assert L.orc_delay_table(500.0, +1.0, 4, TSAMP, 0.0, 1.0, 1, 1, out.ctypes.data) != 0   # foff >= 0
    assert L.orc_delay_table(500.0, -1.0, 0, TSAMP, 0.0, 1.0, 1, 1, out.ctypes.data) != 0
    assert L.orc_delay_table(500.0, -1.0, 4, TSAMP, 0.0, 1.0, 1, 0, out.ctypes.data) != 0
