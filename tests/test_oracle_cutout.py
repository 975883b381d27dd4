"""Pins of the oracle's candidate cut-outs (reading H; Eq. 4 / App. A)."""
import math

import numpy as np

TSAMP = 1.31072e-3


def test_delta_dm_formula_and_the_papers_inconsistency(orc):
    # Eq. 4 as printed: sqrt(pi)/1382 * W_s * (S/S(dDM)) * nu_MHz^3 / dnu_MHz
    w, nu, bw = 2.0e-3, 400.0, 200.0
    assert math.isclose(orc.delta_dm(w, nu, bw), math.sqrt(math.pi) / 1382 * w * 10 * nu ** 3 / bw, rel_tol=1e-15)
    assert math.isclose(orc.delta_dm(w, nu, bw, snr_ratio=0.5) * 5, orc.delta_dm(w, nu, bw), rel_tol=1e-15)
    # The derivation it comes from (Eq. A3 + A4): S(dDM)/S = sqrt(pi)/(2 zeta),
    # zeta = 6.91e-3 dDM dnu_MHz / (W_ms nu_GHz^3).  Solving for dDM gives a constant of 13820, not 1382: with the printed
    # constant the S/N ratio reached at dDM is 0.01, not the 0.1 asked for.  Both facts are pinned here.
    zeta = lambda ddm: 6.91e-3 * ddm * bw / ((w * 1e3) * (nu * 1e-3) ** 3)
    assert math.isclose(math.sqrt(math.pi) / (2 * zeta(orc.delta_dm(w, nu, bw, constant=13820.0))), 0.1, rel_tol=1e-12)
    assert math.isclose(math.sqrt(math.pi) / (2 * zeta(orc.delta_dm(w, nu, bw))), 0.01, rel_tol=1e-12)


def _burst(nchan=64, nsamp=6000, dm=40.0, t0=3000, amp=40):
    fch1, foff = 500.0, -200.0 / nchan
    x = np.full((nchan, nsamp), 10, dtype=np.uint8)
    f = fch1 + np.arange(nchan) * foff
    d = np.floor(4.148808e3 * dm * (f ** -2 - fch1 ** -2) / TSAMP + 0.5).astype(int)
    for c in range(nchan):
        x[c, t0 + d[c]] += amp
    return x, fch1, foff


def test_burst_gives_a_line_and_a_bow_tie(orc):
    x, fch1, foff = _burst()
    nt, ndm, nf = 65, 33, 8
    dds, dmt = orc.cutout(x, fch1, foff, TSAMP, 40.0, 8.0, ndm, 3000 - nt // 2, 1, nt, nf)
    assert np.all(dds.argmax(axis=1) == nt // 2)                       # a straight line across the band at the arrival time
    i, j = np.unravel_index(dmt.argmax(), dmt.shape)
    assert (i, j) == (ndm // 2, nt // 2)                               # the knot of the bow tie: true DM, arrival time
    assert dmt[ndm // 2, nt // 2] == 64 * 50 and dmt[0].max() < dmt[ndm // 2].max()
    assert np.array_equal(dds.sum(axis=0), dmt[ndm // 2])              # centre row of the transform = band-summed spectrum


def test_rows_equal_the_batch_dedispersion(orc):
    rs = np.random.default_rng(2)
    nchan, nsamp = 32, 3000
    x = rs.integers(0, 256, size=(nchan, nsamp), dtype=np.uint8)
    fch1, foff = 500.0, -6.25
    dm0, ddm, ndm, ts, nt = 30.0, 6.0, 7, 500, 100
    dds, dmt = orc.cutout(x, fch1, foff, TSAMP, dm0, ddm, ndm, ts, 1, nt, 4)
    for i in range(ndm):
        dly = orc.delay_table(fch1, foff, nchan, TSAMP, (dm0 - ddm) + i * (2 * ddm / (ndm - 1)), 1.0, 1, 1)
        no = orc.nout(dly, nsamp, 1)
        row, _ = orc.dedisperse(x, dly, no)
        assert np.array_equal(dmt[i], row[ts: ts + nt])
    # time binning is a sum of adjacent samples, frequency bands a sum of adjacent channels
    dds2, dmt2 = orc.cutout(x, fch1, foff, TSAMP, dm0, ddm, ndm, ts, 4, nt // 4, 2)
    assert np.array_equal(dmt2, dmt.reshape(ndm, nt // 4, 4).sum(axis=2))
    assert np.array_equal(dds2, dds.reshape(2, 2, nt // 4, 4).sum(axis=(1, 3)))


def test_samples_outside_the_data_count_as_zero(orc):
    x = np.full((8, 100), 3, dtype=np.uint8)
    dds, dmt = orc.cutout(x, 500.0, -25.0, TSAMP, 0.0, 0.0, 1, -10, 1, 130, 2)
    assert dds[:, :10].sum() == 0 and dds[:, 110:].sum() == 0 and np.all(dds[:, 10:110] == 12)
    assert np.all(dmt[0, 10:110] == 24) and dmt[0, :10].sum() == 0
