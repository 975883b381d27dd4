"""Pins of the oracle's sifting stage (reading G): DBSCAN against scikit-learn's implementation (core
points, noise and the partition of the core points are unique in DBSCAN, so they must agree exactly), hand-made cases
for the cluster representative, the cuts and the anti-coincidence rule."""
import numpy as np
import pytest
import sklearn.cluster as sk   # a hard import: without it the oracle's DBSCAN would have no external pin


@pytest.mark.parametrize("seed", range(5))
def test_dbscan_agrees_with_scikit_learn(orc, seed):
    rs = np.random.default_rng(seed)
    centres = rs.uniform(0, 20, size=(6, 2))
    pts = np.concatenate([c + rs.normal(0, 0.25, size=(40, 2)) for c in centres] + [rs.uniform(0, 20, size=(80, 2))])
    core, label = orc.dbscan(pts[:, 0], pts[:, 1], 0.5, 5)
    ref = sk.DBSCAN(eps=0.5, min_samples=5).fit(pts)
    ref_core = np.zeros(len(pts), dtype=bool)
    ref_core[ref.core_sample_indices_] = True
    assert np.array_equal(core, ref_core)
    # same partition of the core points (label values differ: compare co-membership through a relabelling)
    ci = np.flatnonzero(core)
    pairs = {}
    for i in ci:
        pairs.setdefault(int(label[i]), set()).add(int(ref.labels_[i]))
    assert all(len(v) == 1 for v in pairs.values())
    assert len({next(iter(v)) for v in pairs.values()}) == len(pairs)
    # noise = points that are neither core nor within eps of a core point
    d2 = ((pts[:, None, :] - pts[None, :, :]) ** 2).sum(-1)
    border_or_core = ((d2 <= 0.25) & core[None, :]).any(axis=1)
    assert np.array_equal(ref.labels_ == -1, ~border_or_core)


def _sift(orc, cands, nbeam=1, **kw):
    b, d, t, w, s = (np.array(x) for x in zip(*cands))
    dm = np.arange(100, dtype=np.float64) * 0.5 + 20.0               # trial -> DM (all above the DM cut)
    dec = np.ones(100, dtype=np.int64)
    return [m.tolist() for m in orc.sift(b, d, t, w, s.astype(np.float64), dm, dec, 1e-3, nbeam, **kw)]


def test_cluster_representative_and_noise(orc):
    # five candidates 0.1 s apart on one trial: one cluster, the strongest survives; a sixth far away is noise
    c = [(0, 10, 100 * i, 2, 11.0 + i) for i in range(5)] + [(0, 10, 9000, 2, 50.0)]
    k1, k2, k3 = _sift(orc, c)
    assert k1 == [False, False, False, False, True, False]
    # four points only: no core point (min_pts = 5), everything is noise
    assert _sift(orc, c[:4])[0] == [False] * 4
    # exact S/N tie inside a cluster: the smaller (trial, t) is the representative
    c = [(0, 10, 100 * i, 2, 12.0) for i in range(5)]
    assert _sift(orc, c)[0] == [True, False, False, False, False]


def test_border_point_joins_its_strongest_core_neighbour(orc):
    # two chains of core points (S/N 11 and 13) and one non-core point within eps of the end of both, stronger than all
    left = [(0, 10, 100 * i, 2, 11.0) for i in range(5)]             # t = 0 .. 0.4 s
    right = [(0, 10, 1300 + 100 * i, 2, 13.0) for i in range(5)]     # t = 1.3 .. 1.7 s
    bridge = [(0, 10, 850, 2, 40.0)]                                  # 0.45 s from the left end, 0.45 s from the right end
    k1 = _sift(orc, left + right + bridge)[0]
    # the bridge has 3 points within eps (itself and the two ends) -> not core; it joins the right cluster (13 > 11) and,
    # being the strongest member, represents it; the left cluster keeps its own representative
    assert k1 == [True, False, False, False, False] + [False] * 5 + [True]


def test_cuts(orc):
    mk = lambda snr, trial, width: [(0, trial, 100 * i, width, snr if i == 0 else snr - 1) for i in range(5)]
    # DM of trial d is 20 + 0.5 d; tsamp 1 ms so width 101 samples = 0.101 s
    assert _sift(orc, mk(12.0, 10, 2))[1][0] is True
    assert _sift(orc, mk(9.9, 10, 2))[1][0] is False                  # S/N < 10
    assert _sift(orc, mk(12.0, 10, 101))[1][0] is False               # wider than 100 ms
    assert _sift(orc, mk(12.0, 10, 100))[1][0] is True
    assert _sift(orc, mk(12.0, 10, 2), dm_min=25.5)[1][0] is False    # DM 25 < 25.5


def test_anti_coincidence(orc):
    # the same arrival time in 3 of 4 beams is RFI; a candidate seen in 1 beam survives
    one = lambda beam, t0, snr: [(beam, 10, t0 + 100 * i, 2, snr if i == 0 else snr - 1) for i in range(5)]
    c = one(0, 0, 15.0) + one(1, 3, 16.0) + one(2, -0 + 5, 17.0) + one(3, 50000, 18.0)
    k1, k2, k3 = _sift(orc, c, nbeam=4, coinc_window_s=0.02)
    assert [k2[i] for i in (0, 5, 10, 15)] == [True] * 4
    assert [k3[i] for i in (0, 5, 10, 15)] == [False, False, False, True]
    # with the window switched off nothing is removed
    assert _sift(orc, c, nbeam=4)[2] == k2
