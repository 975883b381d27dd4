"""Candidate sifting (reading G) on the GPU against the oracle: the same list in, the same survivors
out, stage by stage (DBSCAN representatives, cuts, anti-coincidence)."""
import numpy as np
import pytest

from helpers import make_plan
from test_gpu_parity import TSAMP, Shape, mini3, run_gpu

pytestmark = pytest.mark.gpu


def keyset(c):
    return set(zip(c["beam"].tolist(), c["trial"].tolist(), c["t"].tolist()))


def oracle_sift(orc, plan, cands, nbeam, **kw):
    dm, _, dec, _, _ = plan.trial_table()
    return orc.sift(cands["beam"], cands["trial"], cands["t"], cands["width"], cands["snr"].astype(np.float64), dm, dec,
                    TSAMP, nbeam, **kw)


def random_list(api, rs, nbeam, ntrials, n):
    """Clusters, chains, isolated points, many exact S/N ties; unique (beam, trial, t)."""
    rec = {}
    for b in range(nbeam):
        for _ in range(12):
            d0, t0 = int(rs.integers(0, ntrials)), int(rs.integers(0, 40000))
            for _ in range(int(rs.integers(1, 25))):
                d = int(np.clip(d0 + rs.integers(-2, 3), 0, ntrials - 1))
                t = int(max(0, t0 + rs.integers(-300, 301)))
                rec[(b, d, t)] = (int(rs.choice([1, 2, 4, 64, 128])), float(np.round(rs.uniform(8, 14), 1)))
        for _ in range(n // nbeam // 4):
            rec[(b, int(rs.integers(0, ntrials)), int(rs.integers(0, 40000)))] = (1, float(np.round(rs.uniform(8, 30), 1)))
    out = np.zeros(len(rec), dtype=api.CAND_DTYPE)
    for i, ((b, d, t), (w, s)) in enumerate(rec.items()):
        out[i] = (b, d, t, w, s)
    return out[rs.permutation(out.size)]


@pytest.mark.parametrize("seed", range(3))
def test_random_lists_stage_by_stage(cuda, api, orc, seed):
    w = Shape(500.0, -3.125, 64, 65536, [(0.0, 0.5, 60, 1), (30.0, 1.0, 40, 2)], [1, 2, 4], 6.0, nbeam=4)
    plan = make_plan(api, w, nbeam=4)
    rs = np.random.default_rng(seed)
    cands = random_list(api, rs, 4, plan.ntrials, 600)
    kw = dict(eps=0.5, min_pts=5, time_unit_s=1.0, dm_unit=1.0, snr_min=10.0, dm_min=10.0, width_max_s=0.1,
              coinc_window_s=0.05, coinc_beam_fraction=0.5)
    k1, k2, k3 = oracle_sift(orc, plan, cands, 4, **kw)
    got, stages = plan.sift(cands, 4, **kw)
    assert stages == [int(k1.sum()), int(k2.sum()), int(k3.sum())]
    assert keyset(got) == keyset(cands[k3])
    assert 0 < stages[2] <= stages[1] < stages[0] < cands.size
    # another plane scaling (time in 10 ms units, DM in steps of 0.25) and no anti-coincidence
    kw.update(time_unit_s=0.01, dm_unit=0.25, eps=3.0, min_pts=3, coinc_window_s=0.0)
    k1, k2, k3 = oracle_sift(orc, plan, cands, 4, **kw)
    got, stages = plan.sift(cands, 4, **kw)
    assert stages == [int(k1.sum()), int(k2.sum()), int(k3.sum())] and keyset(got) == keyset(cands[k3])


def test_pipeline_search_peaks_sift(cuda, api, orc, synth):
    """The whole chain on the GPU -- search, 3x3/11x11 peak filter, sifting -- against the oracle's sifting of the same peaks."""
    w = mini3(synth, 12)
    fb = synth.generate(w)
    plan, dmt, cands = run_gpu(cuda, api, w, fb[None], cand_capacity=1 << 20)
    peaks = plan.peak_filter((3, 11))
    kw = dict(eps=0.5, min_pts=2, snr_min=8.0, dm_min=10.0, width_max_s=0.1)
    k1, k2, k3 = oracle_sift(orc, plan, peaks, 1, **kw)
    got, stages = plan.sift(peaks, 1, **kw)
    assert keyset(got) == keyset(peaks[k3]) and stages == [int(k1.sum()), int(k2.sum()), int(k3.sum())]
    assert stages[0] > 0


def test_sift_edge_cases(cuda, api):
    w = Shape(500.0, -3.125, 64, 4096, [(0.0, 1.0, 30, 1)], [1, 2], 6.0)
    plan = make_plan(api, w)
    got, stages = plan.sift(np.zeros(0, dtype=api.CAND_DTYPE), 1)
    assert got.size == 0 and stages == [0, 0, 0]
    bad = np.zeros(1, dtype=api.CAND_DTYPE)
    bad["trial"] = 99
    with pytest.raises(api.SptError) as e:
        plan.sift(bad, 1)
    assert e.value.code == api.SPT_ERR_SHAPE
    with pytest.raises(api.SptError) as e:
        plan.sift(np.zeros(1, dtype=api.CAND_DTYPE), 1, eps=0.0)
    assert e.value.code == api.SPT_ERR_INVALID
