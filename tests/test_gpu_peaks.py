"""Peak filtering (reading E) on the GPU against the oracle: (1) as a pure function of a candidate list the
CUDA filter must give exactly what the oracle's filter gives on the same list; (2) end to end, the survivors of the CUDA
path equal the survivors of the oracle's path except where two competing candidates are tied within 1e-3 in S/N."""
import numpy as np
import pytest

from helpers import SNR_TOL, make_plan
from test_gpu_parity import Shape, mini3, oracle_path, run_gpu

pytestmark = pytest.mark.gpu


def as_set(c):
    return {(int(r["beam"]), int(r["trial"]), int(r["t"]), int(r["width"]), float(r["snr"])) for r in c}


def oracle_filter_of_list(orc, plan, cands, windows):
    _, rg, _, _, _ = plan.trial_table()
    keep = orc.peak_filter(cands["beam"], cands["trial"], cands["t"], cands["snr"].astype(np.float64), rg, windows)
    return cands[keep]


@pytest.mark.parametrize("lookup", [0, 1, 2])
@pytest.mark.parametrize("windows", [(3,), (11,), (3, 11), (5, 3, 7)])
def test_filter_is_exact_on_the_same_list(cuda, api, orc, synth, windows, lookup):
    """lookup: how the filter finds a neighbour's S/N -- chosen by the list's density, hash table, dense plane."""
    w = mini3(synth, 12)
    fb = synth.generate(w)
    plan, dmt, cands = run_gpu(cuda, api, w, fb[None], cand_capacity=1 << 20)
    assert cands.size > 1000
    plan.set_option("peaks_lookup", lookup)
    peaks = plan.peak_filter(windows)
    expect = oracle_filter_of_list(orc, plan, cands, windows)
    assert 0 < peaks.size < cands.size
    assert as_set(peaks) == as_set(expect)
    assert as_set(plan.candidates_read()) == as_set(cands)            # the candidate list is left untouched
    assert as_set(plan.peak_filter(windows)) == as_set(expect)        # the lookup plane was cleared: same answer again


def test_quantised_ties_and_multibeam(cuda, api, orc):
    """Small integers everywhere: many exact S/N ties between neighbours, two beams, several ranges, row ends."""
    w = Shape(420.0, -1.0, 16, 3000, [(3.0, 0.7, 30, 1), (60.0, 1.1, 20, 2)], [1, 2, 4], 1.0, nbeam=2)
    rs = np.random.default_rng(3)
    fb = rs.integers(0, 3, size=(2, w.nchan, w.nsamp), dtype=np.uint8)
    plan, dmt, cands = run_gpu(cuda, api, w, fb, cand_capacity=1 << 22)
    assert cands.size > 10000
    s = np.sort(cands["snr"])
    assert np.count_nonzero(np.diff(s) == 0) > cands.size // 2        # the premise: exact ties are common
    for windows in ((3,), (3, 11)):
        expect = as_set(oracle_filter_of_list(orc, plan, cands, windows))
        for lookup in (0, 1, 2, 3, 0):          # hash table, one plane for both beams, a one-beam plane passed over twice
            plan.set_option("peaks_lookup", lookup)
            assert as_set(plan.peak_filter(windows)) == expect, lookup


def test_end_to_end_against_the_oracle_path(cuda, api, orc, synth):
    w = mini3(synth, 12)
    fb = synth.generate(w)
    ref = oracle_path(orc, w, fb)
    plan, dmt, cands = run_gpu(cuda, api, w, fb[None], cand_capacity=1 << 20)
    peaks = plan.peak_filter((3, 11))
    _, rg, _, _, _ = plan.trial_table()
    ot, otr, osn = [], [], []
    d0 = 0
    for rr in ref:
        sr = rr.search
        for i in range(len(rr.nout)):
            sl = slice(sr.candoff[i], sr.candoff[i + 1])
            ot.append(sr.t[sl]); osn.append(sr.snr[sl]); otr.append(np.full(sr.t[sl].size, d0 + i, dtype=np.int32))
        d0 += len(rr.nout)
    ot, otr, osn = np.concatenate(ot), np.concatenate(otr), np.concatenate(osn)
    keep = orc.peak_filter(np.zeros(ot.size, dtype=np.int32), otr, ot, osn, rg, (3, 11))
    exp = {(int(a), int(b)) for a, b in zip(otr[keep], ot[keep])}
    got = {(int(r["trial"]), int(r["t"])) for r in peaks}
    assert len(exp) * 5 < ot.size                                     # the filter removes most of the list
    # cells where the two disagree must sit next to a competitor tied within the tolerance
    snr_at = {(int(a), int(b)): float(s) for a, b, s in zip(otr, ot, osn)}
    for (d, t) in exp ^ got:
        s = snr_at.get((d, t))
        assert s is not None
        near = [abs(snr_at[(dd, tt)] - s) for dd in range(d - 5, d + 6) for tt in range(t - 5, t + 6)
                if (dd, tt) != (d, t) and (dd, tt) in snr_at]
        assert near and min(near) <= SNR_TOL, (d, t, s)
    assert len(exp ^ got) <= max(2, len(exp) // 100)


def test_empty_and_error_paths(cuda, api, synth):
    w = synth.workload(1)
    fb = synth.generate(w)
    plan = make_plan(api, w, cand_capacity=4)
    with pytest.raises(api.SptError) as e:
        plan.peak_filter()                                             # nothing searched yet
    assert e.value.code == api.SPT_ERR_STATE
    plan.search_host(fb[None], 2.0)                                    # overflows the 4-record list
    with pytest.raises(api.SptError) as e:
        plan.peak_filter()
    assert e.value.code == api.SPT_ERR_SHAPE
    plan.search_host(fb[None], 1000.0)                                 # no candidates at all
    assert plan.peak_filter().size == 0
    with pytest.raises(api.SptError) as e:
        plan.peak_filter((4,))
    assert e.value.code == api.SPT_ERR_INVALID


def test_dense_plane_at_volume(cuda, api, orc, synth):
    """The dense-plane lookups at the density they exist for (PAPER.md:96 on unmitigated RFI): config 5's beam -- zero-DM
    spikes and persistent narrowband RFI put a sizeable fraction of all cells above threshold -- searched over 48 trials of
    two DM ranges across the whole 2^18-sample row, millions of records.  The plane over all beams (lookup 2), the
    one-beam plane (3) and the hash table (1) must each keep exactly what the oracle's filter keeps of the same list."""
    w5 = synth.workload(5)
    fb = synth.generate(w5)
    w = Shape(w5.fch1, w5.foff, w5.nchan, w5.nsamp, [(0.0, 0.2, 32, 1), (500.0, 0.5, 16, 2)], w5.widths, w5.threshold)
    plan = make_plan(api, w, cand_capacity=1 << 24)
    d_dmt = plan.search(cuda.from_numpy(fb[None]).cuda(), w.threshold)
    total, ovf = plan.candidates_count()
    assert not ovf and total > 1_000_000, total
    cands = plan.candidates_read()
    del d_dmt
    expect = as_set(oracle_filter_of_list(orc, plan, cands, (3, 11)))
    assert 0 < len(expect) < cands.size // 10
    for lookup in (2, 3, 1):
        plan.set_option("peaks_lookup", lookup)
        assert as_set(plan.peak_filter((3, 11))) == expect, lookup
