"""The comparison code of the parity tests is itself held to account here, without a GPU: fed the oracle's own candidate
list it must pass, and it must catch each kind of discrepancy rules D2 forbid."""
import numpy as np
import pytest

from helpers import SNR_TOL, check_candidates_dense

CAND_DTYPE = np.dtype([("beam", "<i4"), ("trial", "<i4"), ("t", "<i4"), ("width", "<i4"), ("snr", "<f4")])


@pytest.fixture(scope="module")
def case(orc, synth):
    w = synth.workload(1)
    fb = synth.generate(w)
    ranges = [(0.0, 1.0, 60, 1), (60.0, 2.0, 20, 2)]
    ref = orc.run_path(fb, w.fch1, w.foff, w.tsamp, ranges, w.widths, 4.5)
    recs, d0 = [], 0
    for rr in ref:
        sr = rr.search
        tr = np.repeat(np.arange(len(rr.nout)), sr.count) + d0
        c = np.zeros(sr.t.size, dtype=CAND_DTYPE)
        c["trial"], c["t"], c["width"], c["snr"] = tr, sr.t, sr.w, sr.snr
        recs.append(c)
        d0 += len(rr.nout)
    cands = np.concatenate(recs)
    assert cands.size > 500
    return w, ref, cands


def run(orc, case, cands):
    w, ref, _ = case
    return check_candidates_dense(orc, None, cands, ref, w.widths, 4.5)


def test_oracle_list_passes_in_any_order(orc, case):
    _, _, cands = case
    rs = np.random.default_rng(0)
    st = run(orc, case, cands[rs.permutation(cands.size)])
    assert st["matched"] == st["oracle"] == cands.size and st["near_threshold_only_gpu"] == 0


def test_missing_extra_duplicate_and_wrong_values_are_caught(orc, case):
    _, _, cands = case
    strong = int(np.argmax(cands["snr"]))
    with pytest.raises(AssertionError):                       # a strong candidate missing on the CUDA side
        run(orc, case, np.delete(cands, strong))
    dup = np.concatenate([cands, cands[strong: strong + 1]])
    with pytest.raises(AssertionError):                       # the same (trial, t) twice
        run(orc, case, dup)
    bad = cands.copy()
    bad["snr"][strong] += 10 * SNR_TOL
    with pytest.raises(AssertionError):                       # S/N off by more than the tolerance
        run(orc, case, bad)
    bad = cands.copy()
    bad["width"][strong] = 64 if bad["width"][strong] != 64 else 1
    with pytest.raises(AssertionError):                       # a width that is not a near tie
        run(orc, case, bad)
    extra = cands[strong: strong + 1].copy()
    taken = set(cands["t"][cands["trial"] == extra["trial"][0]].tolist())
    extra["t"] = next(t for t in range(2000) if t not in taken)
    with pytest.raises(AssertionError):                       # a candidate the oracle does not have, far from threshold
        run(orc, case, np.concatenate([cands, extra]))
    bad = cands.copy()
    bad["trial"][strong] = 80                                  # outside the plan
    with pytest.raises(AssertionError):
        run(orc, case, bad)
