"""Pins of the oracle's peak filter (reading E of DESIGN.md; sliding 3x3 and 11x11 windows in the DM-time
plane keep the highest-S/N peak).  Hand-made cases with known answers, invariants, and an independent brute-force
restatement in Python on random small sets."""
import numpy as np
import pytest


def brute_force(beam, trial, t, snr, rot, windows):
    """Independent statement: all pairs, no map.  alive[i] unless some live j != i in the window is stronger."""
    n = len(beam)
    alive = [True] * n
    for w in windows:
        h = (w - 1) // 2
        nxt = list(alive)
        for i in range(n):
            if not alive[i]:
                continue
            for j in range(n):
                if j == i or not alive[j] or beam[j] != beam[i] or rot[trial[j]] != rot[trial[i]]:
                    continue
                if abs(trial[j] - trial[i]) > h or abs(t[j] - t[i]) > h:
                    continue
                if snr[j] > snr[i] or (snr[j] == snr[i] and (trial[j], t[j]) < (trial[i], t[i])):
                    nxt[i] = False
                    break
        alive = nxt
    return np.array(alive)


ROT = np.zeros(64, dtype=np.int32)


def run(orc, cands, windows=(3,), rot=ROT):
    b, d, t, s = (np.array(x) for x in zip(*cands))
    return orc.peak_filter(b, d, t, s.astype(np.float64), rot, windows).tolist()


def test_hand_made_cases(orc):
    assert run(orc, [(0, 5, 100, 7.0)]) == [True]                                         # alone
    assert run(orc, [(0, 5, 100, 7.0), (0, 5, 101, 9.0)]) == [False, True]                # neighbour in time
    assert run(orc, [(0, 5, 100, 7.0), (0, 6, 101, 9.0)]) == [False, True]                # diagonal neighbour
    assert run(orc, [(0, 5, 100, 7.0), (0, 5, 102, 9.0)]) == [True, True]                 # outside a 3x3 window
    assert run(orc, [(0, 5, 100, 7.0), (0, 5, 102, 9.0)], (5,)) == [False, True]          # inside a 5x5 window
    assert run(orc, [(0, 5, 100, 7.0), (0, 10, 100, 9.0)], (11,)) == [False, True]        # edge of an 11x11 window
    assert run(orc, [(0, 5, 100, 7.0), (0, 11, 100, 9.0)], (11,)) == [True, True]         # just outside it
    assert run(orc, [(0, 5, 100, 8.0), (0, 5, 101, 8.0)]) == [True, False]                # exact tie: smaller t survives
    assert run(orc, [(0, 6, 100, 8.0), (0, 5, 101, 8.0)]) == [False, True]                # exact tie: smaller trial survives
    assert run(orc, [(0, 5, 100, 7.0), (1, 5, 101, 9.0)]) == [True, True]                 # other beam: no interaction


def test_ranges_do_not_interact(orc):
    rot = np.array([0] * 10 + [1] * 10, dtype=np.int32)                                    # trials 0-9 range 0, 10-19 range 1
    assert run(orc, [(0, 9, 50, 7.0), (0, 10, 50, 9.0)], (3,), rot) == [True, True]
    assert run(orc, [(0, 8, 50, 7.0), (0, 9, 50, 9.0)], (3,), rot) == [False, True]


def test_stencils_are_applied_in_sequence(orc):
    """A < B < C on a line, B next to A, C five cells from B and six from A.  3x3: B removes A.  11x11 among the
    survivors: C removes B.  A single 11x11 pass over all three would also remove A through B; in sequence A is
    already gone -- and a candidate that died in the first pass no longer shields or kills anyone in the second."""
    c = [(0, 5, 100, 7.0), (0, 5, 101, 8.0), (0, 5, 106, 9.0)]
    assert run(orc, c, (3,)) == [False, True, True]
    assert run(orc, c, (3, 11)) == [False, False, True]
    # D strongest but killed by nobody; E only beaten by a candidate that the first pass removed
    c = [(0, 5, 100, 9.0), (0, 5, 101, 8.0), (0, 5, 104, 7.5)]
    assert run(orc, c, (3,)) == [True, False, True]
    assert run(orc, c, (3, 11)) == [True, False, False]      # E is within 11x11 of the 9.0 survivor


@pytest.mark.parametrize("seed", range(6))
def test_matches_brute_force_on_random_sets(orc, seed):
    rs = np.random.default_rng(seed)
    rot = np.array([0] * 12 + [1] * 8, dtype=np.int32)
    n = 300
    cells = rs.choice(2 * 20 * 60, size=n, replace=False)                                  # unique (beam, trial, t)
    beam, trial, t = cells // (20 * 60), (cells // 60) % 20, cells % 60
    snr = np.round(rs.uniform(6, 12, size=n), 1)                                           # many exact ties
    for windows in ((3,), (11,), (3, 11), (5, 3)):
        got = orc.peak_filter(beam, trial, t, snr, rot, windows)
        assert np.array_equal(got, brute_force(beam, trial, t, snr, rot, windows)), windows


def test_invariants(orc):
    rs = np.random.default_rng(42)
    n = 400
    cells = rs.choice(30 * 200, size=n, replace=False)
    beam, trial, t = np.zeros(n, dtype=np.int32), cells // 200, cells % 200
    snr = rs.uniform(6, 30, size=n)
    rot = np.zeros(30, dtype=np.int32)
    k3 = orc.peak_filter(beam, trial, t, snr, rot, (3,))
    k311 = orc.peak_filter(beam, trial, t, snr, rot, (3, 11))
    assert k3[np.argmax(snr)] and k311[np.argmax(snr)]                                     # the global maximum always survives
    assert not np.any(k311 & ~k3)                                                          # later stencils only remove
    # idempotent: filtering the survivors again removes nothing
    again = orc.peak_filter(beam[k311], trial[k311], t[k311], snr[k311], rot, (3, 11))
    assert again.all()
    # no two survivors of a stencil share a window
    s = np.flatnonzero(k311)
    for i in s:
        near = s[(np.abs(trial[s] - trial[i]) <= 5) & (np.abs(t[s] - t[i]) <= 5)]
        assert near.size == 1
    with pytest.raises(RuntimeError):
        orc.peak_filter(beam, trial, t, snr, rot, (4,))                                    # even window
