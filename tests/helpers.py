"""Shared comparison code of the parity tests: CUDA path (through the C ABI) vs the oracle.

The rules are those of BASELINE.json north_star / DESIGN.md section 4: bit-exact delay tables, decimated series,
int32 DM transform and integer statistics; |dSNR| <= 1e-3; candidate lists identical except for events whose oracle
S/N lies within 1e-3 of the threshold (and widths that are tied within 1e-3).
"""
from __future__ import annotations

import numpy as np

SNR_TOL = 1e-3


def make_plan(api, w, nbeam=None, cand_capacity=1 << 22, options=None, ranges=None, widths=None, nsamp=None):
    return api.Plan(w.fch1, w.foff, w.nchan, w.tsamp, nsamp or w.nsamp, ranges or w.ranges, widths or w.widths,
                    max_beams=nbeam or w.nbeam, cand_capacity=cand_capacity, options=options)


def check_plan_against_oracle(orc, plan, w, ranges=None, stride=1):
    """Trial list, delay rows, nout and row offsets, bit-exact."""
    ranges = ranges or w.ranges
    dm, rg, dec, nout, off = plan.trial_table()
    d = 0
    expect_off = 0
    for ri, (lo, step, ndm, k) in enumerate(ranges):
        dly = orc.delay_table(w.fch1, w.foff, w.nchan, w.tsamp, lo, step, ndm, k)
        no = orc.nout(dly, plan.nsamp, k)
        for i in range(ndm):
            assert rg[d] == ri and dec[d] == k
            assert dm[d] == lo + float(i) * step
            assert nout[d] == no[i], (d, nout[d], no[i])
            assert off[d] == expect_off
            expect_off += (int(no[i]) + 31) // 32 * 32
            if i % stride == 0 or i == ndm - 1:
                assert np.array_equal(plan.delays(d), dly[i]), ("delay row", d)
            d += 1
    assert d == plan.ntrials and expect_off == plan.dmt_elems_per_beam


def rows_of(plan, dmt_host, beam=0):
    """Yield (trial, row view) of one beam of a host copy of the DM transform."""
    _, _, _, nout, off = plan.trial_table()
    base = dmt_host[beam]
    for d in range(plan.ntrials):
        yield d, base[off[d]: off[d] + nout[d]]


def check_dmt_against_oracle(plan, dmt_host, oracle_ranges, beam=0):
    """Every valid element of every row equals the oracle's, bit for bit."""
    _, _, _, nout, off = plan.trial_table()
    d = 0
    for rr in oracle_ranges:
        for i in range(len(rr.nout)):
            got = dmt_host[beam][off[d]: off[d] + nout[d]]
            exp = rr.dmt[rr.rowoff[i]: rr.rowoff[i + 1]]
            assert nout[d] == rr.nout[i]
            if not np.array_equal(got, exp):
                bad = np.flatnonzero(got != exp)
                raise AssertionError(f"DM transform mismatch: trial {d} (range row {i}), {bad.size} of {exp.size} samples, "
                                     f"first at t={bad[0]}: got {got[bad[0]]} expected {exp[bad[0]]}")
            d += 1
    assert d == plan.ntrials


def check_stats_against_oracle(plan, oracle_ranges, beam=0, nbeam=1):
    s, q = plan.trial_stats_all(nbeam)
    d = 0
    for rr in oracle_ranges:
        for i in range(len(rr.nout)):
            assert int(s[beam, d]) == int(rr.search.sum[i]), ("sum", d)
            assert int(q[beam, d]) == int(rr.search.sumsq[i]), ("sumsq", d)
            d += 1


def check_candidates_against_oracle(orc, plan, cands, oracle_ranges, widths, threshold, beam=0):
    """cands: structured array from spt_candidates_read (all beams).  Returns a dict of counts for the report."""
    mine = cands[cands["beam"] == beam]
    order = np.lexsort((mine["t"], mine["trial"]))
    mine = mine[order]
    # unique key (trial, t)
    key = mine["trial"].astype(np.int64) << 32 | mine["t"].astype(np.int64)
    assert np.unique(key).size == key.size, "duplicate (trial, t) in the candidate list"
    starts = np.searchsorted(mine["trial"], np.arange(plan.ntrials + 1))
    stats = dict(oracle=0, gpu=int(mine.size), matched=0, near_threshold_only_oracle=0, near_threshold_only_gpu=0,
                 width_near_ties=0, max_dsnr=0.0)
    d = 0
    for rr in oracle_ranges:
        sr = rr.search
        for i in range(len(rr.nout)):
            o_t = sr.t[sr.candoff[i]: sr.candoff[i + 1]]
            o_w = sr.w[sr.candoff[i]: sr.candoff[i + 1]]
            o_s = sr.snr[sr.candoff[i]: sr.candoff[i + 1]]
            g = mine[starts[d]: starts[d + 1]]
            stats["oracle"] += int(o_t.size)
            if o_t.size or g.size:
                row = rr.dmt[rr.rowoff[i]: rr.rowoff[i + 1]]
                common, io, ig = np.intersect1d(o_t, g["t"], assume_unique=True, return_indices=True)
                ds = np.abs(o_s[io] - g["snr"][ig].astype(np.float64))
                if ds.size:
                    stats["max_dsnr"] = max(stats["max_dsnr"], float(ds.max()))
                    assert ds.max() <= SNR_TOL, f"trial {d}: |dSNR| = {ds.max()}"
                wbad = np.flatnonzero(o_w[io] != g["width"][ig])
                for j in wbad:  # allowed only for a near tie between widths (rule D2 iv)
                    alt = orc.snr_at(row, int(g["width"][ig[j]]), int(common[j]))
                    assert abs(alt - o_s[io[j]]) <= SNR_TOL, f"trial {d} t {common[j]}: width {g['width'][ig[j]]} vs {o_w[io[j]]}"
                    stats["width_near_ties"] += 1
                stats["matched"] += int(common.size)
                only_o = np.setdiff1d(np.arange(o_t.size), io)
                for j in only_o:
                    assert abs(o_s[j] - threshold) <= SNR_TOL, f"trial {d} t {o_t[j]}: oracle-only candidate snr {o_s[j]}"
                    stats["near_threshold_only_oracle"] += 1
                only_g = np.setdiff1d(np.arange(g.size), ig)
                if only_g.size:
                    best, _ = orc.best_width(row, widths)
                    for j in only_g:
                        b = best[int(g["t"][j])]
                        assert abs(b - threshold) <= SNR_TOL, f"trial {d} t {g['t'][j]}: GPU-only candidate, oracle best {b}"
                        stats["near_threshold_only_gpu"] += 1
            d += 1
    return stats


def check_candidates_dense(orc, plan, cands, oracle_ranges, widths, threshold, beam=None):
    """Rules D2 at any volume: instead of sorting 1e8 records, the CUDA path's records of one DM
    range are scattered into dense rows laid out like the oracle's packed DM transform and read back at the oracle's
    (sorted) candidate positions.  cands: the records of ONE beam (beam=None: all of them are)."""
    mine = cands if beam is None else cands[cands["beam"] == beam]
    stats = dict(oracle=0, gpu=int(mine.size), matched=0, near_threshold_only_oracle=0, near_threshold_only_gpu=0,
                 width_near_ties=0, max_dsnr=0.0)
    d0 = 0
    seen = 0
    for rr in oracle_ranges:
        ndm = len(rr.nout)
        sr = rr.search
        g = mine[(mine["trial"] >= d0) & (mine["trial"] < d0 + ndm)]
        seen += int(g.size)
        nelem = int(rr.rowoff[-1])
        tl = g["trial"].astype(np.int64) - d0
        assert np.all((g["t"] >= 0) & (g["t"] < rr.nout[tl])), "candidate outside its row"
        dense_s = np.full(nelem, np.nan, dtype=np.float32)
        dense_w = np.zeros(nelem, dtype=np.int16)
        gkey = rr.rowoff[tl] + g["t"]
        dense_s[gkey] = g["snr"]
        dense_w[gkey] = g["width"]
        assert int(np.count_nonzero(~np.isnan(dense_s))) == g.size, "duplicate (trial, t) in the candidate list"
        del gkey, tl
        okey = sr.t.astype(np.int64) + np.repeat(rr.rowoff[:-1], sr.count)
        stats["oracle"] += int(okey.size)
        gs, gw = dense_s[okey], dense_w[okey]
        have = ~np.isnan(gs)
        # (ii) an event only the oracle has must sit within the tolerance of the threshold
        only_o = np.flatnonzero(~have)
        assert np.all(np.abs(sr.snr[only_o] - threshold) <= SNR_TOL), "oracle-only candidate away from the threshold"
        stats["near_threshold_only_oracle"] += int(only_o.size)
        # (iii) matched events
        ds = np.abs(sr.snr[have] - gs[have].astype(np.float64))
        if ds.size:
            stats["max_dsnr"] = max(stats["max_dsnr"], float(ds.max()))
            assert ds.max() <= SNR_TOL, f"range of trial {d0}: |dSNR| = {ds.max()}"
        stats["matched"] += int(ds.size)
        # (iv) widths, up to near ties
        for j in np.flatnonzero(have & (gw != sr.w)):
            i = int(np.searchsorted(rr.rowoff, okey[j], side="right")) - 1
            row = rr.dmt[rr.rowoff[i]: rr.rowoff[i + 1]]
            alt = orc.snr_at(row, int(gw[j]), int(sr.t[j]))
            assert abs(alt - sr.snr[j]) <= SNR_TOL, f"trial {d0 + i} t {sr.t[j]}: width {gw[j]} vs {sr.w[j]}"
            stats["width_near_ties"] += 1
        # (ii) again: what is left after taking the oracle's positions out exists on the CUDA side only
        dense_s[okey] = np.nan
        best_cache = {}
        for key in np.flatnonzero(~np.isnan(dense_s)):
            i = int(np.searchsorted(rr.rowoff, key, side="right")) - 1
            if i not in best_cache:
                best_cache[i] = orc.best_width(rr.dmt[rr.rowoff[i]: rr.rowoff[i + 1]], widths)[0]
            b = best_cache[i][int(key - rr.rowoff[i])]
            assert abs(b - threshold) <= SNR_TOL, f"trial {d0 + i} t {key - rr.rowoff[i]}: GPU-only candidate, oracle best {b}"
            stats["near_threshold_only_gpu"] += 1
        del dense_s, dense_w, okey, gs, gw
        d0 += ndm
    assert seen == mine.size, "candidate with a trial index outside the plan"
    return stats


def check_segment_against_oracle(orc, plan, dmt_beam, orows, trials, widths, threshold, nnew, cands, s_row, q_row, sentinel=None):
    """One pushed stream segment of one beam (reading F), for the trials named.  orows[d] = the ORACLE's dedispersed row d of
    the oracle's stream buffer.  Checked: the window the search reads (the last nnew/k + wmax - 1 outputs of the row) equals
    the oracle's, bit for bit; with `sentinel`, nothing before the window was written; the window's exact statistics; the
    candidates of the segment's start positions under rules D2 (identical except within SNR_TOL of the threshold)."""
    _, _, dec, nout, off = plan.trial_table()
    got = {}
    for c in cands:
        got.setdefault(int(c["trial"]), []).append((int(c["t"]), int(c["width"]), float(c["snr"])))
    nchecked = 0
    for d in trials:
        n, k = int(nout[d]), int(dec[d])
        row = orows[d]
        assert row.size == n
        win = min(n, nnew // k + max(widths) - 1)
        mine = dmt_beam[off[d]: off[d] + n]
        assert np.array_equal(mine[n - win:], row[n - win:]), ("window of trial", d)
        if sentinel is not None:
            assert np.all(mine[: n - win] == sentinel), ("outputs before the window of trial", d)
        sx, sxx, t, bw, snr = orc.search_segment(row, widths, threshold, nnew // k)
        assert (int(s_row[d]), int(q_row[d])) == (sx, sxx), ("statistics of trial", d)
        g = sorted(got.get(d, []))
        exp = sorted(zip(t.tolist(), bw.tolist(), snr.tolist()))
        near = [x for x in exp if abs(x[2] - threshold) <= SNR_TOL]
        assert abs(len(g) - len(exp)) <= len(near), (d, len(g), len(exp))
        ge = {x[0]: x for x in g}
        for (tt, ww, ss) in exp:
            if tt in ge:
                assert ge[tt][1] == ww and abs(ge[tt][2] - ss) <= SNR_TOL, (d, tt)
            else:
                assert abs(ss - threshold) <= SNR_TOL
        et = {x[0] for x in exp}
        for (tt, ww, ss) in g:                                    # an event only the CUDA path has sits at the threshold too
            assert tt in et or abs(ss - threshold) <= 2 * SNR_TOL, (d, tt, ss)
        lo = n - win
        assert all(lo <= x[0] < lo + nnew // k for x in g)        # only this segment's start positions
        nchecked += len(exp)
    return nchecked
