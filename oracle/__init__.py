"""oracle -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

ctypes access to oracle.cpp, the plain CPU statement of the SPOTLIGHT search hot path
(arxiv/paper_2606_27262).  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package.  It imports nothing from
paper_2606_27262_b200 and the product imports nothing from here.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass
from typing import List, Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.cpp")
_SO = os.path.join(_HERE, "liboracle.so")

CXXFLAGS = ["-O2", "-fopenmp", "-ffp-contract=off", "-std=c++17", "-shared", "-fPIC"]
# ORACLE_SANITIZE=1: the same source built with AddressSanitizer + UndefinedBehaviorSanitizer into its own library, for
#   ORACLE_SANITIZE=1 LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 python -m pytest tests -m "not gpu"
# (the result of the last such run is recorded in DESIGN.md section 3)
if os.environ.get("ORACLE_SANITIZE") == "1":
    CXXFLAGS = CXXFLAGS[:1] + ["-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined"] + CXXFLAGS[1:]
    _SO = os.path.join(_HERE, "liboracle_san.so")


def build(force: bool = False) -> str:
    """g++ oracle.cpp -> liboracle.so (rebuilt when the source is newer)."""
    if force or (not os.path.exists(_SO)) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.run(["g++", *CXXFLAGS, "-o", _SO, _SRC], check=True)
    return _SO


_lib = None
_i32p = ctypes.POINTER(ctypes.c_int32)


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_SO)
        vp, i32, i64, f64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_double
        L.orc_num_threads.restype = ctypes.c_int
        L.orc_delay_table.argtypes = [f64, f64, i32, f64, f64, f64, i32, i32, vp]
        L.orc_nout.argtypes = [vp, i32, i32, i64, i32, vp]
        L.orc_decimate.argtypes = [vp, i32, i64, i32, vp]
        L.orc_dedisperse_u16.argtypes = [vp, i32, i64, vp, i32, vp, vp, vp]
        L.orc_dedisperse_u8.argtypes = [vp, i32, i64, vp, i32, vp, vp, vp]
        L.orc_dedisperse_point_u8.argtypes = [vp, i32, i64, vp, i32, i64, vp]
        L.orc_stats.argtypes = [vp, i64, vp, vp]
        L.orc_mean_sigma.argtypes = [i64, i64, ctypes.c_uint64, vp, vp]
        L.orc_boxcar_snr.argtypes = [vp, i64, i32, vp]
        L.orc_best_width.argtypes = [vp, i64, vp, i32, vp, vp]
        L.orc_snr_at.argtypes = [vp, i64, i32, i64, vp]
        L.orc_search_plane.argtypes = [vp, i32, vp, vp, vp, i32, f64, vp, vp, vp, vp, vp, vp, vp]
        L.orc_cutout.argtypes = [vp, i32, i64, f64, f64, f64, f64, f64, i32, i64, i32, i32, i32, vp, vp]
        L.orc_cutout.restype = ctypes.c_int
        L.orc_delta_dm.argtypes = [f64, f64, f64, f64, f64]
        L.orc_delta_dm.restype = f64
        L.orc_peak_filter.argtypes = [i64, vp, vp, vp, vp, vp, i32, i32, vp]
        L.orc_peak_filter.restype = ctypes.c_int
        for name in ("orc_delay_table", "orc_nout", "orc_decimate", "orc_dedisperse_u16", "orc_dedisperse_u8",
                     "orc_dedisperse_point_u8", "orc_stats", "orc_mean_sigma", "orc_boxcar_snr", "orc_best_width",
                     "orc_snr_at", "orc_search_plane"):
            getattr(L, name).restype = ctypes.c_int
        _lib = L
    return _lib


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data


def _check(rc: int, what: str):
    if rc != 0:
        raise RuntimeError(f"oracle: {what} failed (rc={rc})")


def num_threads() -> int:
    return int(lib().orc_num_threads())


# ---- A. plan -----------------------------------------------------------------------------------
def delay_table(fch1: float, foff: float, nchan: int, tsamp: float, dm_lo: float, dm_step: float, ndm: int,
                decim: int) -> np.ndarray:
    out = np.empty((ndm, nchan), dtype=np.int32)
    _check(lib().orc_delay_table(fch1, foff, nchan, tsamp, dm_lo, dm_step, ndm, decim, _ptr(out)), "delay_table")
    return out


def nout(delay: np.ndarray, nsamp: int, decim: int) -> np.ndarray:
    delay = np.ascontiguousarray(delay, dtype=np.int32)
    out = np.empty(delay.shape[0], dtype=np.int32)
    _check(lib().orc_nout(_ptr(delay), delay.shape[0], delay.shape[1], nsamp, decim, _ptr(out)), "nout")
    return out


# ---- B. decimation and dedispersion -----------------------------------------------------------------
def decimate(x: np.ndarray, k: int) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.uint8)
    nchan, nsamp = x.shape
    y = np.empty((nchan, nsamp // k), dtype=np.uint16)
    _check(lib().orc_decimate(_ptr(x), nchan, nsamp, k, _ptr(y)), "decimate")
    return y


def dedisperse(y: np.ndarray, delay: np.ndarray, nout_: np.ndarray) -> Tuple[np.ndarray, np.ndarray]:
    """DM transform of one range.  y is uint8 (k = 1) or uint16 (decimated).  Returns (packed rows, row offsets)."""
    delay = np.ascontiguousarray(delay, dtype=np.int32)
    nout_ = np.ascontiguousarray(nout_, dtype=np.int32)
    y = np.ascontiguousarray(y)
    nchan, nk = y.shape
    ndm = delay.shape[0]
    rowoff = np.zeros(ndm + 1, dtype=np.int64)
    np.cumsum(nout_.astype(np.int64), out=rowoff[1:])
    out = np.empty(int(rowoff[-1]), dtype=np.int32)
    if y.dtype == np.uint8:
        rc = lib().orc_dedisperse_u8(_ptr(y), nchan, nk, _ptr(delay), ndm, _ptr(nout_), _ptr(rowoff), _ptr(out))
    elif y.dtype == np.uint16:
        rc = lib().orc_dedisperse_u16(_ptr(y), nchan, nk, _ptr(delay), ndm, _ptr(nout_), _ptr(rowoff), _ptr(out))
    else:
        raise TypeError("dedisperse wants uint8 or uint16 input")
    _check(rc, "dedisperse")
    return out, rowoff


def dedisperse_point(x: np.ndarray, delay_row: np.ndarray, k: int, t: int) -> int:
    """One output sample of one trial straight from the raw uint8 filterbank (decimation folded in)."""
    x = np.ascontiguousarray(x, dtype=np.uint8)
    delay_row = np.ascontiguousarray(delay_row, dtype=np.int32)
    out = ctypes.c_int32(0)
    _check(lib().orc_dedisperse_point_u8(_ptr(x), x.shape[0], x.shape[1], _ptr(delay_row), k, t,
                                         ctypes.addressof(out)), "dedisperse_point")
    return int(out.value)


# ---- C. statistics, boxcar, best width ------------------------------------------------------------
def stats(x: np.ndarray) -> Tuple[int, int]:
    x = np.ascontiguousarray(x, dtype=np.int32)
    s, q = ctypes.c_int64(0), ctypes.c_uint64(0)
    _check(lib().orc_stats(_ptr(x), x.size, ctypes.addressof(s), ctypes.addressof(q)), "stats")
    return int(s.value), int(q.value)


def mean_sigma(n: int, s: int, q: int) -> Tuple[float, float]:
    mu, sg = ctypes.c_double(0), ctypes.c_double(0)
    _check(lib().orc_mean_sigma(n, s, q, ctypes.addressof(mu), ctypes.addressof(sg)), "mean_sigma")
    return float(mu.value), float(sg.value)


def boxcar_snr(x: np.ndarray, w: int) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.int32)
    out = np.zeros(max(0, x.size - w + 1), dtype=np.float64)
    _check(lib().orc_boxcar_snr(_ptr(x), x.size, w, _ptr(out)), "boxcar_snr")
    return out


def best_width(x: np.ndarray, widths: Sequence[int]) -> Tuple[np.ndarray, np.ndarray]:
    x = np.ascontiguousarray(x, dtype=np.int32)
    wa = np.asarray(widths, dtype=np.int32)
    nb = max(0, x.size - int(wa[0]) + 1)
    b = np.zeros(nb, dtype=np.float64)
    bw = np.zeros(nb, dtype=np.int32)
    _check(lib().orc_best_width(_ptr(x), x.size, _ptr(wa), wa.size, _ptr(b), _ptr(bw)), "best_width")
    return b, bw


def snr_at(x: np.ndarray, w: int, t: int) -> float:
    x = np.ascontiguousarray(x, dtype=np.int32)
    out = ctypes.c_double(0)
    _check(lib().orc_snr_at(_ptr(x), x.size, w, t, ctypes.addressof(out)), "snr_at")
    return float(out.value)


@dataclass
class PlaneSearch:
    sum: np.ndarray       # int64  [ntrial]
    sumsq: np.ndarray     # uint64 [ntrial]
    count: np.ndarray     # int64  [ntrial]
    candoff: np.ndarray   # int64  [ntrial+1]
    t: np.ndarray         # int32  [ncand]  (increasing within a trial)
    w: np.ndarray         # int32  [ncand]
    snr: np.ndarray       # float64 [ncand]


def search_plane(dmt: np.ndarray, rowoff: np.ndarray, nout_: np.ndarray, widths: Sequence[int],
                 threshold: float, want_candidates: bool = True) -> PlaneSearch:
    dmt = np.ascontiguousarray(dmt, dtype=np.int32)
    rowoff = np.ascontiguousarray(rowoff, dtype=np.int64)
    nout_ = np.ascontiguousarray(nout_, dtype=np.int32)
    wa = np.asarray(widths, dtype=np.int32)
    nt = nout_.size
    s = np.zeros(nt, dtype=np.int64)
    q = np.zeros(nt, dtype=np.uint64)
    cnt = np.zeros(nt, dtype=np.int64)
    _check(lib().orc_search_plane(_ptr(dmt), nt, _ptr(rowoff), _ptr(nout_), _ptr(wa), wa.size, threshold,
                                  _ptr(s), _ptr(q), _ptr(cnt), None, None, None, None), "search_plane(count)")
    candoff = np.zeros(nt + 1, dtype=np.int64)
    np.cumsum(cnt, out=candoff[1:])
    n = int(candoff[-1])
    ct = np.zeros(n, dtype=np.int32)
    cw = np.zeros(n, dtype=np.int32)
    cs = np.zeros(n, dtype=np.float64)
    if want_candidates and n > 0:
        _check(lib().orc_search_plane(_ptr(dmt), nt, _ptr(rowoff), _ptr(nout_), _ptr(wa), wa.size, threshold,
                                      _ptr(s), _ptr(q), _ptr(cnt), _ptr(candoff), _ptr(ct), _ptr(cw), _ptr(cs)),
               "search_plane(fill)")
    return PlaneSearch(s, q, cnt, candoff, ct, cw, cs)


# ---- F. corner turn and overlap-save -- plain definitions ---------------------------
def corner_turn(x_time_major: np.ndarray, flip: bool = False) -> np.ndarray:
    """[nsamp][nchan] (time-major block) -> [nchan][nsamp]; flip = the block has the lowest frequency first."""
    y = np.ascontiguousarray(np.asarray(x_time_major, dtype=np.uint8).T)
    return np.ascontiguousarray(y[::-1]) if flip else y


def corner_turn_spliced(block: np.ndarray, flip: bool = False) -> List[np.ndarray]:
    """A time-spliced block [nsamp][nbeam][nchan] (the beams of one host interleaved sample by sample) ->
    per beam the channel-major [nchan][nsamp] array: beam b's samples are block[:, b, :]."""
    block = np.asarray(block, dtype=np.uint8)
    return [corner_turn(block[:, b, :], flip) for b in range(block.shape[1])]


def overlap_save_buffers(blocks_time_major: Sequence[np.ndarray], nsamp: int, flip: bool = False) -> List[np.ndarray]:
    """The working buffer ([nchan][nsamp]) after each push of a stream that starts on a history of zeros: the last
    nsamp samples of zeros ++ block 0 ++ block 1 ++ ... (every trial of a dedispersion of it has its full sweep when
    nsamp - len(block) >= the longest sweep)."""
    nchan = blocks_time_major[0].shape[1]
    stream = np.zeros((nchan, nsamp), dtype=np.uint8)
    out = []
    for blk in blocks_time_major:
        stream = np.concatenate([stream, corner_turn(blk, flip)], axis=1)
        out.append(np.ascontiguousarray(stream[:, -nsamp:]))
    return out


def search_segment(row: np.ndarray, widths: Sequence[int], threshold: float, nnew_k: int):
    """Search of one pushed segment of one trial (reading F): the window is the last nnew_k + wmax - 1 samples of the row,
    statistics and S/N are the window's (readings C1-C5 applied to it), and only the start positions in its first nnew_k
    samples are reported.  Returns (sum, sumsq, t, width, snr) with t an index into the row."""
    row = np.ascontiguousarray(row, dtype=np.int32)
    L = int(nnew_k) + int(max(widths)) - 1
    lo = max(0, row.size - L)
    win = row[lo:]
    sx, sxx = stats(win)
    best, bw = best_width(win, widths)
    tt = np.flatnonzero(best[: int(nnew_k)] >= threshold)
    return sx, sxx, (tt + lo).astype(np.int32), bw[tt], best[tt]


# ---- E. peak filtering --------------------------------------------------------------------
def peak_filter(beam: np.ndarray, trial: np.ndarray, t: np.ndarray, snr: np.ndarray, range_of_trial: np.ndarray,
                windows: Sequence[int] = (3, 11)) -> np.ndarray:
    """Boolean mask of the candidates that survive the stencils applied one after the other."""
    beam = np.ascontiguousarray(beam, dtype=np.int32)
    trial = np.ascontiguousarray(trial, dtype=np.int32)
    t = np.ascontiguousarray(t, dtype=np.int32)
    snr = np.ascontiguousarray(snr, dtype=np.float64)
    rot = np.ascontiguousarray(range_of_trial, dtype=np.int32)
    alive = np.ones(beam.size, dtype=np.uint8)
    for w in windows:
        _check(lib().orc_peak_filter(beam.size, _ptr(beam), _ptr(trial), _ptr(t), _ptr(snr), _ptr(rot), rot.size, int(w),
                                     _ptr(alive)), "peak_filter")
    return alive.astype(bool)


# ---- G. candidate sifting ---------------------------------------------------------------
def dbscan(x: np.ndarray, y: np.ndarray, eps: float, min_pts: int) -> Tuple[np.ndarray, np.ndarray]:
    """DBSCAN (Ester et al. 1996) written out: a point is a CORE point when at least min_pts points (itself included)
    lie within eps of it; core points within eps of each other are in the same cluster (transitively); a non-core point
    within eps of a core point is a BORDER point.  Returns (is_core, core_label) where core_label[i] for a core point is
    the smallest index among the core points of its cluster (-1 for non-core points)."""
    x = np.asarray(x, dtype=np.float64)
    y = np.asarray(y, dtype=np.float64)
    n = x.size
    dx = x[:, None] - x[None, :]
    dy = y[:, None] - y[None, :]
    near = (dx * dx + dy * dy) <= eps * eps
    core = near.sum(axis=1) >= min_pts
    label = np.full(n, -1, dtype=np.int64)
    for i in range(n):                                   # flood fill over core points, smallest index first
        if not core[i] or label[i] >= 0:
            continue
        label[i] = i
        stack = [i]
        while stack:
            a = stack.pop()
            for b in np.flatnonzero(near[a] & core & (label < 0)):
                label[b] = i
                stack.append(int(b))
    return core, label


def sift(beam, trial, t, width, snr, dm_of_trial, decim_of_trial, tsamp: float, nbeam: int, eps: float = 0.5,
         min_pts: int = 5, time_unit_s: float = 1.0, dm_unit: float = 1.0, snr_min: float = 10.0, dm_min: float = 10.0,
         width_max_s: float = 0.1, coinc_window_s: float = 0.0, coinc_beam_fraction: float = 0.5):
    """The candidate optimisation of PAPER.md:104/112 (reading G), stage by stage; returns the boolean masks after
    (clustering, cuts, anti-coincidence) over the input list.
      1 per beam: DBSCAN in the plane (arrival time / time_unit_s, DM / dm_unit); clusters need a core point (>= min_pts
        points within eps); a border point joins the cluster of its strongest core neighbour (largest S/N, then smallest
        (trial, t)); out of each cluster the member with the highest S/N (then smallest (trial, t)) is kept; points in no
        cluster are rejected.
      2 cuts: rejected when S/N < snr_min, DM < dm_min or width (seconds) > width_max_s.
      3 anti-coincidence (coinc_window_s > 0): a survivor is rejected when survivors of MORE than coinc_beam_fraction * nbeam
        distinct beams (its own included) arrive within coinc_window_s of it."""
    beam = np.asarray(beam); trial = np.asarray(trial); t = np.asarray(t); width = np.asarray(width)
    snr = np.asarray(snr, dtype=np.float64)
    dm = np.asarray(dm_of_trial, dtype=np.float64)[trial]
    k = np.asarray(decim_of_trial, dtype=np.int64)[trial]
    arrival = (t.astype(np.float64) * k.astype(np.float64)) * tsamp            # seconds, at the top of the band
    wsec = (width.astype(np.float64) * k.astype(np.float64)) * tsamp
    n = beam.size
    keep1 = np.zeros(n, dtype=bool)

    def stronger(a, b):                                  # is candidate a stronger than b
        return snr[a] > snr[b] or (snr[a] == snr[b] and (trial[a], t[a]) < (trial[b], t[b]))

    for b in np.unique(beam):
        idx = np.flatnonzero(beam == b)
        xs, ys = arrival[idx] / time_unit_s, dm[idx] / dm_unit
        core, label = dbscan(xs, ys, eps, min_pts)
        member = label.copy()
        dx = xs[:, None] - xs[None, :]
        dy = ys[:, None] - ys[None, :]
        near = (dx * dx + dy * dy) <= eps * eps
        for i in np.flatnonzero(~core):
            best = -1
            for j in np.flatnonzero(near[i] & core):
                if best < 0 or stronger(idx[j], idx[best]):
                    best = int(j)
            if best >= 0:
                member[i] = label[best]
        for c in np.unique(member[member >= 0]):
            mem = np.flatnonzero(member == c)
            top = mem[0]
            for j in mem[1:]:
                if stronger(idx[j], idx[top]):
                    top = j
            keep1[idx[top]] = True
    keep2 = keep1 & (snr >= snr_min) & (dm >= dm_min) & (wsec <= width_max_s)
    keep3 = keep2.copy()
    if coinc_window_s > 0.0:
        s = np.flatnonzero(keep2)
        for i in s:
            beams = set(int(beam[j]) for j in s if abs(arrival[j] - arrival[i]) <= coinc_window_s)
            if len(beams) > coinc_beam_fraction * nbeam:
                keep3[i] = False
    return keep1, keep2, keep3


# ---- H. candidate cut-outs (Eq. 4) -------------------------------------------------------
def cutout(x: np.ndarray, fch1: float, foff: float, tsamp: float, dm0: float, ddm: float, ndm: int, ts: int, tbin: int,
           nt: int, nf: int) -> Tuple[np.ndarray, np.ndarray]:
    """(dedispersed dynamic spectrum [nf][nt], DM transform [ndm][nt]) of one candidate, integers."""
    x = np.ascontiguousarray(x, dtype=np.uint8)
    dds = np.zeros((nf, nt), dtype=np.int32)
    dmt = np.zeros((ndm, nt), dtype=np.int32)
    _check(lib().orc_cutout(_ptr(x), x.shape[0], x.shape[1], fch1, foff, tsamp, dm0, ddm, ndm, ts, tbin, nt, nf, _ptr(dds),
                            _ptr(dmt)), "cutout")
    return dds, dmt


def delta_dm(width_s: float, nu_mhz: float, bw_mhz: float, snr_ratio: float = 0.1, constant: float = 1382.0) -> float:
    """Eq. 4: half-width of the DM range over which the S/N drops to snr_ratio of its peak."""
    return float(lib().orc_delta_dm(width_s, 1.0 / snr_ratio, nu_mhz, bw_mhz, constant))


# ---- whole path over a plan (one beam) ----------------------------------------------------------------
@dataclass
class RangeResult:
    dm: np.ndarray        # float64 [ndm]
    decim: int
    delay: np.ndarray     # int32 [ndm][nchan]
    nout: np.ndarray      # int32 [ndm]
    series: Optional[np.ndarray]   # decimated input (uint16) or None for k == 1
    dmt: np.ndarray       # int32 packed rows
    rowoff: np.ndarray    # int64 [ndm+1]
    search: Optional[PlaneSearch]


def run_path(fb: np.ndarray, fch1: float, foff: float, tsamp: float,
             ranges: Sequence[Tuple[float, float, int, int]], widths: Sequence[int], threshold: float,
             do_search: bool = True) -> List[RangeResult]:
    """delay table -> decimate -> dedisperse -> single-pulse search, range by range, for one beam."""
    fb = np.ascontiguousarray(fb, dtype=np.uint8)
    nchan, nsamp = fb.shape
    out = []
    for (dm_lo, dm_step, ndm, k) in ranges:
        dly = delay_table(fch1, foff, nchan, tsamp, dm_lo, dm_step, ndm, k)
        no = nout(dly, nsamp, k)
        y = None if k == 1 else decimate(fb, k)
        dmt, rowoff = dedisperse(fb if k == 1 else y, dly, no)
        sr = search_plane(dmt, rowoff[:-1], no, widths, threshold) if do_search else None
        dms = dm_lo + np.arange(ndm, dtype=np.float64) * dm_step
        out.append(RangeResult(dms, k, dly, no, y, dmt, rowoff, sr))
    return out
