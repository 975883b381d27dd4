"""Thin ctypes binding of libspt (include/spt.h): argument marshalling only.

Every step of the path (decimation, dedispersion, single-pulse search, candidate append) runs in the CUDA
kernels behind the C ABI; torch is used here for device memory and streams.  There is no CPU fallback: if
libspt.so is missing or no CUDA device is usable the calls raise.
"""
from __future__ import annotations

import ctypes
import os
from typing import List, Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libspt.so")

SPT_OK = 0
SPT_ERR_INVALID, SPT_ERR_UNSUPPORTED, SPT_ERR_NOMEM, SPT_ERR_CUDA, SPT_ERR_SHAPE, SPT_ERR_STATE = -1, -2, -3, -4, -5, -6


class spt_dm_range(ctypes.Structure):
    _fields_ = [("dm_lo", ctypes.c_double), ("dm_step", ctypes.c_double), ("ndm", ctypes.c_int32),
                ("decim", ctypes.c_int32)]


class spt_candidate(ctypes.Structure):
    _fields_ = [("beam", ctypes.c_int32), ("trial", ctypes.c_int32), ("t", ctypes.c_int32),
                ("width", ctypes.c_int32), ("snr", ctypes.c_float)]


class spt_cutout_params(ctypes.Structure):
    _fields_ = [("dm0", ctypes.c_double), ("ddm", ctypes.c_double), ("ts", ctypes.c_int64), ("tbin", ctypes.c_int32),
                ("beam", ctypes.c_int32)]


class spt_sift_params(ctypes.Structure):
    _fields_ = [("eps", ctypes.c_double), ("time_unit_s", ctypes.c_double), ("dm_unit", ctypes.c_double),
                ("min_pts", ctypes.c_int32), ("snr_min", ctypes.c_float), ("dm_min", ctypes.c_double),
                ("width_max_s", ctypes.c_double), ("coinc_window_s", ctypes.c_double),
                ("coinc_beam_fraction", ctypes.c_double)]


PEAKS_STATIC_MAX = 262144       # SPT_PEAKS_STATIC_MAX of include/spt.h: records spt_peak_filter_static takes at most

CAND_DTYPE = np.dtype([("beam", "<i4"), ("trial", "<i4"), ("t", "<i4"), ("width", "<i4"), ("snr", "<f4")])

# every symbol include/spt.h declares: name -> (restype, argtypes)
_vp, _i32, _i64, _f64, _f32 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_double, ctypes.c_float
_P = ctypes.POINTER
SYMBOLS = {
    "spt_plan_create": (ctypes.c_int, [_f64, _f64, _i32, _f64, _i64, _P(spt_dm_range), _i32, _P(_i32), _i32, _i32, _i64,
                                       _P(_vp)]),
    "spt_plan_destroy": (ctypes.c_int, [_vp]),
    "spt_plan_info": (ctypes.c_int, [_vp, _P(_i32), _P(_i64)]),
    "spt_plan_trial": (ctypes.c_int, [_vp, _i32, _P(_f64), _P(_i32), _P(_i32), _P(_i32), _P(_i64)]),
    "spt_plan_delays": (ctypes.c_int, [_vp, _i32, _vp]),
    "spt_plan_set_option": (ctypes.c_int, [_vp, ctypes.c_char_p, _i64]),
    "spt_plan_tiling_info": (ctypes.c_int, [_vp, _i32, _P(_i64), _P(_i64), _P(_i64), _P(_i64), _P(_i64), _P(_i64)]),
    "spt_plan_tiling_cost": (ctypes.c_int, [_vp, _i32, _P(_i64), _P(_i64), _P(_i64), _P(_i64)]),
    "spt_plan_tiling_choice": (ctypes.c_int, [_vp, _i32, _P(_i32), _P(_i32), _P(_i32), _P(_i32)]),
    "spt_plan_tiling_delays": (ctypes.c_int, [_vp, _i32, _vp]),
    "spt_dedisperse": (ctypes.c_int, [_vp, _vp, _i32, _vp, _vp]),
    "spt_decimated": (ctypes.c_int, [_vp, _i32, _P(_vp), _P(_i64)]),
    "spt_decimated_stride": (ctypes.c_int, [_vp, _i32, _P(_i64)]),
    "spt_decimated_read": (ctypes.c_int, [_vp, _i32, _i32, _vp]),
    "spt_decimated_compact": (ctypes.c_int, [_vp, _i32, _P(_i32), _P(ctypes.c_uint32), _P(ctypes.c_uint32)]),
    "spt_single_pulse_search": (ctypes.c_int, [_vp, _vp, _i32, _f32, _vp]),
    "spt_search": (ctypes.c_int, [_vp, _vp, _i32, _vp, _f32, _vp]),
    "spt_trial_stats": (ctypes.c_int, [_vp, _i32, _i32, _P(_i64), _P(_i64), _P(ctypes.c_uint64)]),
    "spt_trial_stats_all": (ctypes.c_int, [_vp, _i32, _vp, _vp]),
    "spt_candidates_count": (ctypes.c_int, [_vp, _P(_i64), _P(_i32)]),
    "spt_candidates_read": (ctypes.c_int, [_vp, _vp, _i64, _P(_i64)]),
    "spt_search_host": (ctypes.c_int, [_vp, _vp, _i32, _f32, _vp, _P(_i64), _P(_i32)]),
    "spt_peak_filter": (ctypes.c_int, [_vp, _P(_i32), _i32, _vp]),
    "spt_peak_filter_static": (ctypes.c_int, [_vp, _vp, _i64, _P(_i32), _i32, _vp, _vp, _vp]),
    "spt_peaks_count": (ctypes.c_int, [_vp, _P(_i64)]),
    "spt_peaks_read": (ctypes.c_int, [_vp, _vp, _i64, _P(_i64)]),
    "spt_corner_turn": (ctypes.c_int, [_vp, _i32, _i64, _i32, _i32, _i32, _vp, _vp]),
    "spt_segment_info": (ctypes.c_int, [_vp, _P(_i64), _P(_i64), _P(_i64)]),
    "spt_segment_search": (ctypes.c_int, [_vp, _vp, _i32, _i64, _f32, _vp]),
    "spt_segment_push": (ctypes.c_int, [_vp, _vp, _i32, _i64, _i32, _i32, _i32, _vp, _vp]),
    "spt_cutout": (ctypes.c_int, [_vp, _i32, _i64, _f64, _f64, _f64, _f64, _f64, _i32, _i64, _i32, _i32, _i32, _vp, _vp, _vp]),
    "spt_cutout_batch": (ctypes.c_int, [_vp, _i32, _i32, _i64, _f64, _f64, _f64, _P(spt_cutout_params), _i32, _i32, _i32, _i32, _vp,
                                        _vp, _vp]),
    "spt_delta_dm": (_f64, [_f64, _f64, _f64, _f64]),
    "spt_sift": (ctypes.c_int, [_vp, _vp, _i64, _i32, _P(spt_sift_params), _vp, _i64, _P(_i64), _P(_i64)]),
    "spt_stream_push": (ctypes.c_int, [_vp, _vp, _i32, _f32]),
    "spt_stream_pop": (ctypes.c_int, [_vp, _P(_i64), _P(_i32)]),
    "spt_plan_kernel_times": (ctypes.c_int, [_vp, _i32, _vp, _vp, _vp, _P(_i32)]),
    "spt_plan_launches": (ctypes.c_int, [_vp, _P(_i64)]),
    "spt_probe": (ctypes.c_int, [_i32, _i32, _P(_f64), _P(_f64)]),
    "spt_strerror": (ctypes.c_char_p, [ctypes.c_int]),
    "spt_last_error": (ctypes.c_char_p, []),
}

_lib = None


def lib() -> ctypes.CDLL:
    """Load libspt.so (built in-tree by paper_2606_27262_b200.build); fails loudly when it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2606_27262_b200.build` "
                               "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


class SptError(RuntimeError):
    def __init__(self, code: int, what: str):
        L = lib()
        msg = L.spt_strerror(code).decode()
        detail = L.spt_last_error().decode()
        super().__init__(f"{what}: {msg} ({code})" + (f" [{detail}]" if detail and code == SPT_ERR_CUDA else ""))
        self.code = code


def _check(rc: int, what: str):
    if rc != SPT_OK:
        raise SptError(rc, what)


def _dev_ptr(t) -> int:
    """Raw device pointer of a CUDA torch tensor (contiguous)."""
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous CUDA tensor")
    return t.data_ptr()


def _stream_ptr(stream=None) -> int:
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return s.cuda_stream


class Plan:
    """Owner of one spt_plan; method names follow the C calls."""

    def __init__(self, fch1: float, foff: float, nchan: int, tsamp: float, nsamp: int,
                 ranges: Sequence[Tuple[float, float, int, int]], widths: Sequence[int], max_beams: int = 1,
                 cand_capacity: int = 1 << 20, options: Optional[dict] = None):
        L = lib()
        arr = (spt_dm_range * len(ranges))(*[spt_dm_range(float(a), float(b), int(c), int(d)) for a, b, c, d in ranges])
        w = (ctypes.c_int32 * len(widths))(*[int(x) for x in widths])
        h = ctypes.c_void_p()
        _check(L.spt_plan_create(fch1, foff, nchan, tsamp, nsamp, arr, len(ranges), w, len(widths), max_beams,
                                 cand_capacity, ctypes.byref(h)), "spt_plan_create")
        self._h = h
        self.nchan, self.nsamp, self.max_beams, self.cand_capacity = nchan, nsamp, max_beams, cand_capacity
        self.ranges = [tuple(r) for r in ranges]
        self.widths = list(widths)
        n, e = ctypes.c_int32(), ctypes.c_int64()
        _check(L.spt_plan_info(h, ctypes.byref(n), ctypes.byref(e)), "spt_plan_info")
        self.ntrials, self.dmt_elems_per_beam = int(n.value), int(e.value)
        for k, v in (options or {}).items():
            self.set_option(k, v)
        self._meta = None

    def close(self):
        if getattr(self, "_h", None):
            lib().spt_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- host-side plan ------------------------------------------------------------------------------------------
    def set_option(self, name: str, value: int):
        _check(lib().spt_plan_set_option(self._h, name.encode(), int(value)), f"spt_plan_set_option({name})")

    def trial(self, d: int):
        dm, rg, k, no, off = ctypes.c_double(), ctypes.c_int32(), ctypes.c_int32(), ctypes.c_int32(), ctypes.c_int64()
        _check(lib().spt_plan_trial(self._h, d, ctypes.byref(dm), ctypes.byref(rg), ctypes.byref(k), ctypes.byref(no),
                                    ctypes.byref(off)), "spt_plan_trial")
        return dm.value, rg.value, k.value, no.value, off.value

    def trial_table(self):
        """(dm[ntrials], range, decim, nout, offset) as numpy arrays."""
        if self._meta is None:
            rows = [self.trial(d) for d in range(self.ntrials)]
            self._meta = (np.array([r[0] for r in rows]), np.array([r[1] for r in rows], dtype=np.int32),
                          np.array([r[2] for r in rows], dtype=np.int32), np.array([r[3] for r in rows], dtype=np.int32),
                          np.array([r[4] for r in rows], dtype=np.int64))
        return self._meta

    def delays(self, d: int) -> np.ndarray:
        out = np.empty(self.nchan, dtype=np.int32)
        _check(lib().spt_plan_delays(self._h, d, out.ctypes.data), "spt_plan_delays")
        return out

    def tiling_info(self, rng: int) -> dict:
        v = [ctypes.c_int64() for _ in range(6)]
        _check(lib().spt_plan_tiling_info(self._h, rng, *[ctypes.byref(x) for x in v]), "spt_plan_tiling_info")
        keys = ("ntiles_dm", "nstages", "ngroups", "nvariants", "ntiles_t", "max_stage_words")
        return {k: int(x.value) for k, x in zip(keys, v)}

    def tiling_cost(self, rng: int) -> dict:
        v = [ctypes.c_int64() for _ in range(4)]
        _check(lib().spt_plan_tiling_cost(self._h, rng, *[ctypes.byref(x) for x in v]), "spt_plan_tiling_cost")
        return {k: int(x.value) for k, x in zip(("ntasks", "task_entries", "task_variants", "presum_rounds"), v)}

    def tiling_choice(self, rng: int) -> dict:
        v = [ctypes.c_int32() for _ in range(4)]
        _check(lib().spt_plan_tiling_choice(self._h, rng, *[ctypes.byref(x) for x in v]), "spt_plan_tiling_choice")
        return {k: int(x.value) for k, x in zip(("tile_words", "max_entries", "group", "has_compact"), v)}

    def tiling_delays(self, d: int) -> np.ndarray:
        out = np.empty(self.nchan, dtype=np.int32)
        _check(lib().spt_plan_tiling_delays(self._h, d, out.ctypes.data), "spt_plan_tiling_delays")
        return out

    # ---- device path ---------------------------------------------------------------------------------------------
    def dedisperse(self, d_fb, d_dmt=None, stream=None):
        """d_fb: CUDA uint8 tensor [nbeam][nchan][nsamp].  Returns the int32 DM transform tensor [nbeam][dmt_elems]."""
        import torch
        if d_fb.dim() == 2:
            d_fb = d_fb.unsqueeze(0)
        nbeam = d_fb.shape[0]
        assert d_fb.dtype == torch.uint8 and tuple(d_fb.shape[1:]) == (self.nchan, self.nsamp)
        if d_dmt is None:
            d_dmt = torch.empty((nbeam, self.dmt_elems_per_beam), dtype=torch.int32, device=d_fb.device)
        _check(lib().spt_dedisperse(self._h, _dev_ptr(d_fb), nbeam, _dev_ptr(d_dmt), _stream_ptr(stream)),
               "spt_dedisperse")
        return d_dmt

    def decimated_read(self, rng: int, beam: int = 0) -> Optional[np.ndarray]:
        """Decimated series of range `rng`, one beam, as a host uint16 array [nchan][nsamp_k] (None when decim == 1)."""
        p, n = ctypes.c_void_p(), ctypes.c_int64()
        _check(lib().spt_decimated(self._h, rng, ctypes.byref(p), ctypes.byref(n)), "spt_decimated")
        if not p.value:
            return None
        out = np.empty((self.nchan, int(n.value)), dtype=np.uint16)
        _check(lib().spt_decimated_read(self._h, rng, beam, out.ctypes.data), "spt_decimated_read")
        return out

    def decimated_compact(self, rng: int) -> Tuple[bool, int, int]:
        """(in_use, floor, span): whether the last dedispersion read range `rng`'s series through its 8-bit copy."""
        u, f, sp = ctypes.c_int32(), ctypes.c_uint32(), ctypes.c_uint32()
        _check(lib().spt_decimated_compact(self._h, rng, ctypes.byref(u), ctypes.byref(f), ctypes.byref(sp)), "spt_decimated_compact")
        return bool(u.value), int(f.value), int(sp.value)

    def single_pulse_search(self, d_dmt, threshold: float, stream=None):
        nbeam = d_dmt.shape[0] if d_dmt.dim() == 2 else 1
        _check(lib().spt_single_pulse_search(self._h, _dev_ptr(d_dmt), nbeam, float(threshold), _stream_ptr(stream)),
               "spt_single_pulse_search")

    def search(self, d_fb, threshold: float, d_dmt=None, stream=None):
        """dedisperse + single_pulse_search in one call (spt_search): every DM range is searched as soon as its rows are
        done.  Returns the DM transform tensor."""
        import torch
        if d_fb.dim() == 2:
            d_fb = d_fb.unsqueeze(0)
        nbeam = d_fb.shape[0]
        assert d_fb.dtype == torch.uint8 and tuple(d_fb.shape[1:]) == (self.nchan, self.nsamp)
        if d_dmt is None:
            d_dmt = torch.empty((nbeam, self.dmt_elems_per_beam), dtype=torch.int32, device=d_fb.device)
        _check(lib().spt_search(self._h, _dev_ptr(d_fb), nbeam, _dev_ptr(d_dmt), float(threshold), _stream_ptr(stream)),
               "spt_search")
        return d_dmt

    def trial_stats(self, beam: int, trial: int):
        n, s, q = ctypes.c_int64(), ctypes.c_int64(), ctypes.c_uint64()
        _check(lib().spt_trial_stats(self._h, beam, trial, ctypes.byref(n), ctypes.byref(s), ctypes.byref(q)),
               "spt_trial_stats")
        return int(n.value), int(s.value), int(q.value)

    def trial_stats_all(self, nbeam: int = 1):
        s = np.empty((nbeam, self.ntrials), dtype=np.int64)
        q = np.empty((nbeam, self.ntrials), dtype=np.uint64)
        _check(lib().spt_trial_stats_all(self._h, nbeam, s.ctypes.data, q.ctypes.data), "spt_trial_stats_all")
        return s, q

    def candidates_count(self):
        t, o = ctypes.c_int64(), ctypes.c_int32()
        _check(lib().spt_candidates_count(self._h, ctypes.byref(t), ctypes.byref(o)), "spt_candidates_count")
        return int(t.value), bool(o.value)

    def candidates_read(self, cap: Optional[int] = None) -> np.ndarray:
        total, _ = self.candidates_count()
        n = min(total, self.cand_capacity if cap is None else cap)
        out = np.empty(max(n, 1), dtype=CAND_DTYPE)
        w = ctypes.c_int64()
        _check(lib().spt_candidates_read(self._h, out.ctypes.data, n, ctypes.byref(w)), "spt_candidates_read")
        return out[: int(w.value)]

    def search_host(self, h_fb, threshold: float, h_dmt=None):
        """Whole path from a HOST uint8 array/tensor [nbeam][nchan][nsamp]; returns (ncand, overflowed)."""
        ptr, nbeam = _host_ptr_and_beams(h_fb, self.nchan, self.nsamp)
        dptr = None
        if h_dmt is not None:
            dptr = h_dmt.ctypes.data if isinstance(h_dmt, np.ndarray) else h_dmt.data_ptr()
        n, o = ctypes.c_int64(), ctypes.c_int32()
        _check(lib().spt_search_host(self._h, ptr, nbeam, float(threshold), dptr, ctypes.byref(n), ctypes.byref(o)),
               "spt_search_host")
        return int(n.value), bool(o.value)

    def peak_filter(self, windows: Sequence[int] = (3, 11), stream=None) -> np.ndarray:
        """Peak filtering of the last search's candidates; returns the surviving records."""
        w = (ctypes.c_int32 * len(windows))(*[int(x) for x in windows])
        _check(lib().spt_peak_filter(self._h, w, len(windows), _stream_ptr(stream)), "spt_peak_filter")
        n = ctypes.c_int64()
        _check(lib().spt_peaks_count(self._h, ctypes.byref(n)), "spt_peaks_count")
        out = np.empty(max(int(n.value), 1), dtype=CAND_DTYPE)
        k = ctypes.c_int64()
        _check(lib().spt_peaks_read(self._h, out.ctypes.data, int(n.value), ctypes.byref(k)), "spt_peaks_read")
        return out[: int(k.value)]

    def peak_filter_static(self, d_cand, n: int, windows: Sequence[int], d_peaks, d_count, stream=None) -> None:
        """spt_peak_filter_static: the peak filter for callers that may not allocate device memory (a real-time loop that
        cannot take the device-wide stall of a cudaMalloc; a process whose memory another allocator owns).  Working
        memory is a fixed block inside libspt.so, so n <= PEAKS_STATIC_MAX.  d_cand: CUDA tensor holding n candidate
        records (20 bytes each) of a search made with this plan; d_peaks: CUDA tensor with room for n records; d_count:
        CUDA int64 tensor of one element.  Only enqueues: synchronise the stream before reading d_count / d_peaks.  Calls
        share the block: do not let two of them overlap on the GPU."""
        w = (ctypes.c_int32 * len(windows))(*[int(x) for x in windows])
        rc = lib().spt_peak_filter_static(self._h, _dev_ptr(d_cand), int(n), w, len(windows), _dev_ptr(d_peaks),
                                          _dev_ptr(d_count), _stream_ptr(stream))
        if rc == SPT_ERR_UNSUPPORTED:
            raise SptError(rc, "spt_peak_filter_static: " + lib().spt_last_error().decode())
        _check(rc, "spt_peak_filter_static")

    def segment_info(self):
        """(min_history, min_history_search, granule) in raw samples for spt_segment_push / spt_segment_search."""
        h, hs, g = ctypes.c_int64(), ctypes.c_int64(), ctypes.c_int64()
        _check(lib().spt_segment_info(self._h, ctypes.byref(h), ctypes.byref(hs), ctypes.byref(g)), "spt_segment_info")
        return int(h.value), int(hs.value), int(g.value)

    def segment_search(self, d_dmt, nnew: int, threshold: float, stream=None):
        """Search of the segment just pushed (window = last nnew/k + wmax - 1 samples of every row)."""
        _check(lib().spt_segment_search(self._h, _dev_ptr(d_dmt), d_dmt.shape[0], int(nnew), float(threshold),
                                        _stream_ptr(stream)), "spt_segment_search")

    def segment_push(self, d_new, flip: bool = False, d_dmt=None, stream=None, spliced: bool = False, whole_rows: bool = True):
        """Overlap-save push of a time-major CUDA uint8 block, [nbeam][nnew][nchan] or (spliced) [nnew][nbeam][nchan];
        whole_rows=False computes only the new tail of every row.  Returns the DM transform tensor."""
        import torch
        if spliced:
            nnew, nbeam, nchan = d_new.shape
        else:
            nbeam, nnew, nchan = d_new.shape
        if nchan != self.nchan or d_new.dtype != torch.uint8:
            raise ValueError("block must be uint8 [nbeam][nnew][nchan] or [nnew][nbeam][nchan]")
        if d_dmt is None:
            d_dmt = torch.empty((nbeam, self.dmt_elems_per_beam), dtype=torch.int32, device=d_new.device)
        _check(lib().spt_segment_push(self._h, _dev_ptr(d_new), nbeam, nnew, int(bool(flip)), int(bool(spliced)),
                                      int(bool(whole_rows)), _dev_ptr(d_dmt), _stream_ptr(stream)), "spt_segment_push")
        return d_dmt

    def sift(self, cands: np.ndarray, nbeam: int, eps: float = 0.5, min_pts: int = 5, time_unit_s: float = 1.0,
             dm_unit: float = 1.0, snr_min: float = 10.0, dm_min: float = 10.0, width_max_s: float = 0.1,
             coinc_window_s: float = 0.0, coinc_beam_fraction: float = 0.5):
        """Candidate optimisation of a host list of records; returns (survivors, stage counts)."""
        cands = np.ascontiguousarray(cands, dtype=CAND_DTYPE)
        prm = spt_sift_params(eps, time_unit_s, dm_unit, min_pts, snr_min, dm_min, width_max_s, coinc_window_s,
                              coinc_beam_fraction)
        out = np.empty(max(cands.size, 1), dtype=CAND_DTYPE)
        nw = ctypes.c_int64()
        stages = (ctypes.c_int64 * 3)()
        _check(lib().spt_sift(self._h, cands.ctypes.data, cands.size, nbeam, ctypes.byref(prm), out.ctypes.data, cands.size,
                              ctypes.byref(nw), stages), "spt_sift")
        return out[: int(nw.value)], [int(v) for v in stages]

    def stream_push(self, h_fb, threshold: float):
        """Enqueue one batch (HOST uint8 [nbeam][nchan][nsamp], pinned) into the two-deep pipeline; returns at once."""
        ptr, nbeam = _host_ptr_and_beams(h_fb, self.nchan, self.nsamp)
        _check(lib().spt_stream_push(self._h, ptr, nbeam, float(threshold)), "spt_stream_push")

    def stream_pop(self):
        """Wait for the oldest batch in flight; returns (ncand, overflowed)."""
        n, o = ctypes.c_int64(), ctypes.c_int32()
        _check(lib().spt_stream_pop(self._h, ctypes.byref(n), ctypes.byref(o)), "spt_stream_pop")
        return int(n.value), bool(o.value)

    def kernel_times(self):
        """[(kind, range, ms)] of the last dedisperse + search (option "profile" = 1); kinds 1 decimate, 2 dedisperse, 3 search."""
        cap = 64
        k = np.zeros(cap, dtype=np.int32)
        r = np.zeros(cap, dtype=np.int32)
        ms = np.zeros(cap, dtype=np.float64)
        n = ctypes.c_int32()
        _check(lib().spt_plan_kernel_times(self._h, cap, k.ctypes.data, r.ctypes.data, ms.ctypes.data, ctypes.byref(n)),
               "spt_plan_kernel_times")
        return [(int(k[i]), int(r[i]), float(ms[i])) for i in range(n.value)]

    def launches(self) -> int:
        n = ctypes.c_int64()
        _check(lib().spt_plan_launches(self._h, ctypes.byref(n)), "spt_plan_launches")
        return int(n.value)


def _host_ptr_and_beams(h_fb, nchan, nsamp):
    if isinstance(h_fb, np.ndarray):
        assert h_fb.dtype == np.uint8 and h_fb.flags.c_contiguous
        shape, ptr = h_fb.shape, h_fb.ctypes.data
    else:  # torch CPU tensor (pinned or not)
        assert not h_fb.is_cuda and h_fb.is_contiguous()
        shape, ptr = tuple(h_fb.shape), h_fb.data_ptr()
    if len(shape) == 2:
        shape = (1,) + tuple(shape)
    assert tuple(shape[1:]) == (nchan, nsamp)
    return ptr, shape[0]


def cutout(d_fb, fch1: float, foff: float, tsamp: float, dm0: float, ddm: float, ndm: int, ts: int, tbin: int, nt: int, nf: int,
           stream=None):
    """(dedispersed dynamic spectrum [nf][nt], DM transform [ndm][nt]) of one candidate from a CUDA uint8 [nchan][nsamp] beam."""
    import torch
    nchan, nsamp = d_fb.shape
    dds = torch.empty((nf, nt), dtype=torch.int32, device=d_fb.device)
    dmt = torch.empty((ndm, nt), dtype=torch.int32, device=d_fb.device)
    _check(lib().spt_cutout(_dev_ptr(d_fb), nchan, nsamp, fch1, foff, tsamp, dm0, ddm, ndm, ts, tbin, nt, nf, _dev_ptr(dds),
                            _dev_ptr(dmt), _stream_ptr(stream)), "spt_cutout")
    return dds, dmt


def cutout_batch(d_fb, fch1: float, foff: float, tsamp: float, cands, ndm: int, nt: int, nf: int, stream=None):
    """The cut-outs of many candidates in one launch.  d_fb: CUDA uint8 [nbeam][nchan][nsamp]; cands: sequence of
    (dm0, ddm, ts, tbin, beam).  Returns (dds [ncand][nf][nt], dmt [ncand][ndm][nt]) int32 CUDA tensors."""
    import torch
    if d_fb.dim() == 2:
        d_fb = d_fb.unsqueeze(0)
    nbeam, nchan, nsamp = d_fb.shape
    n = len(cands)
    arr = (spt_cutout_params * n)(*[spt_cutout_params(float(a), float(b), int(c), int(d), int(e)) for a, b, c, d, e in cands])
    dds = torch.empty((n, nf, nt), dtype=torch.int32, device=d_fb.device)
    dmt = torch.empty((n, ndm, nt), dtype=torch.int32, device=d_fb.device)
    _check(lib().spt_cutout_batch(_dev_ptr(d_fb), nbeam, nchan, nsamp, fch1, foff, tsamp, arr, n, ndm, nt, nf, _dev_ptr(dds),
                                  _dev_ptr(dmt), _stream_ptr(stream)), "spt_cutout_batch")
    return dds, dmt


def delta_dm(width_s: float, nu_mhz: float, bw_mhz: float, snr_ratio: float = 0.1) -> float:
    return float(lib().spt_delta_dm(width_s, snr_ratio, nu_mhz, bw_mhz))


def corner_turn(d_in, flip: bool = False, stream=None, spliced: bool = False):
    """Time-major CUDA uint8 [nbeam][nsamp][nchan] (spliced: [nsamp][nbeam][nchan]) -> channel-major [nbeam][nchan][nsamp]
    (optionally band-flipped)."""
    import torch
    if spliced:
        nsamp, nbeam, nchan = d_in.shape
    else:
        nbeam, nsamp, nchan = d_in.shape
    out = torch.empty((nbeam, nchan, nsamp), dtype=torch.uint8, device=d_in.device)
    _check(lib().spt_corner_turn(_dev_ptr(d_in), nbeam, nsamp, nchan, int(bool(flip)), int(bool(spliced)), _dev_ptr(out),
                                 _stream_ptr(stream)), "spt_corner_turn")
    return out


def probe(kind: int, reps: int = 5) -> Tuple[float, float]:
    """(warp instructions per second, elapsed ms) of roofline probe `kind` (see spt_probe in spt.h)."""
    r, ms = ctypes.c_double(), ctypes.c_double()
    _check(lib().spt_probe(kind, reps, ctypes.byref(r), ctypes.byref(ms)), "spt_probe")
    return float(r.value), float(ms.value)
