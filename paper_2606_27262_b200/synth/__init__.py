"""Seeded synthetic workloads (the five BASELINE.json configs) -- input generator only.

This module makes the bytes that BOTH the CUDA path and the oracle are fed, and the
plain workload parameters (band, plan ranges, widths, threshold).  It holds none of the
method's arithmetic: no delay table, no dedispersion, no boxcar, no S/N (see synth.c).

The inputs stand in for uGMRT beams, which are not in the container (the paper measures on
Cycle 49/50 observations): 8-bit samples, channel 0 = highest frequency,
tsamp = 1.31072 ms, 200 MHz bands.  Recipe: SURVEY.md section 8(d),
restated in DESIGN.md.
"""
from __future__ import annotations

import ctypes
import math
import os
import subprocess
from dataclasses import dataclass, field
from typing import List, Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libsptsynth.so")
_SRC = os.path.join(_HERE, "synth.c")

TSAMP = 1.31072e-3


def build(force: bool = False) -> str:
    """Compile synth.c into libsptsynth.so (gcc, OpenMP)."""
    if force or (not os.path.exists(_SO)) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC", "-o", _SO, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _SO


class _Burst(ctypes.Structure):
    _fields_ = [("dm", ctypes.c_double), ("amp", ctypes.c_double), ("t0", ctypes.c_int64),
                ("width", ctypes.c_int32), ("pad_", ctypes.c_int32)]


class _Tone(ctypes.Structure):
    _fields_ = [("offset", ctypes.c_double), ("amp", ctypes.c_double), ("period", ctypes.c_double),
                ("phase", ctypes.c_double), ("chan", ctypes.c_int32), ("pad_", ctypes.c_int32)]


class _Spike(ctypes.Structure):
    _fields_ = [("amp", ctypes.c_double), ("t0", ctypes.c_int64), ("dur", ctypes.c_int32),
                ("pad_", ctypes.c_int32)]


_lib = None


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_SO)
        lib.synth_filterbank.restype = ctypes.c_int
        lib.synth_filterbank.argtypes = [
            ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_double, ctypes.c_double, ctypes.c_double,
            ctypes.c_double, ctypes.c_double, ctypes.c_uint64, ctypes.c_uint64,
            ctypes.c_void_p, ctypes.c_int32, ctypes.c_void_p, ctypes.c_int32, ctypes.c_void_p, ctypes.c_int32,
            ctypes.c_int32]
        lib.synth_checksum.restype = ctypes.c_uint64
        lib.synth_checksum.argtypes = [ctypes.c_void_p, ctypes.c_int64]
        lib.synth_sweep_samples.restype = ctypes.c_int
        lib.synth_sweep_samples.argtypes = [ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_int32,
                                            ctypes.c_double, ctypes.POINTER(ctypes.c_int64)]
        _lib = lib
    return _lib


@dataclass
class Burst:
    dm: float
    t0: int
    width: int
    snr: float          # injected matched-filter S/N at the exact DM and width
    amp: float          # counts per channel per sample
    truncated: bool = False   # the sweep does not fit in nsamp (cfg 4, high DM)


@dataclass
class Workload:
    """One BASELINE.json config: band, length, plan, search parameters, signal recipe."""
    name: str
    index: int                      # 1-based config number
    nbeam: int
    nchan: int
    nsamp: int
    fch1: float
    foff: float
    tsamp: float
    mean: float
    std: float
    ranges: List[Tuple[float, float, int, int]]     # (dm_lo, dm_step, ndm, decim)
    widths: List[int]
    threshold: float
    seed: int
    bursts: List[List[Burst]] = field(default_factory=list)   # per beam
    tones: list = field(default_factory=list)                  # (chan, offset, amp, period, phase)
    spikes: list = field(default_factory=list)                 # (t0, dur, amp)

    @property
    def ntrials(self) -> int:
        return sum(r[2] for r in self.ranges)

    def beam_seed(self, beam: int) -> int:
        return self.seed + beam if self.nbeam > 1 else self.seed


def sweep_samples(dm: float, fch1: float, foff: float, chan: int, tsamp: float) -> int:
    """Sample offset of a burst in channel `chan` (the generator's own sweep, see synth.c)."""
    out = ctypes.c_int64(0)
    _load().synth_sweep_samples(dm, fch1, foff, chan, tsamp, ctypes.byref(out))
    return int(out.value)


def _pow2_widths(wmax: int) -> List[int]:
    return [1 << i for i in range(int(math.log2(wmax)) + 1)]


_PLAN3 = [(0.0, 0.2, 2500, 1), (500.0, 0.5, 1000, 2), (1000.0, 1.0, 1001, 4)]


def _draw_bursts(rng, n, nchan, nsamp, fch1, foff, tsamp, std, dm_lo, dm_hi, width_fn, snr_lo, snr_hi):
    out = []
    for _ in range(n):
        dm = float(rng.uniform(dm_lo, dm_hi))
        w = int(width_fn(rng))
        snr = float(rng.uniform(snr_lo, snr_hi))
        sweep = sweep_samples(dm, fch1, foff, nchan - 1, tsamp)
        room = nsamp - sweep - w
        if room > 0:
            t0 = int(rng.integers(0, room + 1))
            trunc = False
        else:
            t0 = int(rng.integers(0, max(1, nsamp // 2)))
            trunc = True
        amp = snr * std / math.sqrt(nchan * w)
        out.append(Burst(dm=dm, t0=t0, width=w, snr=snr, amp=amp, truncated=trunc))
    return out


def workload(index: int, nsamp: Optional[int] = None, nbeam: Optional[int] = None) -> Workload:
    """BASELINE.json configs[index-1] (index 6: the Band-5 workload of SURVEY.md NEXT-4).  `nsamp`/`nbeam` override the
    length (reduced-size parity cases)."""
    if index == 1:
        w = Workload("cfg1-tiny", 1, 1, 64, 4096, 500.0, -3.125, TSAMP, 128.0, 16.0,
                     [(0.0, 1.0, 101, 1)], _pow2_widths(64), 6.0, 0)
        if nsamp:
            w.nsamp = nsamp
        w.bursts = [[Burst(dm=50.0, t0=1000, width=4, snr=24.0, amp=24.0)]]
        return w
    if index == 2:
        w = Workload("cfg2-band4", 2, 1, 2048, 65536, 750.0, -0.09765625, TSAMP, 128.0, 12.0,
                     [(0.0, 0.5, 2048, 1)], _pow2_widths(256), 6.0, 1)
        if nsamp:
            w.nsamp = nsamp
        rng = np.random.default_rng(w.seed)
        w.bursts = [_draw_bursts(rng, 5, w.nchan, w.nsamp, w.fch1, w.foff, w.tsamp, w.std, 50.0, 1000.0,
                                 lambda r: int(r.choice([1, 4, 16, 64])), 8.0, 30.0)]
        return w
    if index == 3:
        w = Workload("cfg3-spotlight", 3, 1, 4096, 1 << 17, 500.0, -0.048828125, TSAMP, 128.0, 10.0,
                     list(_PLAN3), _pow2_widths(512), 7.0, 2)
        if nsamp:
            w.nsamp = nsamp
        rng = np.random.default_rng(w.seed)

        def wfn(r):
            wms = math.exp(r.uniform(math.log(0.5), math.log(40.0)))
            return max(1, int(round(wms * 1e-3 / TSAMP)))
        w.bursts = [_draw_bursts(rng, 20, w.nchan, w.nsamp, w.fch1, w.foff, w.tsamp, w.std, 10.0, 2000.0,
                                 wfn, 7.0, 50.0)]
        return w
    if index == 4:
        w = Workload("cfg4-multibeam", 4, 64, 4096, 1 << 15, 500.0, -0.048828125, TSAMP, 128.0, 10.0,
                     list(_PLAN3), _pow2_widths(512), 7.0, 1000)
        if nsamp:
            w.nsamp = nsamp
        if nbeam:
            w.nbeam = nbeam
        w.bursts = []
        for b in range(w.nbeam):
            rng = np.random.default_rng(w.seed + b)
            n = int(rng.integers(0, 4))
            w.bursts.append(_draw_bursts(rng, n, w.nchan, w.nsamp, w.fch1, w.foff, w.tsamp, w.std, 10.0, 2000.0,
                                         lambda r: int(r.integers(1, 65)), 7.0, 40.0))
        return w
    if index == 5:
        w = Workload("cfg5-rfi", 5, 1, 4096, 1 << 18, 500.0, -0.048828125, TSAMP, 128.0, 10.0,
                     list(_PLAN3), _pow2_widths(1024), 6.0, 4)
        if nsamp:
            w.nsamp = nsamp
        rng = np.random.default_rng(w.seed)

        def wfn(r):
            return max(1, int(round(math.exp(r.uniform(0.0, math.log(512.0))))))
        w.bursts = [_draw_bursts(rng, 50, w.nchan, w.nsamp, w.fch1, w.foff, w.tsamp, w.std, 5.0, 2000.0,
                                 wfn, 6.0, 20.0)]
        nbad = int(round(0.05 * w.nchan))
        chans = np.sort(rng.choice(w.nchan, size=nbad, replace=False))
        for c in chans:
            period = math.exp(rng.uniform(math.log(64.0), math.log(4096.0)))
            phase = rng.uniform(0.0, 2.0 * math.pi)
            w.tones.append((int(c), 40.0, 10.0, float(period), float(phase)))
        for _ in range(200):
            w.spikes.append((int(rng.integers(0, w.nsamp)), int(rng.integers(1, 9)), 30.0))
        return w
    if index == 6:
        # Not a BASELINE.json config: SURVEY.md section 8(f) NEXT-4's second workload, the SPOTLIGHT beam of config 3 observed
        # in uGMRT Band 5 (1060-1460 MHz), 400 MHz over 4096 channels.  Sweeps are about ten times shorter
        # (DM 2000: 2666 samples instead of 44996), so tiles see few distinct delays per channel group.
        w = Workload("cfg6-band5", 6, 1, 4096, 1 << 17, 1460.0, -0.09765625, TSAMP, 128.0, 10.0,
                     list(_PLAN3), _pow2_widths(512), 7.0, 6)
        if nsamp:
            w.nsamp = nsamp
        rng = np.random.default_rng(w.seed)

        def wfn(r):
            wms = math.exp(r.uniform(math.log(0.5), math.log(40.0)))
            return max(1, int(round(wms * 1e-3 / TSAMP)))
        w.bursts = [_draw_bursts(rng, 20, w.nchan, w.nsamp, w.fch1, w.foff, w.tsamp, w.std, 10.0, 2000.0,
                                 wfn, 7.0, 50.0)]
        return w
    raise ValueError("config index must be 1..6")


def generate(w: Workload, beam: int = 0, out: Optional[np.ndarray] = None, nthreads: int = 0) -> np.ndarray:
    """uint8 filterbank [nchan][nsamp] of one beam of workload `w`."""
    lib = _load()
    if out is None:
        out = np.empty((w.nchan, w.nsamp), dtype=np.uint8)
    assert out.dtype == np.uint8 and out.shape == (w.nchan, w.nsamp) and out.flags.c_contiguous
    bl = w.bursts[beam] if beam < len(w.bursts) else []
    barr = (_Burst * max(1, len(bl)))()
    for i, b in enumerate(bl):
        barr[i] = _Burst(b.dm, b.amp, b.t0, b.width, 0)
    tarr = (_Tone * max(1, len(w.tones)))()
    for i, (c, off, amp, per, ph) in enumerate(w.tones):
        tarr[i] = _Tone(off, amp, per, ph, c, 0)
    sarr = (_Spike * max(1, len(w.spikes)))()
    for i, (t0, dur, amp) in enumerate(w.spikes):
        sarr[i] = _Spike(amp, t0, dur, 0)
    rc = lib.synth_filterbank(out.ctypes.data, w.nchan, w.nsamp, w.fch1, w.foff, w.tsamp, w.mean, w.std,
                              w.beam_seed(beam), beam, barr, len(bl), tarr, len(w.tones), sarr, len(w.spikes),
                              nthreads)
    if rc != 0:
        raise RuntimeError("synth_filterbank failed")
    return out


def uniform_bytes(nchan: int, nsamp: int, seed: int) -> np.ndarray:
    """uint8 [nchan][nsamp] of i.i.d. uniform bytes 0..255 (numpy PCG64, seeded): the full-range input of the worst-case
    legs (8-bit telescope data with unmitigated RFI can span the whole range); no signal in it."""
    return np.random.default_rng(seed).integers(0, 256, size=(nchan, nsamp), dtype=np.uint8)


def checksum(buf: np.ndarray) -> int:
    buf = np.ascontiguousarray(buf).view(np.uint8).reshape(-1)
    return int(_load().synth_checksum(buf.ctypes.data, buf.size))
