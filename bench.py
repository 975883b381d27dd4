#!/usr/bin/env python
"""bench.py -- one JSON line per run: throughput of the whole hot path (decimate + dedisperse + single-pulse search
+ candidate-count readback) on seeded synthetic uGMRT-shaped beams.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..6] [--impl reference]
    python bench.py --all-configs            # configs 1-5 (+ the Band-5 workload): rates, RTF, per-kernel fractions
    python bench.py --stream                 # the overlap-save stream front end against the batch rate
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A step = one pass of the whole path over one batch (config 3: one SPOTLIGHT-like beam, 4096 ch x 2^17 samples,
4501 DM trials up to 2000 pc cm^-3).  metric = algorithmic DM-trial x channel x sample additions per second
(BASELINE.json); the JSON line also carries the real-time factor (data seconds per processing second, > 1 is faster
than real time: the reciprocal of the paper's Fig. 9 convention) and the roofline / cpu_baseline objects.
N > 1: beams are sharded over ranks (one process per GPU), no data-path collective (weak scaling).
"""
from __future__ import annotations

import argparse
import csv
import ctypes
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "DM-trial*chan*samples/s and real-time beams per B200 (dedisp + boxcar SPS)"
UNIT = "DM-trial*chan*samples/s"

# `ncu --set full` capture of the dominant kernel, as `ncu -i ... --page raw --csv --print-units base` wrote it
# (profiles/r02_final_raw.md names the commands); roofline.traffic and the shared-memory / issue-slot fractions are read
# from this file, per launch.
NCU_RAW_CSV = os.path.join(ROOT, "profiles", "r03_final_raw.csv")
NCU_STAMP = os.path.join(ROOT, "profiles", "r03_final_raw.stamp.json")   # written by `python bench.py --stamp-ncu` beside the CSV


def sources_sha16():
    """Hash of everything libspt.so is built from: says whether the ncu capture still describes the kernels that run."""
    import hashlib
    from paper_2606_27262_b200 import build
    h = hashlib.sha256()
    for f in sorted(build.SOURCES + build.HEADERS):
        with open(os.path.join(build.CSRC, f), "rb") as fh:
            h.update(f.encode() + b"\0" + fh.read())
    return h.hexdigest()[:16]


def stamp_ncu():
    """Run here (where .git is) after copying a new capture to profiles/: records the commit and the source hash it was made at."""
    import subprocess
    commit = subprocess.run(["git", "rev-parse", "HEAD"], cwd=ROOT, capture_output=True, text=True).stdout.strip()
    dirty = bool(subprocess.run(["git", "status", "--porcelain", "--", "paper_2606_27262_b200/csrc", "include"], cwd=ROOT,
                                capture_output=True, text=True).stdout.strip())
    out = {"csv": os.path.relpath(NCU_RAW_CSV, ROOT), "commit": commit, "sources_dirty_at_stamp": dirty, "sources_sha16": sources_sha16()}
    json.dump(out, open(NCU_STAMP, "w"), indent=1)
    print(json.dumps(out))


def ncu_source():
    """Where roofline.traffic / frac_lds / issue_frac come from, and whether the kernels have changed since (stale)."""
    st = json.load(open(NCU_STAMP)) if os.path.exists(NCU_STAMP) else {}
    return {"csv": os.path.relpath(NCU_RAW_CSV, ROOT), "captured_at_commit": st.get("commit"),
            "captured_sources_sha16": st.get("sources_sha16"), "sources_sha16_now": sources_sha16(),
            "stale": st.get("sources_sha16") != sources_sha16()}
CAND_CAPACITY = {1: 1 << 20, 2: 1 << 24, 3: 1 << 26, 4: 1 << 27, 5: 1 << 29, 6: 1 << 26}


def algorithmic_adds(plan, nchan):
    _, _, _, nout, _ = plan.trial_table()
    return int(nout.astype("int64").sum()) * nchan


def adds_of_range(plan, nchan, rng):
    _, rg, _, nout, _ = plan.trial_table()
    return int(nout[rg == rng].astype("int64").sum()) * nchan


def workload_config(w, world):
    """What was measured -- the same object for our arm and the reference arm (the launch options of our kernels are a
    separate key)."""
    return {"workload": w.name, "nbeam_per_gpu": w.nbeam, "nchan": w.nchan, "nsamp": w.nsamp, "ntrials": w.ntrials,
            "widths": list(w.widths), "threshold": w.threshold,
            "parallelism": f"beams sharded over {world} GPU(s), no collective",
            "l2": "inputs larger than L2 (filterbank %.0f MiB per beam; the DM transform is larger still), no flush needed"
                  % (w.nchan * w.nsamp / 2**20)}


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self._stop_evt = index, [], threading.Event()

    def run(self):
        while not self._stop_evt.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                f = [x.strip() for x in out.strip().split(",")]
                if len(f) >= 7:
                    self.rows.append(f)
            except Exception:
                pass
            self._stop_evt.wait(0.05)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=6)
        sm = sorted(float(r[0]) for r in self.rows if r[0].replace(".", "").isdigit())
        reasons = set()
        for r in self.rows:
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": sm[len(sm) // 2] if sm else None,
                "sm_max_mhz": float(self.rows[0][1]) if self.rows else None,
                "power_w_max": max((float(r[2]) for r in self.rows if r[2].replace(".", "").isdigit()), default=None),
                "samples": len(self.rows), "reasons": sorted(reasons)}


# ---- the oracle on the host cores (cpu_baseline, --impl reference) ---------------------------------------------------
def cpu_info():
    model = "unknown"
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.startswith("model name"):
                model = ln.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    import oracle
    try:
        gxx = subprocess.run(["g++", "--version"], capture_output=True, text=True).stdout.splitlines()[0]
    except Exception:
        gxx = "g++"
    return {"cpu_model": model, "logical_cpus": os.cpu_count(), "compiler": gxx, "flags": " ".join(oracle.CXXFLAGS)}


def set_omp_threads(n):
    """Thread count of the OpenMP runtime the oracle library is linked against (the oracle itself is not touched)."""
    ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))


def oracle_run(w, fb, per_range=None):
    """The oracle, as it stands, over one beam: delay table + decimation + dedispersion + search of every range.
    per_range: {decim: number of trials} evenly spaced over each range (None = every trial).  Returns (seconds, adds, text)."""
    import numpy as np
    import oracle
    oracle.build()
    t_total, adds, picked = 0.0, 0, []
    for (lo, step, ndm, k) in w.ranges:
        n = ndm if per_range is None else max(1, min(ndm, per_range.get(k, 16)))
        idx = np.arange(ndm) if n == ndm else np.linspace(0, ndm - 1, n).astype(int)
        t0 = time.perf_counter()
        dly_all = oracle.delay_table(w.fch1, w.foff, w.nchan, w.tsamp, lo, step, ndm, k)
        dly = dly_all if n == ndm else np.ascontiguousarray(dly_all[idx])
        no = oracle.nout(dly, fb.shape[1], k)
        y = fb if k == 1 else oracle.decimate(fb, k)
        dmt, rowoff = oracle.dedisperse(y, dly, no)
        oracle.search_plane(dmt, rowoff[:-1], no, w.widths, w.threshold)
        t_total += time.perf_counter() - t0
        adds += int(no.astype("int64").sum()) * w.nchan
        picked.append(f"{n} of {ndm} trials (decim {k})")
        del dmt, y
    return t_total, adds, ", ".join(picked)


def sample_sizes(seconds_target):
    """Trials per range of a bounded sample: 96 / 64 / 64 trials take about 2 s on 16 host threads."""
    f = max(0.25, seconds_target / 2.0)
    return {1: int(96 * f), 2: int(64 * f), 4: int(64 * f)}


def cpu_baseline(w, fb, full=True):
    """cpu_baseline object: a FULL oracle run of the workload's beam 0 on all host threads (bounded sample when the workload
    is too large for that: more than ~4e12 adds), plus a single-thread figure on a stated subset."""
    import oracle
    info = cpu_info()
    threads = oracle.num_threads()
    est_adds = sum(ndm for (_, _, ndm, _) in w.ranges) * w.nchan * w.nsamp   # upper bound
    whole = full and est_adds < 6e12
    t, adds, what = oracle_run(w, fb, None if whole else sample_sizes(10.0))
    out = {"value": adds / t, "unit": UNIT, "cores": threads, "kind": "oracle",
           "sample": ("config %d, beam 0, the WHOLE workload: " % w.index if whole else "config %d, beam 0, bounded sample: " % w.index)
                     + what + f"; delay table + decimation + dedispersion + search, {t:.1f} s on {threads} threads",
           "seconds": t, "adds": adds, "whole_workload": whole}
    try:
        set_omp_threads(1)
        t1, adds1, what1 = oracle_run(w, fb, sample_sizes(0.6) if w.index > 1 else None)
        out["single_thread"] = {"value": adds1 / t1, "unit": UNIT, "cores": 1, "sample": what1 + f", {t1:.1f} s", "seconds": t1}
    finally:
        set_omp_threads(threads)
    out.update(info)
    return out


def run_reference(args, rank, world):
    """--impl reference: the oracle on the host cores (rank 0 only), same metric and config; every step is the same bounded
    sample of the workload, sized so that the whole run ends within a few minutes."""
    if rank != 0:
        return
    import oracle
    from paper_2606_27262_b200 import synth
    w = synth.workload(args.config)
    fb = synth.generate(w, beam=0)
    steps, warm = max(1, args.steps), max(0, args.warmup)
    t_sum, adds_sum, what = 0.0, 0.0, ""
    sizes = sample_sizes(min(10.0, 150.0 / (steps + warm)))
    for i in range(warm + steps):
        t, adds, what = oracle_run(w, fb, sizes if w.index > 1 else None)
        if i >= warm:
            t_sum += t
            adds_sum += adds
    rate = adds_sum / t_sum
    threads = oracle.num_threads()
    # whole-workload figures follow from the rate: the sampled trials are evenly spaced over every range
    plan_adds = None
    try:
        import numpy as np
        tot = 0
        for (lo, step, ndm, k) in w.ranges:
            dly = oracle.delay_table(w.fch1, w.foff, w.nchan, w.tsamp, lo, step, ndm, k)
            tot += int(oracle.nout(dly, w.nsamp, k).astype(np.int64).sum()) * w.nchan
        plan_adds = tot * w.nbeam
    except Exception:
        pass
    sample = f"config {w.index}, beam 0: {what}; delay table + decimation + dedispersion + search"
    cb = {"value": rate, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample}
    cb.update(cpu_info())
    line = {"impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
            "warmup": warm, "ms_per_step": 1e3 * t_sum / steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int32", "data": "synthetic", "config": workload_config(w, max(1, args.gpus)),
            "step": {"what": "a bounded sample of the workload (the trials named in cpu_baseline.sample), the same every step; "
                             "ms_per_step is the measured time of that sample, not of the whole workload",
                     "adds_per_step": adds_sum / steps, "adds_whole_workload": plan_adds,
                     "ms_whole_workload_extrapolated": (1e3 * plan_adds / rate) if plan_adds else None},
            "cpu_baseline": cb,
            "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ---- ncu capture -> per-launch counters of the dominant kernel -------------------------------------------------------
def ncu_counters(path=NCU_RAW_CSV, kernel_substr="dedisp_tiled_kernel", pick=0):
    """{metric: value} of the pick-th launch whose kernel name contains kernel_substr, from `ncu --page raw --csv
    --print-units base`.  None when the file is missing."""
    if not os.path.exists(path):
        return None
    rows = list(csv.reader(open(path, newline="")))
    hdr = next((i for i, r in enumerate(rows) if "Kernel Name" in r), None)
    if hdr is None:
        return None
    names = rows[hdr]
    kcol = names.index("Kernel Name")
    hits = [r for r in rows[hdr + 2:] if len(r) == len(names) and kernel_substr in r[kcol]]
    if len(hits) <= pick:
        return None
    out = {"Kernel Name": hits[pick][kcol]}
    for n, v in zip(names, hits[pick]):
        try:
            out[n] = float(v.replace(",", ""))
        except ValueError:
            pass
    return out


# ---- our arm ---------------------------------------------------------------------------------------------------------
class Measurement:
    """One workload on this rank's GPU: buffers, plan, and the timed loops."""

    def __init__(self, args, w, rank, world, data="synthetic"):
        import torch
        from paper_2606_27262_b200 import api, shard, synth
        self.torch, self.api, self.shard = torch, api, shard
        self.args, self.w, self.rank, self.world = args, w, rank, world
        nbeam = w.nbeam
        self.h_fb = torch.empty((nbeam, w.nchan, w.nsamp), dtype=torch.uint8, pin_memory=True)
        hv = self.h_fb.numpy()
        for b, gb in enumerate(shard.beams_of_rank(rank, world, nbeam)):   # every rank brings its own beams (weak scaling)
            if data == "uniform":
                hv[b] = synth.uniform_bytes(w.nchan, w.nsamp, seed=1000 + gb)
            else:
                synth.generate(w, beam=gb, out=hv[b])
        opts = {"profile": 1}
        if args.group:
            opts["group"] = args.group
        if args.dm_tile:
            opts["dm_tile"] = args.dm_tile
        if args.max_entries:
            opts["max_entries"] = args.max_entries
        for kv in args.opt or []:                      # any other plan option, e.g. --opt compact=0
            k, v = kv.split("=")
            opts[k] = int(v)
        self.plan = api.Plan(w.fch1, w.foff, w.nchan, w.tsamp, w.nsamp, w.ranges, w.widths, max_beams=nbeam,
                             cand_capacity=CAND_CAPACITY[w.index], options=opts)
        self.adds_step = algorithmic_adds(self.plan, w.nchan) * nbeam
        self.d_fb = self.h_fb.cuda()
        self.d_dmt = torch.empty((nbeam, self.plan.dmt_elems_per_beam), dtype=torch.int32, device="cuda")
        self.stream = torch.cuda.current_stream()
        self.data_s = nbeam * w.nsamp * w.tsamp

    def capture(self):
        """--graph: spt_search only enqueues, so the step's launches can be captured once into a CUDA graph and replayed (what
        a launch-bound small plan wants); the count readback stays outside."""
        torch = self.torch
        self.plan.set_option("profile", 0)
        self.plan.search(self.d_fb, self.w.threshold, self.d_dmt, self.stream)
        torch.cuda.synchronize()
        self.gstream = torch.cuda.Stream()
        self.graph = torch.cuda.CUDAGraph()
        l0 = self.plan.launches()
        with torch.cuda.graph(self.graph, stream=self.gstream):
            self.plan.search(self.d_fb, self.w.threshold, self.d_dmt, self.gstream)
        self.graph_launches = self.plan.launches() - l0        # kernel nodes of the graph: every replay launches them again
        torch.cuda.synchronize()

    def step(self):
        p, w = self.plan, self.w
        if getattr(self, "graph", None) is not None:
            self.graph.replay()
            return p.candidates_count()
        if self.args.two_calls:             # spt_dedisperse, then spt_single_pulse_search
            p.dedisperse(self.d_fb, self.d_dmt, self.stream)
            p.single_pulse_search(self.d_dmt, w.threshold, self.stream)
        else:                               # spt_search: the same two steps enqueued by one call
            p.search(self.d_fb, w.threshold, self.d_dmt, self.stream)
        return p.candidates_count()         # a5: stream sync + 8-byte readback

    def barrier(self):
        import torch.distributed as dist
        if self.world > 1:
            dist.barrier()
        self.torch.cuda.synchronize()

    def kernel_times(self, nsteps=3):
        """Per-launch device times with the library's event bracketing on (launches then run one after the other)."""
        self.plan.set_option("profile", 1)
        kt = {}
        for _ in range(nsteps):
            self.step()
            for kind, rng, ms in self.plan.kernel_times():
                kt.setdefault((kind, rng), []).append(ms)
        self.plan.set_option("profile", 0)
        return {k: sum(v) / len(v) for k, v in kt.items()}

    def timed(self, steps, warm, local_rank):
        torch = self.torch
        for _ in range(warm):
            self.step()
        self.ktimes = self.kernel_times()
        if self.args.graph:
            self.capture()
        ncand, ovf = self.step()            # profiling off: the timed region runs as a user would run it
        launches0 = self.plan.launches()
        sampler = ClockSampler(local_rank)
        sampler.start()
        self.barrier()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]      # one event between steps: median and min
        e0, e1 = ev[0], ev[-1]
        e0.record(self.stream)
        for i in range(steps):
            ncand, ovf = self.step()
            ev[i + 1].record(self.stream)
        self.barrier()
        clocks = sampler.stop()
        ms_total = self.shard.max_over_ranks(e0.elapsed_time(e1), device="cuda")
        per = sorted(ev[i].elapsed_time(ev[i + 1]) for i in range(steps))
        self.step_ms = {"median": per[len(per) // 2] if len(per) % 2 else 0.5 * (per[len(per) // 2 - 1] + per[len(per) // 2]),
                        "min": per[0], "max": per[-1], "note": "this rank's steps, each between its own pair of CUDA events"}
        nl = self.plan.launches() - launches0
        if getattr(self, "graph", None) is not None:
            nl = steps * self.graph_launches
        return {"ms_total": ms_total, "launches": nl, "clocks": clocks,
                "ncand": ncand, "overflowed": ovf}

    def peak_filter(self):
        """NEXT-1, outside the timed step: 3x3 then 11x11 peak filtering of the step's candidate list."""
        torch = self.torch
        pk0, pk1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ncand, _ = self.plan.candidates_count()
        self.plan.peak_filter((3, 11), self.stream)            # warm-up (allocates the filter's buffers)
        pk0.record(self.stream)
        npeaks = int(self.plan.peak_filter((3, 11), self.stream).size)
        pk1.record(self.stream)
        torch.cuda.synchronize()
        return {"windows": [3, 11], "candidates_in": int(ncand), "peaks_out": npeaks, "ms_with_readback": pk0.elapsed_time(pk1)}

    def e2e(self, steps):
        """The same path from HOST memory through the library's streaming entry points (spt_stream_push / pop): every
        step's filterbank is copied from pinned host memory inside the timed region (the copy of step i+1 overlaps the
        kernels of step i, two batches in flight) and every step's candidate count is read back to the host."""
        p, w = self.plan, self.w
        p.search_host(self.h_fb, w.threshold)
        for _ in range(2):                       # warm-up of the pipeline (allocates both batches' buffers)
            p.stream_push(self.h_fb, w.threshold)
        for _ in range(2):
            p.stream_pop()
        self.barrier()
        t0 = time.perf_counter()
        p.stream_push(self.h_fb, w.threshold)
        ncand = 0
        for i in range(steps):
            if i + 1 < steps:
                p.stream_push(self.h_fb, w.threshold)
            ncand, _ = p.stream_pop()
        self.torch.cuda.synchronize()
        e2e_s = self.shard.max_over_ranks(time.perf_counter() - t0, device="cuda")
        t0 = time.perf_counter()
        nsync = min(steps, 5)
        for _ in range(nsync):                   # and unpipelined (one synchronous spt_search_host per step), for the record
            p.search_host(self.h_fb, w.threshold)
        sync_ms = 1e3 * (time.perf_counter() - t0) / nsync
        # what the host link gives on this box: the same pinned buffer copied alone (the floor of any end-to-end step)
        c0, c1 = self.torch.cuda.Event(enable_timing=True), self.torch.cuda.Event(enable_timing=True)
        self.d_fb.copy_(self.h_fb, non_blocking=True)
        c0.record(self.stream)
        for _ in range(3):
            self.d_fb.copy_(self.h_fb, non_blocking=True)
        c1.record(self.stream)
        self.torch.cuda.synchronize()
        h2d_ms = c0.elapsed_time(c1) / 3
        return {"value": self.adds_step * self.world * steps / e2e_s, "unit": UNIT,
                "h2d_bytes_per_step": int(self.h_fb.numel()), "d2h_bytes_per_step": 8, "ms_per_step": 1e3 * e2e_s / steps,
                "rtf": self.data_s * self.world * steps / e2e_s,
                "api": "spt_stream_push/spt_stream_pop (two batches in flight)",
                "ms_per_step_synchronous_call": sync_ms, "h2d_copy_alone_ms": h2d_ms,
                "h2d_copy_alone_gbs": self.h_fb.numel() / h2d_ms / 1e6}, ncand

    def per_kernel(self, peaks_adds, hbm_gbs):
        """Every kernel of the step against the roofline SURVEY.md 8(d) assigns it: dedispersion vs the measured INT32 add
        peak, decimation and search vs the measured copy bandwidth."""
        w, plan = self.w, self.plan
        _, rg, dec, nout, _ = plan.trial_table()
        out = {}
        for (k, r), ms in sorted(self.ktimes.items()):
            if k == 2:
                adds = adds_of_range(plan, w.nchan, r) * w.nbeam
                out[f"dedisperse_range{r}"] = {"bound": "alu", "adds": adds, "ms": ms, "achieved_tadds": adds / ms / 1e9,
                                               "frac": adds / (ms * 1e-3) / peaks_adds}
            elif k == 1:
                kdec = int(dec[rg == r][0])
                nbytes = (w.nchan * w.nsamp + 2 * w.nchan * (w.nsamp // kdec)) * w.nbeam
                if not any(o.startswith("compact=0") for o in (self.args.opt or [])):
                    nbytes += 3 * w.nchan * (w.nsamp // kdec) * w.nbeam      # the 8-bit copy: uint16 series read, bytes written
                out[f"decimate_range{r}"] = {"bound": "hbm", "bytes": nbytes, "ms": ms, "achieved_gbs": nbytes / ms / 1e6,
                                             "frac": nbytes / ms / 1e6 / hbm_gbs,
                                             "span": "decimation + bounds pass + 8-bit copy of the series"}
            elif k == 3:
                nbytes = 4 * int(nout.astype("int64").sum()) * w.nbeam
                out["single_pulse_search"] = {"bound": "hbm", "bytes": nbytes, "ms": ms, "achieved_gbs": nbytes / ms / 1e6,
                                              "frac": nbytes / ms / 1e6 / hbm_gbs,
                                              "span": "all per-range search launches (statistics pass + boxcar pass over the DM transform)"}
        return out


def measured_peaks(api, torch, local_rank):
    peaks = {}
    pk_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(pk_path):
        peaks = json.load(open(pk_path))
    probe = {}
    for kind, name in ((0, "iadd3"), (1, "imad"), (2, "iadd3+imad"), (3, "lds32"), (4, "lds128")):
        r, _ = api.probe(kind, 3)
        probe[name + "_warp_instr_per_s"] = r
    nsm = torch.cuda.get_device_properties(local_rank).multi_processor_count
    return peaks, probe, nsm


def init_dist(local_rank, world):
    import torch
    import torch.distributed as dist
    # SPT_BENCH_BACKEND=gloo exists for one purpose: running the N > 1 plumbing (sharding, barriers, reductions, rank-0
    # output) on a box with fewer GPUs than ranks; numbers from such a run mean nothing.
    backend = os.environ.get("SPT_BENCH_BACKEND", "nccl")
    if backend != "nccl":
        local_rank %= torch.cuda.device_count()
    torch.cuda.set_device(local_rank)
    if world > 1:
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        else:
            dist.init_process_group(backend)
    return local_rank


def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist

    from paper_2606_27262_b200 import api, build, synth
    build.build()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the path has no CPU fallback")
    local_rank = init_dist(local_rank, world)
    w = synth.workload(args.config)
    nbeam = w.nbeam                        # beams per GPU (weak scaling: every rank gets its own beams)
    warm = max(3, args.warmup)
    steps = max(1, args.steps)
    m = Measurement(args, w, rank, world)
    plan = m.plan
    t = m.timed(steps, warm, local_rank)
    ms_total = t["ms_total"]
    value = m.adds_step * world * steps / (ms_total * 1e-3)
    rtf = m.data_s * world * steps / (ms_total * 1e-3)
    peak_info = m.peak_filter()
    e2e, ncand_e2e = m.e2e(steps)
    assert ncand_e2e == t["ncand"], (ncand_e2e, t["ncand"])
    ncand = m.shard.sum_over_ranks(t["ncand"], device="cuda")

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (dedispersion of range 0) ---------------------------------------------------
    peaks, probe, nsm = measured_peaks(api, torch, local_rank)
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    hbm_gbs = float(peaks.get("hbm_gbs", 6650.0))
    # peak INT32 add rate of the chip = what the two integer pipes can retire together:
    # ALU pipe 64 lanes/SM/clk of IADD3 (two 2-input adds each) + FMA pipe 64 lanes/SM/clk of IMAD (one add each)
    # = 192 adds/SM/clk (B300_MICROARCH.md "Pipe rates"; both rates re-measured by the in-library probes in this run:
    # kind 0 retires 2 counted adds per IADD3, kind 1 one per IMAD).  `peak` is the MEASURED sum.
    iadd3_adds = probe["iadd3_warp_instr_per_s"] * 32      # counted adds/s (= 2 x IADD3 lanes/s)
    imad_adds = probe["imad_warp_instr_per_s"] * 32
    peak_adds = iadd3_adds + imad_adds
    nominal_adds = 192.0 * nsm * sm_max * 1e6
    dom_ms = m.ktimes.get((2, 0))
    dom_adds = adds_of_range(plan, w.nchan, 0) * nbeam
    _, rg, _, nout, _ = plan.trial_table()
    hbm_bytes = (w.nchan * w.nsamp + 4 * int(nout[rg == 0].astype("int64").sum())) * nbeam

    def roofline_of(ms, label):
        achieved = dom_adds / (ms * 1e-3)
        t_alu, t_hbm = dom_adds / peak_adds, hbm_bytes / (hbm_gbs * 1e9)
        return {"bound": "alu", "kernel": "dedisp_tiled_kernel<uint8> (range 0)", "input": label, "achieved": achieved / 1e12,
                "peak": peak_adds / 1e12, "unit": "Tadd/s", "frac": achieved / peak_adds,
                "frac_of_one_add_per_lane_clk": achieved / (128.0 * nsm * sm_max * 1e6),
                "launch_ms": ms, "adds_per_launch": dom_adds,
                "roofline_ms": {"alu": t_alu * 1e3, "hbm": t_hbm * 1e3, "hbm_peak_gbs": hbm_gbs,
                                "hbm_peak_source": "MEASURED_PEAKS.json" if "hbm_gbs" in peaks else "fallback"},
                "algorithmic_hbm_bytes": hbm_bytes}

    roof = None
    if dom_ms:
        roof = roofline_of(dom_ms, "the workload's own data (Gaussian, std %.0f)" % w.std)
        roof["peak_source"] = ("measured in this run by spt_probe: IADD3 (ALU pipe, 2 adds each) %.1f + IMAD (FMA pipe) %.1f Tadd/s; "
                               "nominal 192 adds/SM/clk x %d SMs x %.0f MHz = %.1f. NOTE: frac counts ALGORITHMIC adds; packed "
                               "16-bit lanes and shared pre-sums retire several per instruction, so frac can exceed 1 -- the "
                               "unit that actually bounds the kernel is the shared-memory pipe, see frac_lds" %
                               (iadd3_adds / 1e12, imad_adds / 1e12, nsm, sm_max, nominal_adds / 1e12))
        roof["launch_ms_source"] = ("CUDA events recorded by the library on the launching stream around this kernel, mean of "
                                    "3 steps run just before the timed region (option profile = 1: launches one after the "
                                    "other; the timed region itself lets the DM ranges share the GPU)")
        # the bounds the kernel does obey, from the committed ncu capture (per launch) and the probes of this run
        c = ncu_counters() if (w.index == 3 and nbeam == 1) else None
        lds_peak = probe["lds32_warp_instr_per_s"]          # conflict-free LDS.32: one wavefront per warp instruction
        issue_peak = 4.0 * nsm * sm_max * 1e6               # one warp instruction per clock per SM sub-partition
        roof["lds_peak_per_s"] = lds_peak
        roof["issue_peak_per_s"] = issue_peak
        if c:
            wf = c.get("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum")
            inst = c.get("smsp__inst_executed.sum")
            rd, wr = c.get("dram__bytes_read.sum"), c.get("dram__bytes_write.sum")
            roof["traffic"] = (rd + wr) if (rd is not None and wr is not None) else None
            roof["traffic_source"] = "dram__bytes_read.sum + dram__bytes_write.sum of this kernel, one launch, from the committed ncu capture"
            roof["ncu_source"] = ncu_source()       # "stale": true = the sources changed after the capture: counters of an older kernel
            if wf:
                roof["lds_wavefronts_per_launch"] = wf
                roof["frac_lds"] = wf / (dom_ms * 1e-3) / lds_peak
            if inst:
                roof["inst_executed_per_launch"] = inst
                roof["issue_frac"] = inst / (dom_ms * 1e-3) / issue_peak
            roof["ncu_capture_ms"] = (c.get("gpu__time_duration.sum") or 0.0) / 1e6
        else:
            roof["traffic"] = None
    other = m.per_kernel(peak_adds, hbm_gbs)
    kernels = {f"kind{k}_range{r}": ms for (k, r), ms in sorted(m.ktimes.items())}

    # ---- the same kernels on the data the 16-bit lanes like least: uniform bytes 0..255 (lane capacity at its floor) ----
    worst = None
    if not args.no_worst_case and world == 1:
        del m.d_fb, m.d_dmt
        mw = Measurement(args, w, rank, world, data="uniform")
        for _ in range(3):
            mw.step()
        kt = mw.kernel_times()
        mw.step()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        nws = max(3, min(steps, 10))
        torch.cuda.synchronize()
        e0.record(mw.stream)
        for _ in range(nws):
            mw.step()
        e1.record(mw.stream)
        torch.cuda.synchronize()
        if kt.get((2, 0)):
            worst = roofline_of(kt[(2, 0)], "i.i.d. uniform bytes 0..255: lane capacity 257/decim, the floor")
            worst["ms_per_step"] = e0.elapsed_time(e1) / nws
            worst["value"] = mw.adds_step / (worst["ms_per_step"] * 1e-3)
            worst["kernel_ms"] = {f"kind{k}_range{r}": ms for (k, r), ms in sorted(kt.items())}
        del mw

    cpu = None
    if not args.no_cpu_baseline and world == 1:      # rank 0 at N = 1 only
        cpu = cpu_baseline(w, m.h_fb.numpy()[0])

    # vs_baseline stays null: BASELINE.md holds no published number for this metric on this workload (the paper's figures
    # are whole-pipeline beams per A100); the oracle's rate on the host cores is reported in cpu_baseline, not as a baseline ratio
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warm,
            "ms_per_step": ms_total / steps, "ms_per_step_stats": getattr(m, "step_ms", None),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "int32", "data": "synthetic", "config": workload_config(w, world),
            "launch": {"per_range": [plan.tiling_choice(r) for r in range(len(w.ranges))],     # what the plan actually chose
                       "dm_tile": args.dm_tile or 64,
                       "step_api": "spt_dedisperse + spt_single_pulse_search + spt_candidates_count" if args.two_calls
                                   else ("CUDA graph of spt_search, replayed + spt_candidates_count" if args.graph
                                         else "spt_search + spt_candidates_count"),
                       "dmt_mib_per_beam": plan.dmt_elems_per_beam * 4 / 2**20},
            "rtf": rtf, "realtime_beams": rtf, "candidates": ncand, "overflowed": t["overflowed"],
            "e2e": e2e, "peak_filter": peak_info, "gpu_launches": t["launches"], "clocks": t["clocks"], "kernel_ms": kernels,
            "probe": probe, "roofline": roof, "roofline_worst": worst, "roofline_other": other, "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_all_configs(args, local_rank):
    """Configs 1-5 of BASELINE.json (+ 6, the Band-5 workload) back to back on one GPU: rates, RTF, e2e and every kernel's
    fraction of its roofline, one JSON object (committed as profiles/r02_all_configs.json)."""
    import torch

    from paper_2606_27262_b200 import api, build, synth
    build.build()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    peaks, probe, nsm = measured_peaks(api, torch, local_rank)
    hbm_gbs = float(peaks.get("hbm_gbs", 6650.0))
    peak_adds = (probe["iadd3_warp_instr_per_s"] + probe["imad_warp_instr_per_s"]) * 32
    out = {"metric": METRIC, "unit": UNIT, "n_gpus": 1, "peak_adds_per_s": peak_adds, "hbm_peak_gbs": hbm_gbs, "probe": probe,
           "rtf_convention": "data seconds per processing second (> 1 = faster than real time; reciprocal of PAPER.md:199)",
           "configs": {}}
    for cfg in (1, 2, 3, 4, 5, 6):
        w = synth.workload(cfg)
        steps = {1: 50, 2: 20, 3: 10, 4: 3, 5: 5, 6: 10}[cfg] if args.steps == 30 else args.steps
        m = Measurement(args, w, 0, 1)
        t = m.timed(steps, 3, local_rank)
        ms = t["ms_total"] / steps
        pf = m.peak_filter()
        e2e, _ = m.e2e(steps)
        out["configs"][str(cfg)] = {
            "config": workload_config(w, 1), "steps": steps, "ms_per_step": ms,
            "value": m.adds_step / (ms * 1e-3), "adds_per_step": m.adds_step,
            "rtf": m.data_s / (ms * 1e-3), "realtime_beams": m.data_s / (ms * 1e-3),
            "candidates": t["ncand"], "overflowed": t["overflowed"], "gpu_launches_per_step": t["launches"] / steps,
            "e2e": e2e, "peak_filter": pf, "clocks": t["clocks"],
            "kernels": m.per_kernel(peak_adds, hbm_gbs)}
        del m
        torch.cuda.empty_cache()
    print(json.dumps(out), flush=True)


def run_stream(args, local_rank):
    """NEXT-2 timed: a sustained stream of time-major blocks of 102400 new samples (the paper's 4-block
    segment) on the config-3 geometry -- corner turn + overlap-save push + dedispersion of the new outputs + segment
    search + count readback per push -- against the batch rate on the same GPU."""
    import torch

    from paper_2606_27262_b200 import api, build, synth
    build.build()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    w = synth.workload(3)
    nnew = 102400
    probe_plan = api.Plan(w.fch1, w.foff, w.nchan, w.tsamp, 1 << 17, w.ranges, w.widths)
    hmin, hsearch, gran = probe_plan.segment_info()
    probe_plan.close()
    nsamp = nnew + (hsearch + 511) // 512 * 512
    plan = api.Plan(w.fch1, w.foff, w.nchan, w.tsamp, nsamp, w.ranges, w.widths, max_beams=1, cand_capacity=1 << 26)
    # the stream: consecutive blocks cut from one long synthetic beam, handed over time-major as the telescope's rings do
    nblk = 4
    long_w = synth.workload(3, nsamp=nnew * nblk)
    fb = synth.generate(long_w)
    blocks = [torch.from_numpy(fb[:, i * nnew:(i + 1) * nnew].T.copy()).cuda()[:, None, :] for i in range(nblk)]   # [t][beam][chan]
    d_dmt = torch.empty((1, plan.dmt_elems_per_beam), dtype=torch.int32, device="cuda")
    stream = torch.cuda.current_stream()
    _, _, dec, nout, _ = plan.trial_table()
    adds_new = int(sum(nnew // int(k) for k in dec)) * w.nchan          # algorithmic adds of the NEW outputs of a push
    adds_full = int(nout.astype("int64").sum()) * w.nchan                 # what recomputing the whole buffer costs

    def push(i, incremental=True):
        plan.segment_push(blocks[i % nblk], False, d_dmt, stream, spliced=True, whole_rows=not incremental)
        plan.segment_search(d_dmt, nnew, w.threshold, stream)
        return plan.candidates_count()

    for i in range(4):
        push(i)
    steps = max(4, args.steps if args.steps != 30 else 12)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for i in range(steps):
        ncand, ovf = push(i)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    e0.record(stream)
    for i in range(4):                          # for the record: every push recomputing the whole buffer (whole_rows = 1)
        push(i, incremental=False)
    e1.record(stream)
    torch.cuda.synchronize()
    ms_whole = e0.elapsed_time(e1) / 4
    # the corner turn of one block alone (HBM bound: reads and writes nnew x nchan bytes)
    ct = torch.empty((1, w.nchan, nnew), dtype=torch.uint8, device="cuda")

    def turn(i):
        rc = api.lib().spt_corner_turn(blocks[i % nblk].data_ptr(), 1, nnew, w.nchan, 0, 1, ct.data_ptr(), stream.cuda_stream)
        assert rc == 0, rc

    turn(0)
    e0.record(stream)
    for i in range(10):
        turn(i)
    e1.record(stream)
    torch.cuda.synchronize()
    ms_ct = e0.elapsed_time(e1) / 10
    del ct
    # batch rate on the same GPU for comparison: config 3 as bench.py times it
    mb = Measurement(args, w, 0, 1)
    tb = mb.timed(10, 3, local_rank)
    ms_b = tb["ms_total"] / 10
    out = {"stream": {"nnew": nnew, "history": nsamp - nnew, "min_history_search": hsearch, "nsamp_buffer": nsamp, "pushes": steps,
                      "ms_per_push": ms, "ms_per_push_whole_rows": ms_whole, "corner_turn_ms": ms_ct,
                      "corner_turn_gbs": 2.0 * nnew * w.nchan / ms_ct / 1e6, "rtf": nnew * w.tsamp / (ms * 1e-3), "adds_new_per_push": adds_new,
                      "adds_if_whole_buffer_recomputed": adds_full, "value_new_outputs": adds_new / (ms * 1e-3),
                      "candidates_last_push": ncand, "api": "spt_segment_push + spt_segment_search + spt_candidates_count"},
           "batch": {"workload": w.name, "ms_per_step": ms_b, "rtf": mb.data_s / (ms_b * 1e-3), "value": mb.adds_step / (ms_b * 1e-3)},
           "stream_rtf_over_batch_rtf": (nnew * w.tsamp / (ms * 1e-3)) / (mb.data_s / (ms_b * 1e-3)),
           "stream_rate_over_batch_rate": (adds_new / (ms * 1e-3)) / (mb.adds_step / (ms_b * 1e-3)),
           "note": "a stream yields nnew/decim outputs per trial per nnew samples; the batch call yields nout < nsamp/decim (the "
                   "sweep is lost at the end of its buffer), i.e. %.1f %% fewer additions per second of data: the RTF ratio "
                   "cannot exceed %.3f at equal addition rates" % (
                       100.0 * (1.0 - (mb.adds_step / mb.data_s) / (adds_new / (nnew * w.tsamp))),
                       (mb.adds_step / mb.data_s) / (adds_new / (nnew * w.tsamp))),
           "unit": UNIT}
    print(json.dumps(out), flush=True)


def run_cutouts(args, local_rank):
    """NEXT-4 timed: the classifier's two 256 x 256 features for a batch of 64 candidates on the
    config-3 beam (4096 channels), DM ranges from Eq. 4 as printed -- ms per candidate, against one call per candidate."""
    import numpy as np
    import torch

    from paper_2606_27262_b200 import api, build, synth
    build.build()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    w = synth.workload(3)
    d_fb = torch.from_numpy(synth.generate(w)).cuda()[None]
    rs = np.random.default_rng(0)
    ncand, ndm, nt, nf = 64, 256, 256, 256
    cands = []
    for _ in range(ncand):
        width_s = float(np.exp(rs.uniform(np.log(1e-3), np.log(20e-3))))
        dm0 = float(rs.uniform(20.0, 1900.0))
        ddm = min(dm0, api.delta_dm(width_s, 400.0, 200.0))               # Eq. 4, ratio 0.1
        cands.append((dm0, ddm, int(rs.integers(0, w.nsamp - 70000)), 1, 0))
    stream = torch.cuda.current_stream()

    def timed(fn, reps):
        fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(reps):
            fn()
        e1.record(stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    ms_batch = timed(lambda: api.cutout_batch(d_fb, w.fch1, w.foff, w.tsamp, cands, ndm, nt, nf, stream), 5)
    ms_single = timed(lambda: [api.cutout(d_fb[0], w.fch1, w.foff, w.tsamp, c[0], c[1], ndm, c[2], 1, nt, nf, stream) for c in cands[:8]], 3) / 8
    adds = ncand * (ndm * nt * w.nchan + nt * w.nchan)
    # bytes a candidate must read at least: every channel's window once per 32-trial group is the kernel's traffic; the
    # compulsory figure is one window per channel
    out = {"cutouts": {"ncand": ncand, "shape": [ndm, nt, nf], "nchan": w.nchan, "tbin": 1,
                       "ms_per_candidate_batch": ms_batch / ncand, "ms_per_candidate_single_calls": ms_single,
                       "adds_per_s": adds / (ms_batch * 1e-3), "api": "spt_cutout_batch (one launch of 64)",
                       "mean_ddm": float(np.mean([c[1] for c in cands]))}}
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5, 6])
    ap.add_argument("--group", type=int, default=0)
    ap.add_argument("--dm-tile", type=int, default=0)
    ap.add_argument("--max-entries", type=int, default=0)
    ap.add_argument("--opt", action="append", help="plan option name=value (spt_plan_set_option), may be repeated")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-worst-case", action="store_true")
    ap.add_argument("--all-configs", action="store_true")
    ap.add_argument("--stream", action="store_true")
    ap.add_argument("--cutouts", action="store_true")
    ap.add_argument("--stamp-ncu", action="store_true", help="record the commit and source hash of profiles/r03_final_raw.csv (no GPU)")
    ap.add_argument("--graph", action="store_true", help="replay a CUDA graph of spt_search instead of calling it every step")
    ap.add_argument("--two-calls", action="store_true", help="step = spt_dedisperse + spt_single_pulse_search instead of spt_search")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.stamp_ncu:
        stamp_ncu()
    elif args.impl == "reference":
        run_reference(args, rank, world)
    elif args.all_configs:
        run_all_configs(args, local_rank)
    elif args.stream:
        run_stream(args, local_rank)
    elif args.cutouts:
        run_cutouts(args, local_rank)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
