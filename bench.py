#!/usr/bin/env python
"""bench.py -- one JSON line per run: throughput of the whole hot path (decimate + dedisperse + single-pulse search
+ candidate-count readback) on seeded synthetic uGMRT-shaped beams.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A step = one pass of the whole path over one batch (config 3: one SPOTLIGHT-like beam, 4096 ch x 2^17 samples,
4501 DM trials up to 2000 pc cm^-3).  metric = algorithmic DM-trial x channel x sample additions per second
(BASELINE.json); the JSON line also carries the real-time factor (data seconds per processing second, > 1 is faster
than real time: the reciprocal of the paper's Fig. 9 convention) and the roofline / cpu_baseline objects.
N > 1: beams are sharded over ranks (one process per GPU), no data-path collective (weak scaling).
"""
from __future__ import annotations

import argparse
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

# DRAM bytes per launch of the dominant kernel (dedisp_tiled, range 0 of config 3) from the committed
# `ncu --set full` capture (profiles/): dram__bytes_read.sum + dram__bytes_write.sum.
NCU_TRAFFIC_BYTES = {3: 2257476000}   # profiles/r01_final_summary.md: 0.83 GB read + 1.43 GB written


def algorithmic_adds(plan, nchan):
    _, _, _, nout, _ = plan.trial_table()
    return int(nout.astype("int64").sum()) * nchan


def adds_of_range(plan, nchan, rng):
    _, rg, _, nout, _ = plan.trial_table()
    return int(nout[rg == rng].astype("int64").sum()) * nchan


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


def oracle_sample(w, fb, seconds_target=10.0):
    """The oracle, as it stands, on a bounded sample of the same workload: a few trials of every range dedispersed
    and searched on the host cores.  Returns (adds per second, cores, description)."""
    import numpy as np
    import oracle
    oracle.build()
    cores = oracle.num_threads()
    # 96 / 64 / 64 trials of the three ranges take about 2 s on 16 host threads; scaled to the target
    f = max(0.25, seconds_target / 2.0)
    per_range = {1: int(96 * f), 2: int(64 * f), 4: int(64 * f)}
    t_total, adds, picked = 0.0, 0, []
    for (lo, step, ndm, k) in w.ranges:
        n = min(ndm, per_range.get(k, 16))
        idx = np.linspace(0, ndm - 1, n).astype(int)
        t0 = time.perf_counter()
        dly_all = oracle.delay_table(w.fch1, w.foff, w.nchan, w.tsamp, lo, step, ndm, k)
        dly = np.ascontiguousarray(dly_all[idx])
        no = oracle.nout(dly, fb.shape[1], k)
        y = fb if k == 1 else oracle.decimate(fb, k)
        dmt, rowoff = oracle.dedisperse(y, dly, no)
        oracle.search_plane(dmt, rowoff[:-1], no, w.widths, w.threshold)
        t_total += time.perf_counter() - t0
        adds += int(no.astype("int64").sum()) * w.nchan
        picked.append(f"{n} of {ndm} trials (decim {k})")
    desc = "config %d, beam 0: " % w.index + ", ".join(picked) + \
        f"; delay table + decimation + dedispersion + search, {t_total:.1f} s"
    return adds / t_total, cores, desc, t_total, adds


def run_reference(args, rank, world):
    """--impl reference: the oracle on the host cores (rank 0 only), same metric and config."""
    if rank != 0:
        return
    import numpy as np
    from paper_2606_27262_b200 import synth
    w = synth.workload(args.config)
    fb = synth.generate(w, beam=0)
    steps, warm = args.steps, args.warmup
    rate, cores, sample = 0.0, 1, ""
    t_sum, adds_sum = 0.0, 0.0
    for i in range(warm + steps):
        # each step is the same bounded sample, sized so that the whole run ends within a few minutes
        r, cores, sample, t, adds = oracle_sample(w, fb, seconds_target=min(10.0, 150.0 / (steps + warm)))
        if i >= warm:
            t_sum += t
            adds_sum += adds
    rate = adds_sum / t_sum
    line = {"impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
            "warmup": warm, "ms_per_step": 1e3 * t_sum / steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int32", "data": "synthetic",
            "config": {"workload": w.name, "nbeam": 1, "nchan": w.nchan, "nsamp": w.nsamp, "ntrials": w.ntrials,
                       "step": "bounded sample of the workload (see cpu_baseline.sample)"},
            "cpu_baseline": {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def run_ours(args, rank, world, local_rank):
    import numpy as np
    import torch
    import torch.distributed as dist

    from paper_2606_27262_b200 import api, build, shard, synth
    build.build()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the path has no CPU fallback")
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

    w = synth.workload(args.config)
    nbeam = w.nbeam                        # beams per GPU (weak scaling: every rank gets its own beams)
    warm = max(3, args.warmup)
    steps = max(1, args.steps)

    # seeded synthetic input of this rank, in pinned host memory (the e2e leg copies from it every step)
    h_fb = torch.empty((nbeam, w.nchan, w.nsamp), dtype=torch.uint8, pin_memory=True)
    hv = h_fb.numpy()
    for b, gb in enumerate(shard.beams_of_rank(rank, world, nbeam)):   # every rank brings its own beams (weak scaling)
        synth.generate(w, beam=gb, out=hv[b])
    cap = {1: 1 << 20, 2: 1 << 24, 3: 1 << 26, 4: 1 << 27, 5: 1 << 29, 6: 1 << 26}[w.index]
    opts = {"profile": 1}
    if args.group:
        opts["group"] = args.group
    if args.dm_tile:
        opts["dm_tile"] = args.dm_tile
    plan = api.Plan(w.fch1, w.foff, w.nchan, w.tsamp, w.nsamp, w.ranges, w.widths, max_beams=nbeam,
                    cand_capacity=cap, options=opts)
    adds_step = algorithmic_adds(plan, w.nchan) * nbeam
    d_fb = h_fb.cuda()
    d_dmt = torch.empty((nbeam, plan.dmt_elems_per_beam), dtype=torch.int32, device="cuda")
    stream = torch.cuda.current_stream()

    def step():
        if args.two_calls:                  # spt_dedisperse, then spt_single_pulse_search
            plan.dedisperse(d_fb, d_dmt, stream)
            plan.single_pulse_search(d_dmt, w.threshold, stream)
        else:                               # spt_search: the same two steps enqueued by one call
            plan.search(d_fb, w.threshold, d_dmt, stream)
        return plan.candidates_count()      # a5: stream sync + 8-byte readback

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(warm):
        ncand, ovf = step()
    # per-kernel device times: a few steps with the library's event bracketing on (launches then run one after the other)
    ktimes = {}
    for _ in range(3):
        step()
        for kind, rng, ms in plan.kernel_times():
            ktimes.setdefault((kind, rng), []).append(ms)
    plan.set_option("profile", 0)            # the timed region runs as a user would run it
    step()
    launches0 = plan.launches()
    sampler = ClockSampler(local_rank)
    sampler.start()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        ncand, ovf = step()
    e1.record(stream)
    barrier()
    clocks = sampler.stop()
    ms_total = e0.elapsed_time(e1)
    launches = plan.launches() - launches0
    ms_total = shard.max_over_ranks(ms_total, device="cuda")
    value = adds_step * world * steps / (ms_total * 1e-3)
    data_s = nbeam * w.nsamp * w.tsamp
    rtf = data_s * world * steps / (ms_total * 1e-3)

    # ---- NEXT-1, outside the timed step: 3x3 then 11x11 peak filtering of the step's candidate list ------
    pk0, pk1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    plan.peak_filter((3, 11), stream)                      # warm-up (allocates the lookup plane)
    pk0.record(stream)
    npeaks = int(plan.peak_filter((3, 11), stream).size)
    pk1.record(stream)
    torch.cuda.synchronize()
    peak_info = {"windows": [3, 11], "candidates_in": int(ncand), "peaks_out": npeaks,
                 "ms_with_readback": pk0.elapsed_time(pk1)}

    # ---- e2e: the same path from HOST memory through the library's streaming entry points (spt_stream_push / pop): every
    # step's filterbank is copied from pinned host memory inside the timed region (the copy of step i+1 overlaps the kernels
    # of step i, two batches in flight) and every step's candidate count is read back to the host ---------------------
    plan.search_host(h_fb, w.threshold)
    for _ in range(2):                       # warm-up of the pipeline (allocates both batches' buffers)
        plan.stream_push(h_fb, w.threshold)
    for _ in range(2):
        plan.stream_pop()
    barrier()
    t0 = time.perf_counter()
    plan.stream_push(h_fb, w.threshold)
    for i in range(steps):
        if i + 1 < steps:
            plan.stream_push(h_fb, w.threshold)
        ncand_e2e, _ = plan.stream_pop()
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    assert ncand_e2e == ncand, (ncand_e2e, ncand)
    e2e_s = shard.max_over_ranks(e2e_s, device="cuda")
    ncand = shard.sum_over_ranks(ncand, device="cuda")
    # and unpipelined (one synchronous spt_search_host per step), for the record
    t0 = time.perf_counter()
    for _ in range(min(steps, 5)):
        plan.search_host(h_fb, w.threshold)
    e2e_sync_ms = 1e3 * (time.perf_counter() - t0) / min(steps, 5)
    e2e_value = adds_step * world * steps / e2e_s

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (dedispersion of range 0) ---------------------------------------------------
    peaks = {}
    pk_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(pk_path):
        peaks = json.load(open(pk_path))
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    nsm = torch.cuda.get_device_properties(local_rank).multi_processor_count
    probe = {}
    for kind, name in ((0, "iadd3"), (1, "imad"), (2, "iadd3+imad"), (3, "lds32"), (4, "lds128")):
        r, _ = api.probe(kind, 3)
        probe[name + "_warp_instr_per_s"] = r
    # peak INT32 add rate of the chip = what the two integer pipes can retire together:
    # ALU pipe 64 lanes/SM/clk of IADD3 (two 2-input adds each) + FMA pipe 64 lanes/SM/clk of IMAD (one add each)
    # = 192 adds/SM/clk (B300_MICROARCH.md "Pipe rates"; both rates re-measured by the in-library probes in this run:
    # kind 0 retires 2 counted adds per IADD3, kind 1 one per IMAD).  `peak` is the MEASURED sum.
    iadd3_adds = probe["iadd3_warp_instr_per_s"] * 32      # counted adds/s (= 2 x IADD3 lanes/s)
    imad_adds = probe["imad_warp_instr_per_s"] * 32
    peak_adds = iadd3_adds + imad_adds
    nominal_adds = 192.0 * nsm * sm_max * 1e6
    dom = ktimes.get((2, 0), [])
    dom_ms = sum(dom) / len(dom) if dom else None
    dom_adds = adds_of_range(plan, w.nchan, 0) * nbeam
    roof = None
    if dom_ms:
        achieved = dom_adds / (dom_ms * 1e-3)
        # the other leg of north_star's roofline: compulsory HBM bytes of the launch at the measured copy bandwidth
        _, rg, _, nout, _ = plan.trial_table()
        hbm_bytes = (w.nchan * w.nsamp + 4 * int(nout[rg == 0].astype("int64").sum())) * nbeam
        hbm_gbs = float(peaks.get("hbm_gbs", 6650.0))
        t_alu, t_hbm = dom_adds / peak_adds, hbm_bytes / (hbm_gbs * 1e9)
        roof = {"bound": "alu", "kernel": "dedisp_tiled_kernel<uint8> (range 0)", "achieved": achieved / 1e12,
                "peak": peak_adds / 1e12, "unit": "Tadd/s", "frac": achieved / peak_adds,
                "peak_source": "measured in this run by spt_probe: IADD3 (ALU pipe, 2 adds each) %.1f + IMAD (FMA pipe) %.1f Tadd/s; "
                               "nominal 192 adds/SM/clk x %d SMs x %.0f MHz = %.1f" %
                               (iadd3_adds / 1e12, imad_adds / 1e12, nsm, sm_max, nominal_adds / 1e12),
                "frac_of_one_add_per_lane_clk": achieved / (128.0 * nsm * sm_max * 1e6),
                "launch_ms": dom_ms, "adds_per_launch": dom_adds,
                "launch_ms_source": "CUDA events recorded by the library on the launching stream around this kernel, mean of "
                                    "3 steps run just before the timed region (option profile = 1: launches one after the "
                                    "other; the timed region itself lets the DM ranges share the GPU)",
                "roofline_ms": {"alu": t_alu * 1e3, "hbm": t_hbm * 1e3, "hbm_peak_gbs": hbm_gbs,
                                "hbm_peak_source": "MEASURED_PEAKS.json" if "hbm_gbs" in peaks else "fallback"},
                "algorithmic_hbm_bytes": hbm_bytes,
                "traffic": NCU_TRAFFIC_BYTES.get(w.index)}
    kernels = {f"kind{k}_range{r}": sum(v) / len(v) for (k, r), v in sorted(ktimes.items())}
    # SURVEY.md 8(d), metric (3): the HBM-bound kernels against the copy bandwidth (a2: bytes = raw in + uint16 out per
    # decimated range, its timed span includes the pass that finds the bounds of the series; a4: the DM transform read once)
    hbm_gbs = float(peaks.get("hbm_gbs", 6650.0))
    other = {}
    _, rg_all, dec_all, nout_all, _ = plan.trial_table()
    for (k, r), v in sorted(ktimes.items()):
        ms = sum(v) / len(v)
        if k == 1:
            kdec = int(dec_all[rg_all == r][0])
            nbytes = (w.nchan * w.nsamp + 2 * w.nchan * (w.nsamp // kdec)) * nbeam
            other[f"decimate_range{r}"] = {"bound": "hbm", "bytes": nbytes, "ms": ms, "achieved_gbs": nbytes / ms / 1e6,
                                           "frac": nbytes / ms / 1e6 / hbm_gbs}
        elif k == 3:
            nbytes = 4 * int(nout_all.astype("int64").sum()) * nbeam
            other["single_pulse_search"] = {"bound": "hbm", "bytes": nbytes, "ms": ms, "achieved_gbs": nbytes / ms / 1e6,
                                            "frac": nbytes / ms / 1e6 / hbm_gbs}

    cpu = None
    if not args.no_cpu_baseline and world == 1:      # rank 0 at N = 1 only
        rate, cores, sample, _, _ = oracle_sample(w, hv[0])
        cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warm,
            "ms_per_step": ms_total / steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "int32", "data": "synthetic",
            "config": {"workload": w.name, "nbeam_per_gpu": nbeam, "nchan": w.nchan, "nsamp": w.nsamp,
                       "ntrials": plan.ntrials, "widths": w.widths, "threshold": w.threshold,
                       "parallelism": f"beams sharded over {world} GPU(s), no collective",
                       "l2": "inputs larger than L2 (filterbank %.0f MiB, DM transform %.0f MiB per beam)" %
                             (w.nchan * w.nsamp / 2**20, plan.dmt_elems_per_beam * 4 / 2**20),
                       "group": args.group or 8, "dm_tile": args.dm_tile or 64,
                       "step_api": "spt_dedisperse + spt_single_pulse_search + spt_candidates_count" if args.two_calls
                                   else "spt_search + spt_candidates_count"},
            "rtf": rtf, "realtime_beams": rtf, "candidates": ncand, "overflowed": ovf,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h_fb.numel()),
                    "d2h_bytes_per_step": 8, "ms_per_step": 1e3 * e2e_s / steps,
                    "rtf": data_s * world * steps / e2e_s, "api": "spt_stream_push/spt_stream_pop (two batches in flight)",
                    "ms_per_step_synchronous_call": e2e_sync_ms},
            "peak_filter": peak_info, "gpu_launches": launches, "clocks": clocks, "kernel_ms": kernels, "probe": probe,
            "roofline": roof, "roofline_other": other, "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5, 6])
    ap.add_argument("--group", type=int, default=0)
    ap.add_argument("--dm-tile", type=int, default=0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--two-calls", action="store_true", help="step = spt_dedisperse + spt_single_pulse_search instead of spt_search")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
