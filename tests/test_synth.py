"""The seeded input generator: deterministic, thread-count independent, shaped like the configs."""
import math

import numpy as np


def test_deterministic_and_thread_independent(synth):
    w = synth.workload(1)
    a = synth.generate(w, nthreads=1)
    b = synth.generate(w, nthreads=4)
    c = synth.generate(w)
    assert np.array_equal(a, b) and np.array_equal(a, c)
    assert synth.checksum(a) == synth.checksum(b)
    w2 = synth.workload(1)
    w2.seed = 1
    assert synth.checksum(synth.generate(w2)) != synth.checksum(a)


def test_noise_moments_and_quantisation(synth):
    w = synth.workload(1)
    w.bursts = [[]]
    x = synth.generate(w).astype(np.float64)
    n = x.size
    assert abs(x.mean() - 128.0) < 4 * 16 / math.sqrt(n)
    assert abs(x.std() - math.sqrt(16 ** 2 + 1 / 12)) < 0.05         # + uniform quantisation noise
    w.std, w.mean = 100.0, 250.0
    x = synth.generate(w)
    assert x.max() == 255 and x.min() >= 0 and (x == 255).mean() > 0.3    # clipped, not wrapped


def test_burst_follows_the_sweep(synth):
    w = synth.workload(1)
    with_b = synth.generate(w).astype(np.int32)
    w0 = synth.workload(1)
    w0.bursts = [[]]
    diff = with_b - synth.generate(w0).astype(np.int32)
    b = w.bursts[0][0]
    for c in (0, 1, 31, 63):
        on = np.nonzero(diff[c])[0]
        s = synth.sweep_samples(b.dm, w.fch1, w.foff, c, w.tsamp)
        assert on.min() == b.t0 + s and on.max() == b.t0 + s + b.width - 1
        assert np.all(diff[c][on] == 24)
    assert synth.sweep_samples(b.dm, w.fch1, w.foff, 0, w.tsamp) == 0
    assert synth.sweep_samples(50.0, 500.0, -3.125, 63, w.tsamp) == 1089


def test_config_shapes_match_baseline_json(synth):
    shapes = {1: (1, 64, 4096, 101, 7, 6.0), 2: (1, 2048, 65536, 2048, 9, 6.0),
              3: (1, 4096, 1 << 17, 4501, 10, 7.0), 4: (64, 4096, 1 << 15, 4501, 10, 7.0),
              5: (1, 4096, 1 << 18, 4501, 11, 6.0)}
    for i, (nb, nc, ns, nt, nw, thr) in shapes.items():
        w = synth.workload(i)
        assert (w.nbeam, w.nchan, w.nsamp, w.ntrials, len(w.widths), w.threshold) == (nb, nc, ns, nt, nw, thr)
        assert w.tsamp == 1.31072e-3 and w.foff < 0
        assert abs((w.fch1 + w.nchan * w.foff) - {1: 300, 2: 550, 3: 300, 4: 300, 5: 300}[i]) < 1e-9
        assert len(w.bursts) == nb
    w6 = synth.workload(6)                          # NEXT-4's Band-5 workload: cfg 3's shape at 1060-1460 MHz
    assert (w6.nbeam, w6.nchan, w6.nsamp, w6.ntrials, w6.fch1) == (1, 4096, 1 << 17, 4501, 1460.0)
    assert abs(w6.fch1 + w6.nchan * w6.foff - 1060.0) < 1e-9 and len(w6.bursts[0]) == 20
    w3, w4, w5 = synth.workload(3), synth.workload(4), synth.workload(5)
    assert len(w3.bursts[0]) == 20 and all(1 <= b.width <= 31 for b in w3.bursts[0])
    assert all(0 <= len(bl) <= 3 for bl in w4.bursts) and any(b.truncated for bl in w4.bursts for b in bl)
    assert len(w5.tones) == 205 and len(w5.spikes) == 200 and len(w5.bursts[0]) == 50
    assert w4.beam_seed(7) == 1007


def test_cfg5_rfi_terms_present(synth):
    w = synth.workload(5, nsamp=4096)
    w.nchan = 64
    w.tones = [(3, 40.0, 10.0, 100.0, 0.0)]
    w.spikes = [(1000, 4, 30.0)]
    w.bursts = [[]]
    x = synth.generate(w).astype(np.float64)
    assert abs(x[3].mean() - 168.0) < 1.0 and abs(x[2].mean() - 128.0) < 1.0
    assert np.all(x[:, 1000:1004].mean(axis=0) > 150) and x[:, 1004].mean() < 135
