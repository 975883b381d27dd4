"""CPU-side checks of the C ABI: the library builds and loads, exports every symbol include/spt.h declares,
validates arguments, and its host plan (trial list, delay table, nout, offsets, tiling tables) agrees bit for bit
with the oracle.  No compute call is made here; the parity tests proper are the -m gpu tests."""
import ctypes
import os
import re

import numpy as np
import pytest

from helpers import check_plan_against_oracle, make_plan

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "spt.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(spt_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(api):
    L = ctypes.CDLL(api.LIB_PATH)
    names = declared_symbols()
    assert len(names) >= 20
    for n in names:
        assert hasattr(L, n), f"libspt.so does not export {n}"
    assert set(api.SYMBOLS) == set(names), "python binding and header disagree"


def test_strerror_and_argument_validation(api):
    L = api.lib()
    assert L.spt_strerror(0) == b"ok"
    for code in range(-6, 0):
        assert L.spt_strerror(code) not in (b"ok", b"unknown error")
    good = dict(fch1=500.0, foff=-3.125, nchan=64, tsamp=1.31072e-3, nsamp=4096, ranges=[(0.0, 1.0, 101, 1)],
                widths=[1, 2, 4])
    api.Plan(**good).close()
    bad = [
        (dict(foff=3.125), api.SPT_ERR_UNSUPPORTED),                 # band not flipped
        (dict(foff=0.0), api.SPT_ERR_UNSUPPORTED),
        (dict(nchan=0), api.SPT_ERR_INVALID),
        (dict(nsamp=0), api.SPT_ERR_INVALID),
        (dict(widths=[1, 1, 2]), api.SPT_ERR_INVALID),
        (dict(widths=[0, 1]), api.SPT_ERR_INVALID),
        (dict(widths=[4, 2]), api.SPT_ERR_INVALID),
        (dict(ranges=[(0.0, 0.0, 10, 1)]), api.SPT_ERR_INVALID),
        (dict(ranges=[(0.0, 1.0, 0, 1)]), api.SPT_ERR_INVALID),
        (dict(ranges=[(0.0, 1.0, 10, 3)]), api.SPT_ERR_UNSUPPORTED),  # decimation must be a power of two
        (dict(ranges=[(0.0, 1.0, 10, 128)]), api.SPT_ERR_UNSUPPORTED),
        (dict(nchan=200, foff=-3.125), api.SPT_ERR_INVALID),          # lowest channel frequency <= 0
        (dict(widths=[1, 8192]), api.SPT_ERR_UNSUPPORTED),
    ]
    for change, code in bad:
        kw = dict(good)
        kw.update(change)
        with pytest.raises(api.SptError) as e:
            api.Plan(**kw)
        assert e.value.code == code, (change, e.value.code)


def test_sum_of_squares_bound(api):
    """Sxx of a row is a 64-bit integer: a plan whose worst row floor(nsamp/k) * (nchan*255*k)^2 reaches 2^64 is refused at
    creation (it would wrap silently on both sides of the parity test), the largest one below the bound is accepted."""
    nchan, k = 4096, 64
    xmax = nchan * 255 * k                                     # largest sample of the decimated DM transform
    n_ok = (2**64 - 1) // (xmax * xmax)                        # longest row whose worst-case Sxx still fits
    assert n_ok * xmax * xmax < 2**64 <= (n_ok + 1) * xmax * xmax
    kw = dict(fch1=500.0, foff=-0.048828125, nchan=nchan, tsamp=1.31072e-3, ranges=[(0.0, 1.0, 2, k)], widths=[1, 2, 4])
    api.Plan(nsamp=n_ok * k + k - 1, **kw).close()             # floor(nsamp/k) == n_ok
    with pytest.raises(api.SptError) as e:
        api.Plan(nsamp=(n_ok + 1) * k, **kw)
    assert e.value.code == api.SPT_ERR_UNSUPPORTED
    # the BASELINE configs are far below it (config 5, decimation 4: 2^16 * (4096*255*4)^2 = 1.1e18)
    assert (2**18 // 4) * (4096 * 255 * 4) ** 2 < 2**60


def test_options_and_state_errors(api):
    p = api.Plan(500.0, -3.125, 64, 1.31072e-3, 4096, [(0.0, 1.0, 101, 1)], [1, 2, 4])
    p.set_option("group", 8)
    p.set_option("dm_tile", 32)
    p.set_option("dedisp_kernel", 1)
    p.set_option("skew", 0)
    p.set_option("max_entries", 12)
    p.set_option("compact", 0)
    p.set_option("tile_words", 256)
    for name, v in (("group", 3), ("dm_tile", 48), ("dedisp_kernel", 2), ("skew", 2), ("max_entries", 10), ("compact", 2), ("tile_words", 192), ("nonsense", 1)):
        with pytest.raises(api.SptError) as e:
            p.set_option(name, v)
        assert e.value.code == api.SPT_ERR_INVALID
    with pytest.raises(api.SptError) as e:
        p.candidates_count()          # nothing searched yet
    assert e.value.code == api.SPT_ERR_STATE
    with pytest.raises(api.SptError) as e:
        p.trial(101)
    assert e.value.code == api.SPT_ERR_SHAPE


@pytest.mark.parametrize("cfg,stride", [(1, 1), (2, 97), (3, 211)])
def test_plan_matches_oracle(api, orc, synth, cfg, stride):
    w = synth.workload(cfg)
    p = make_plan(api, w)
    check_plan_against_oracle(orc, p, w, stride=stride)


def test_plan_cfg4_zero_length_trials(api, orc, synth):
    """cfg 4 (nsamp = 2^15): trials whose sweep is longer than the data are legal and empty (reading B3)."""
    w = synth.workload(4)
    p = make_plan(api, w, nbeam=1)
    _, _, _, nout, off = p.trial_table()
    assert int((nout == 0).sum()) == 544
    check_plan_against_oracle(orc, p, w, stride=499)


@pytest.mark.parametrize("group,dm_tile,skew,max_ent", [(1, 64, 1, 8), (2, 64, 1, 8), (4, 64, 1, 8), (8, 64, 1, 8), (4, 32, 1, 8),
                                                        (8, 64, 0, 8), (12, 64, 1, 12), (16, 64, 1, 12), (16, 64, 1, 16),
                                                        (16, 32, 0, 16), (8, 64, 1, -8), (16, 64, 1, -12), (0, 64, 1, 0)])
def test_tiling_tables_reproduce_the_delay_table(api, synth, group, dm_tile, skew, max_ent):
    """Host logic of the tiled kernel: the (skew, window, variant, offset) factorisation gives back every delay."""
    for cfg, stride in ((1, 1), (3, 173)):
        w = synth.workload(cfg)
        opts = {"group": group, "dm_tile": dm_tile, "skew": skew, "max_entries": abs(max_ent)}
        if max_ent < 0:
            opts["tile_words"] = 224                      # a negative cap in the parameter list: the narrow time tile
        if group == 0:
            opts = {}                                     # everything chosen by the cost model
        p = make_plan(api, w, options=opts)
        for d in list(range(0, p.ntrials, stride)) + [p.ntrials - 1]:
            assert np.array_equal(p.tiling_delays(d), p.delays(d)), (cfg, d)
        for r in range(len(w.ranges)):
            info = p.tiling_info(r)
            assert info["max_stage_words"] <= 227 * 1024 // 4
            assert info["ngroups"] >= info["ntiles_dm"] * ((w.nchan + max(group, 16) - 1) // max(group, 16))
            assert info["nvariants"] <= 16 * info["ngroups"]


def test_tiling_odd_shapes(api):
    """Channel count not a multiple of the group size, trial count not a multiple of the DM tile."""
    p = api.Plan(420.0, -1.0, 71, 1.31072e-3, 5000, [(3.0, 0.7, 77, 1), (60.0, 1.1, 41, 2), (100.0, 2.0, 5, 8)],
                 [1, 3, 7], options={"group": 4})
    for d in range(p.ntrials):
        assert np.array_equal(p.tiling_delays(d), p.delays(d)), d
    for r in range(3):
        p.tiling_info(r)              # includes the bounds check of every shared-memory address the tables lead to


@pytest.mark.parametrize("opts", [{}, {"max_entries": 12}, {"max_entries": 12, "tile_words": 224}, {"max_entries": 16}])
def test_tiling_large_decimation(api, opts):
    """Ranges decimated by 32 and 64 (their uint16 rows are the widest a stage holds) with the 12- and 16-entry caps: the
    plan builds, both table sets -- the uint16 series' and the 8-bit copy's, rebuilt to share one kernel instance -- pass the
    bounds check, and the factorised tables give back every delay.  (If the shared instance cannot be built for the uint16
    tables the range falls back to its own tables without an 8-bit copy; the plan still has to work.)"""
    nchan = 1024
    p = api.Plan(500.0, -200.0 / nchan, nchan, 1.31072e-3, 1 << 17, [(0.0, 0.2, 64, 1), (100.0, 4.0, 130, 32), (700.0, 8.0, 70, 64)],
                 [1, 2, 4], options=opts)
    for d in list(range(0, p.ntrials, 7)) + [p.ntrials - 1]:
        assert np.array_equal(p.tiling_delays(d), p.delays(d)), d
    for r in range(3):
        info = p.tiling_info(r)
        assert info["max_stage_words"] <= 227 * 1024 // 4
    p.close()


def test_device_calls_fail_loudly_without_gpu(api):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    r, ms = ctypes.c_double(), ctypes.c_double()
    assert api.lib().spt_probe(0, 1, ctypes.byref(r), ctypes.byref(ms)) == api.SPT_ERR_CUDA
    p = api.Plan(500.0, -3.125, 64, 1.31072e-3, 4096, [(0.0, 1.0, 101, 1)], [1, 2, 4])
    fb = np.zeros((1, 64, 4096), dtype=np.uint8)
    with pytest.raises(api.SptError) as e:
        p.search_host(fb, 6.0)
    assert e.value.code == api.SPT_ERR_CUDA       # no CPU fallback
