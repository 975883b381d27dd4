"""Candidate cut-outs (reading H) on the GPU against the oracle: both features bit-exact."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu
TSAMP = 1.31072e-3


@pytest.mark.parametrize("nchan,nsamp,dm0,ddm,ndm,ts,tbin,nt,nf", [
    (4096, 40000, 310.7, 5.38, 256, 9000, 1, 256, 256),      # the classifier's 256 x 256 features on a SPOTLIGHT-shaped beam
    (4096, 40000, 1200.0, 21.5, 64, 2000, 4, 256, 64),       # time-binned, a sweep longer than the window
    (71 * 3, 5003, 37.5, 3.0, 17, -40, 3, 100, 3),           # odd sizes, window starting before the data
    (64, 4096, 0.0, 0.0, 1, 4000, 2, 90, 64),                # DM 0, one row, window running past the end of the data
])
def test_cutout_bit_exact(cuda, api, orc, nchan, nsamp, dm0, ddm, ndm, ts, tbin, nt, nf):
    rs = np.random.default_rng(nchan + ndm)
    x = rs.integers(0, 256, size=(nchan, nsamp), dtype=np.uint8)
    fch1, foff = 500.0, -200.0 / nchan
    dds, dmt = api.cutout(cuda.from_numpy(x).cuda(), fch1, foff, TSAMP, dm0, ddm, ndm, ts, tbin, nt, nf)
    e_dds, e_dmt = orc.cutout(x, fch1, foff, TSAMP, dm0, ddm, ndm, ts, tbin, nt, nf)
    assert np.array_equal(dds.cpu().numpy(), e_dds)
    assert np.array_equal(dmt.cpu().numpy(), e_dmt)


def test_cutout_batch_bit_exact(cuda, api, orc):
    """Many candidates in one call: bins of one and of several samples mixed, two beams, windows hanging off both ends of the
    data, trial and bin counts that are not multiples of the kernel's 32 x 256 tile, a channel count that is not a multiple
    of its 256-channel chunk -- every candidate's two features against the oracle, each at its own index."""
    nbeam, nchan, nsamp = 2, 3 * 160, 30000
    rs = np.random.default_rng(5)
    x = rs.integers(0, 256, size=(nbeam, nchan, nsamp), dtype=np.uint8)
    fch1, foff = 500.0, -200.0 / nchan
    ndm, nt, nf = 75, 300, 32
    cands = [(310.7, 5.38, 9000, 1, 0), (1200.0, 21.5, 2000, 4, 1), (37.5, 3.0, -40, 3, 0), (0.0, 0.0, 29900, 2, 1),
             (5.0, 8.0, 100, 1, 1), (1999.0, 0.5, 12000, 1, 0), (640.0, 60.0, 25000, 7, 0), (88.0, 2.2, 15000, 1, 1)]
    dds, dmt = api.cutout_batch(cuda.from_numpy(x).cuda(), fch1, foff, TSAMP, cands, ndm, nt, nf)
    dds, dmt = dds.cpu().numpy(), dmt.cpu().numpy()
    for k, (dm0, ddm, ts, tbin, b) in enumerate(cands):
        e_dds, e_dmt = orc.cutout(x[b], fch1, foff, TSAMP, dm0, ddm, ndm, ts, tbin, nt, nf)
        assert np.array_equal(dds[k], e_dds), k
        assert np.array_equal(dmt[k], e_dmt), k


def test_cutout_batch_of_more_than_one_launch_and_very_wide_bins(cuda, api, orc):
    """130 candidates (more than one launch's parameter block holds) and a candidate whose bins are too wide for the
    shared-memory kernel (it takes the plain kernel)."""
    nchan, nsamp = 64, 20000
    rs = np.random.default_rng(6)
    x = rs.integers(0, 256, size=(1, nchan, nsamp), dtype=np.uint8)
    fch1, foff = 500.0, -200.0 / nchan
    cands = [(float(10 + 3 * k), 1.0 + 0.1 * k, 50 * k, 1 + (k % 3), 0) for k in range(130)]
    dds, dmt = api.cutout_batch(cuda.from_numpy(x).cuda(), fch1, foff, TSAMP, cands, 9, 40, 8)
    for k in (0, 1, 64, 95, 96, 97, 129):
        e_dds, e_dmt = orc.cutout(x[0], fch1, foff, TSAMP, *cands[k][:2], 9, cands[k][2], cands[k][3], 40, 8)
        assert np.array_equal(dds[k].cpu().numpy(), e_dds) and np.array_equal(dmt[k].cpu().numpy(), e_dmt), k
    wide = [(100.0, 2.0, 0, 400, 0)]
    dds, dmt = api.cutout_batch(cuda.from_numpy(x).cuda(), fch1, foff, TSAMP, wide, 5, 30, 4)
    e_dds, e_dmt = orc.cutout(x[0], fch1, foff, TSAMP, 100.0, 2.0, 5, 0, 400, 30, 4)
    assert np.array_equal(dds[0].cpu().numpy(), e_dds) and np.array_equal(dmt[0].cpu().numpy(), e_dmt)


def test_delta_dm_and_errors(cuda, api, orc):
    assert api.delta_dm(2.6e-3, 400.0, 200.0) == orc.delta_dm(2.6e-3, 400.0, 200.0)
    assert api.delta_dm(2.6e-3, 650.0, 200.0, 0.25) == orc.delta_dm(2.6e-3, 650.0, 200.0, 0.25)
    x = cuda.zeros((64, 1000), dtype=cuda.uint8, device="cuda")
    with pytest.raises(api.SptError) as e:
        api.cutout(x, 500.0, -3.125, TSAMP, 10.0, 1.0, 8, 0, 1, 32, 5)          # 5 bands do not divide 64 channels
    assert e.value.code == api.SPT_ERR_INVALID
    with pytest.raises(api.SptError) as e:
        api.cutout(x, 500.0, 3.125, TSAMP, 10.0, 1.0, 8, 0, 1, 32, 4)           # band not flipped
    assert e.value.code == api.SPT_ERR_UNSUPPORTED
