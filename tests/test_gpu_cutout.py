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
