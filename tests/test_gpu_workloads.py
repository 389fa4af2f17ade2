"""The CUDA input generators (workloads/fill.cu) against the direct host fill (workloads/gen.cpp):
same recipe, <= 1 fp32 ulp per value on 32^3 and 48^3; the device brick cut
equals the host cut bit for bit.  Input generation only -- none of the traced method is involved."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("N,M,kmax", [(32, 64, 8.0), (48, 512, 12.0)])
def test_turbulence_fill_matches_host(wl, N, M, kmax):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    ref = wl.turb_field_cpu(N, M, 1.0, kmax)
    fld, dev = wl.turb_field_cuda(N, M, 1.0, kmax, zchunk=20)      # ragged chunks: 20+20+8
    a = fld.data.view(np.int32).astype(np.int64)
    b = ref.data.view(np.int32).astype(np.int64)
    same_sign = (a >= 0) == (b >= 0)
    ulp = np.where(same_sign, np.abs(a - b), np.abs(fld.data - ref.data) / np.float32(1.4e-45))
    assert ulp.max() <= 1, "max ulp distance %g" % ulp.max()
    assert np.mean(ulp == 0) > 0.99
    rms = np.sqrt(np.mean(np.sum(fld.data.astype(np.float64) ** 2, axis=-1)))
    assert abs(rms - 1.0) < 1e-6
    assert np.array_equal(dev.cpu().numpy(), fld.data)


def test_device_brick_cut_matches_host(wl):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    fld = wl.turb_field_cpu(31, 16, 1.0, 4.0)
    dev = torch.from_numpy(fld.data).cuda()
    for nb in [(2, 2, 2), (3, 2, 1)]:
        host = wl.cut_bricks(fld, nb, 1)
        cut = wl.cut_bricks_cuda(dev, fld.dims, nb, 1)
        assert len(host) == len(cut)
        for h, c in zip(host, cut):
            assert np.array_equal(h, c.cpu().numpy())
