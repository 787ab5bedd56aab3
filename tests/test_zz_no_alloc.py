"""GPU check of west_fft3d_static (include/west.h): the sphere-truncated FFT with its scratch in the library's fixed static device array,
for callers that cannot call cudaMalloc.  Its output must equal west_fft3d's (same kernels, only the scratch pointers differ) on two
calls in a row - the array is shared and keeps the previous call's contents - in both directions and both storage modes; the call must
not change the driver's free memory; a cell whose transform does not fit the array is rejected.

Named test_zz_* so that pytest collects it last (the suite runs with `pytest -x`)."""
import numpy as np
import pytest

from gpu_common import relmax

pytestmark = pytest.mark.gpu
TOL = 1e-9          # the FP64 parity bar of the other GPU tests (north_star); the two paths run the same arithmetic


def _coeffs(w, n, seed, gamma):
    rng = np.random.Generator(np.random.PCG64(seed))
    c = rng.standard_normal((n, w.n_g)) + 1j * rng.standard_normal((n, w.n_g))
    if gamma:
        c[:, 0] = c[:, 0].real          # c(0) of a real function is real
    return c


@pytest.mark.parametrize("L,n2max,N,gamma,n_batch", [(10.0, 25, 24, False, 5), (10.25, 66, 36, True, 7), (20.5, 266, 72, True, 3)])
def test_static_scratch_fft_matches_the_workspace_path_twice(L, n2max, N, gamma, n_batch):
    import torch
    import paper_2203_05623_b200 as wb
    w = wb.West(L, n2max, N, wb.WEST_GAMMA if gamma else wb.WEST_FULL)
    dev = torch.device("cuda:0")
    grid_dt = torch.float64 if gamma else torch.complex128
    assert w.lib.west_static_scratch_bytes() == 8 << 20
    xs = [torch.from_numpy(_coeffs(w, n_batch, 11 + k, gamma)).to(dev) for k in range(2)]
    ref_r = [w.fft3d(+1, x) for x in xs]                                   # existing path (workspace arena)
    ref_g = [w.fft3d(-1, r) for r in ref_r]
    out_r = torch.empty((n_batch, N, N, N), dtype=grid_dt, device=dev)
    out_g = torch.empty((n_batch, w.n_g), dtype=torch.complex128, device=dev)
    torch.cuda.synchronize()
    held = w.device_bytes()
    w.fft3d_static(+1, xs[0], out_r)                                       # first call on this device: address look-up, kernel attributes
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for k in range(2):                                                     # two calls in a row, different inputs, same shared array
        w.fft3d_static(+1, xs[k], out_r)
        assert relmax(out_r.cpu().numpy(), ref_r[k].cpu().numpy()) < TOL
        w.fft3d_static(-1, ref_r[k], out_g)
        assert relmax(out_g.cpu().numpy(), ref_g[k].cpu().numpy()) < TOL
        # round trip on sphere-limited data is the identity
        assert relmax(out_g.cpu().numpy(), xs[k].cpu().numpy()) < TOL
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                           # no cudaMalloc / cudaFree behind the caller's back
    assert w.device_bytes() == held
    w.close()


def test_static_scratch_rejects_a_cell_that_does_not_fit():
    import torch
    import paper_2203_05623_b200 as wb
    w = wb.West(41.0, 1064, 144, wb.WEST_GAMMA)                            # config-5 grid: one slot needs 55 MB > 8 MiB
    x = torch.zeros((2, w.n_g), dtype=torch.complex128, device="cuda:0")
    out = torch.empty((2, 144, 144, 144), dtype=torch.float64, device="cuda:0")
    with pytest.raises(wb.WestError) as e:
        w.fft3d_static(+1, x, out)
    assert e.value.code == wb.binding.WEST_EWORKSPACE and "static array" in str(e.value)
    w.close()
