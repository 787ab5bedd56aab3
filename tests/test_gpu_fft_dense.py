"""Parity of west_fft3d_dense (dense C2C 3D FFT, Fig. 3) with oracle/fft_dense.py through the C ABI.

Tolerances (relative to max|X|): FP64 1e-12 (rounding of ~3 log2(n) butterfly levels, each a few ulp of 1.1e-16, leaves
about 1e-15; north_star's FP64 bar is 1e-9), FP32 5e-6 (same count with ulp 6e-8: about 5e-7 expected)."""
import numpy as np
import pytest

import synth
from gpu_common import relmax
from oracle import fft_dense as ofd

pytestmark = pytest.mark.gpu
TOL = {"f64": 1e-12, "f32": 5e-6}


def _ctx():
    import paper_2203_05623_b200 as wb
    return wb.West(10.0, 25, 24, wb.WEST_FULL)          # the dense transform ignores the context's cell


def _to_dev(x, prec):
    import torch
    return torch.from_numpy(x).to("cuda", dtype=torch.complex128 if prec == "f64" else torch.complex64)


@pytest.mark.parametrize("n,n_batch", [(64, 3), (128, 1)])
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("sign", [1, -1])
def test_every_output_against_the_oracle(n, n_batch, prec, sign):
    w = _ctx()
    x = synth.dense_grid(n, n_batch)
    xd = _to_dev(x, prec)
    ref = ofd.dft3(xd.cpu().numpy().astype(np.complex128), sign)       # the oracle sees the (possibly FP32-rounded) input
    got = w.fft3d_dense(xd, sign)
    assert relmax(got.cpu().numpy(), ref) < TOL[prec]
    inplace = xd.clone()
    w.fft3d_dense(inplace, sign, out=inplace)                          # in place: same kernels, same order -> identical bits
    import torch
    assert torch.equal(torch.view_as_real(inplace), torch.view_as_real(got))
    w.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_256_cubed_sampled_outputs_parseval_and_round_trip(prec):
    import torch
    n = 256
    w = _ctx()
    x = synth.dense_grid(n, 1)
    xd = _to_dev(x, prec)
    xin = xd[0].cpu().numpy().astype(np.complex128)
    X = w.fft3d_dense(xd, -1)
    rng = np.random.Generator(np.random.PCG64(5))
    ks = [tuple(int(v) for v in rng.integers(0, n, 3)) for _ in range(48)]
    ks += [(0, 0, 0), (n - 1, n - 1, n - 1), (0, n - 1, 1), (17, 0, 255), (128, 128, 128), (1, 0, 0), (0, 1, 0), (0, 0, 1)]
    ref = ofd.dft3_at(xin, -1, ks)
    Xh = X[0].cpu().numpy()
    got = np.array([Xh[k] for k in ks])
    scale = float(np.max(np.abs(Xh)))
    assert np.max(np.abs(got - ref)) / scale < TOL[prec]
    # properties over ALL outputs: Parseval and the inverse transform
    e_in, e_out = float(np.sum(np.abs(xin) ** 2)), float(torch.sum(torch.abs(X.to(torch.complex128)) ** 2).item())
    assert abs(e_out - n ** 3 * e_in) < (1e-12 if prec == "f64" else 1e-5) * n ** 3 * e_in
    back = w.fft3d_dense(X, +1)
    err = float(torch.max(torch.abs(back / n ** 3 - xd)).item()) / float(torch.max(torch.abs(xd)).item())
    assert err < TOL[prec]
    w.close()


def test_delta_and_plane_wave_closed_forms():
    import torch
    n = 128
    w = _ctx()
    x = torch.zeros((1, n, n, n), dtype=torch.complex128, device="cuda")
    r0 = (5, 77, 126)
    x[0][r0] = 1.0
    X = w.fft3d_dense(x, +1)[0].cpu().numpy()
    k = np.arange(n)
    m = (k[:, None, None] * r0[0] + k[None, :, None] * r0[1] + k[None, None, :] * r0[2]) % n        # phase index reduced in integers
    pw = np.exp(2j * np.pi * m / n)
    assert np.max(np.abs(X - pw)) < 1e-14
    w.close()


def test_dense_fft_errors_and_empty_batch():
    import torch
    import paper_2203_05623_b200 as wb
    w = _ctx()
    with pytest.raises(wb.WestError) as e:
        w.fft3d_dense(torch.zeros((1, 100, 100, 100), dtype=torch.complex128, device="cuda"), 1)
    assert e.value.code == wb.binding.WEST_EINVAL
    with pytest.raises(wb.WestError):
        w.fft3d_dense(torch.zeros((1, 64, 64, 64), dtype=torch.complex128, device="cuda"), 0)
    assert w.fft3d_dense(torch.zeros((0, 64, 64, 64), dtype=torch.complex64, device="cuda"), -1).shape[0] == 0
    w.close()
