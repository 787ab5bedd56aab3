"""Library yardsticks on the same GPU, next to this package's kernels (context for the roofline numbers; not on any hot path).

    python -m paper_2203_05623_b200.yardsticks

1. FFT path: the unfused library route of the dual-space H*psi (cuFFT on the full grid) - scatter to the
   72^3 grid, cuFFT inverse, x V_loc, cuFFT forward, gather - against west_h_apply's fused, sphere-pruned path (same result).
2. GEMMs: cuBLAS DGEMM (through torch) on the shapes of the KB / P_v contractions against west_gemm_tn / west_gemm_update.
"""
import numpy as np
import torch

import synth

from . import WEST_GAMMA, West


def _time(fn, n=5):
    fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(n):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / n


def fft_yardstick(n_slots=512):
    cfg = synth.get_config("cfg2")
    N = cfg["N"]
    w = West(cfg["L"], cfg["n2max"], N, WEST_GAMMA)
    _, idx, idxm, g2 = w.gsphere()
    dev = torch.device("cuda")
    V = torch.randn((N, N, N), dtype=torch.float64, device=dev)
    w.set_vloc(V)
    B = n_slots
    x = torch.randn((2 * B, w.n_g), dtype=torch.float64, device=dev) + 1j * torch.randn((2 * B, w.n_g), dtype=torch.float64, device=dev)
    x[:, 0] = x[:, 0].real
    it = torch.from_numpy(idx.astype(np.int64)).to(dev)
    im = torch.from_numpy(idxm.astype(np.int64)).to(dev)

    def lib_path():
        a, b = x[0::2], x[1::2]
        grid = torch.zeros((B, N * N * N), dtype=torch.complex128, device=dev)
        grid[:, it] = a + 1j * b
        grid[:, im[1:]] = (a.conj() + 1j * b.conj())[:, 1:]
        r = torch.fft.ifftn(grid.view(B, N, N, N), dim=(1, 2, 3), norm="forward") * V
        f = torch.fft.fftn(r, dim=(1, 2, 3), norm="forward").view(B, -1)
        fp, fm = f[:, it], f[:, im]
        return 0.5 * (fp + fm.conj()), -0.5j * (fp - fm.conj())

    ya, _ = lib_path()
    y = w.h_apply(x)
    ref = ya + torch.from_numpy(g2).to(dev) * x[0::2]
    diff = float((y[0::2] - ref).abs().max() / ref.abs().max())
    grid0 = torch.randn((B, N, N, N), dtype=torch.float64, device=dev) + 0j
    t_lib = _time(lib_path)
    t_cufft = _time(lambda: torch.fft.fftn(torch.fft.ifftn(grid0, dim=(1, 2, 3)), dim=(1, 2, 3)))
    t_west = _time(lambda: w.h_apply(x))
    w.close()
    return {"slots": B, "rel_diff_vs_library_path": diff, "library_path_us_per_slot": 1e3 * t_lib / B,
            "bare_cufft_inv_fwd_us_per_slot": 1e3 * t_cufft / B, "west_h_apply_local_us_per_slot": 1e3 * t_west / B}


def gemm_yardstick(m=384, n=8192, k=18278):
    dev = torch.device("cuda")
    w = West(10.0, 25, 24, 0)
    A = torch.randn(m, k, dtype=torch.float64, device=dev)
    B = torch.randn(n, k, dtype=torch.float64, device=dev)
    Cm = torch.randn(m, n, dtype=torch.float64, device=dev)
    Y = torch.randn(n, k, dtype=torch.float64, device=dev)
    out = torch.empty(m, n, dtype=torch.float64, device=dev)
    sq = torch.randn(8192, 8192, dtype=torch.float64, device=dev)
    fl = 2.0 * m * n * k
    r = {"shape": [m, n, k],
         "cublas_dgemm_8192_tflops": 2.0 * 8192 ** 3 / _time(lambda: sq @ sq.T) / 1e9,
         "cublas_tn_tflops": fl / _time(lambda: A @ B.T) / 1e9,
         "cublas_update_tflops": fl / _time(lambda: Y.addmm_(Cm.T, A)) / 1e9,
         "west_gemm_tn_tflops": fl / _time(lambda: w.gemm_tn(A, B, out)) / 1e9,
         "west_gemm_update_tflops": fl / _time(lambda: w.gemm_update(Cm, A, Y)) / 1e9}
    w.close()
    return r


if __name__ == "__main__":
    import json
    print(json.dumps({"fft": fft_yardstick(), "gemm": gemm_yardstick()}, indent=1))
