"""GPU parity, part 1: G-sphere maps (bit-exact), west_fft3d, west_h_apply, the DMMA GEMMs - all through the C ABI."""
import numpy as np
import pytest

import synth
from oracle import gsphere as ogs
from oracle import hamiltonian as oham
import oracle_problem
from gpu_common import make_west, random_vectors, relmax

pytestmark = pytest.mark.gpu
TOL = 1e-9    # north_star: relative max-norm 1e-9 for FP64


@pytest.mark.parametrize("name", ["cfg1", "mini2", "mini48", "cfg2", "cfg5"])
def test_gsphere_bit_exact(name):
    import paper_2203_05623_b200 as wb
    cfg = synth.get_config(name)
    m = ogs.enumerate_sphere(cfg["n2max"])
    for mode in (wb.WEST_FULL, wb.WEST_GAMMA):
        w = wb.West(cfg["L"], cfg["n2max"], cfg["N"], mode)
        miller, idx, idxm, g2 = w.gsphere()
        ref = m if mode == wb.WEST_FULL else m[ogs.half_sphere_mask(m)]
        assert miller.dtype == np.int32 and np.array_equal(miller, ref)
        assert np.array_equal(idx, ogs.fft_index(ref, cfg["N"]))
        assert np.array_equal(idxm, ogs.fft_index(-ref, cfg["N"]))
        assert np.array_equal(g2, ogs.g2_of(ref, cfg["L"]))      # same expression order -> same bits
        w.close()


@pytest.mark.parametrize("name,n_vec", [("cfg1", 5), ("mini2", 5), ("mini48", 3), ("cfg2", 7), ("cfg5", 3)])
def test_fft3d_vs_library_fft(name, n_vec):
    import torch
    p = oracle_problem.build(name, dense=False)
    w, sel = make_west(p, with_states=False, with_kb=False)
    c, cfull = random_vectors(p, n_vec, 99)
    x = torch.from_numpy(c).cuda()
    r = w.fft3d(+1, x)
    ref = oham.to_real_space(cfull, p.fft_idx, p.N)
    if p.gamma:
        assert np.max(np.abs(ref.imag)) < 1e-9 * np.max(np.abs(ref.real))
        ref = ref.real
    assert relmax(r.cpu().numpy(), ref) < TOL
    # r -> G of a function that is NOT sphere-limited (product of two): truncation of its DFT
    f = ref * ref[::-1].copy()
    back = w.fft3d(-1, torch.from_numpy(np.ascontiguousarray(f)).cuda())
    refc = oham.to_g_space(f, p.fft_idx)[:, sel]
    assert relmax(back.cpu().numpy(), refc) < TOL
    # round trip identity on sphere-limited data
    rt = w.fft3d(-1, r)
    assert relmax(rt.cpu().numpy(), c) < TOL
    w.close()


@pytest.mark.parametrize("name", ["cfg1", "mini2", "mini48"])
def test_h_apply_vs_dense(name):
    import torch
    p = oracle_problem.build(name)
    w, sel = make_west(p, with_states=False)
    c, cfull = random_vectors(p, 7, 98)
    y = w.h_apply(torch.from_numpy(c).cuda()).cpu().numpy()
    ref = (p.H @ cfull.T).T[:, sel]
    assert relmax(y, ref) < TOL
    w.close()


@pytest.mark.parametrize("name,n_vec", [("cfg2", 9), ("cfg5", 4)])
def test_h_apply_vs_matrix_free(name, n_vec):
    import torch
    p = oracle_problem.build(name, dense=False)
    w, sel = make_west(p, with_states=False)
    c, cfull = random_vectors(p, n_vec, 97)
    y = w.h_apply(torch.from_numpy(c).cuda()).cpu().numpy()
    ref = oham.apply_h(cfull, p.miller, p.L, p.N, p.vloc, p.beta, p.dcoef)[:, sel]
    assert relmax(y, ref) < TOL
    # mixed precision: FP32 FFT path, tolerance 1e-4 (config 4)
    import paper_2203_05623_b200 as wb
    ym = w.h_apply(torch.from_numpy(c).cuda(), precision=wb.WEST_MIXED).cpu().numpy()
    assert relmax(ym, ref) < 1e-4
    assert relmax(ym, ref) > 1e-12      # it really ran in FP32
    w.close()


@pytest.mark.parametrize("name,n_vec", [("cfg1", 5), ("mini2", 9), ("cfg2", 70)])
def test_mixed_nonlocal_term_is_fp32_class(name, n_vec):
    """WEST_MIXED applies the KB projectors as 3xTF32 tensor-core GEMMs (FP32 matrix multiplication).  The nonlocal
    term in isolation - H*psi with projectors minus H*psi without, both through the mixed path, whose local part is deterministic -
    must agree with the oracle's sum_k beta_k D_k <beta_k|c> to FP32 class: one dropped lo*hi term, a single-pass TF32
    product (2^-11) or a running sum kept in the tensor core's truncating accumulator would leave 1e-5 .. 5e-4."""
    import torch
    import paper_2203_05623_b200 as wb
    p = oracle_problem.build(name, dense=False)
    c, cfull = random_vectors(p, n_vec, 96)
    x = torch.from_numpy(c).cuda()
    w, sel = make_west(p, with_states=False)
    y_kb = w.h_apply(x, precision=wb.WEST_MIXED).cpu().numpy()
    w.close()
    w0, _ = make_west(p, with_states=False, with_kb=False)
    y_loc = w0.h_apply(x, precision=wb.WEST_MIXED).cpu().numpy()
    w0.close()
    ref = (cfull @ np.conj(p.beta).T * np.asarray(p.dcoef)) @ p.beta
    err = relmax(y_kb - y_loc, ref[:, sel])
    assert err < 2e-6, err      # measured 2.4e-7 .. 4.8e-7; 7e-6 .. 2e-5 when the tensor core's truncating accumulator carried the sum
    assert err > 1e-13          # it did not run in FP64


@pytest.mark.parametrize("m,n,k", [(10, 32, 1030), (384, 1000, 18278), (130, 257, 4098)])
def test_gemm_tn_and_update(m, n, k):
    import torch
    import paper_2203_05623_b200 as wb
    w = wb.West(10.0, 25, 24, wb.WEST_FULL)
    rng = np.random.Generator(np.random.PCG64(5))
    A = rng.standard_normal((m, k))
    B = rng.standard_normal((n, k))
    Cg = w.gemm_tn(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda()).cpu().numpy()
    assert relmax(Cg, A @ B.T) < 1e-12
    ldc = (n + 1) // 2 * 2
    Cm = np.zeros((m, ldc))
    Cm[:, :n] = rng.standard_normal((m, n))
    Y0 = rng.standard_normal((n, k))
    Y = torch.from_numpy(Y0.copy()).cuda()
    w.gemm_update(torch.from_numpy(Cm).cuda(), torch.from_numpy(A).cuda(), Y)
    assert relmax(Y.cpu().numpy(), Y0 + Cm[:, :n].T @ A) < 1e-12
    w.close()


@pytest.mark.parametrize("name,with_kb", [("cfg2", True), ("cfg5", False)])
def test_full_sphere_mode_on_the_large_grids(name, with_kb):
    """WEST_FULL (complex vectors, one transform per vector) on the 72^3 and 144^3 grids, which the configs themselves only use
    in WEST_GAMMA mode: fft3d and h_apply against the library FFT / the oracle's matrix-free H."""
    import torch
    import paper_2203_05623_b200 as wb
    p = oracle_problem.build(name, dense=False)
    w = wb.West(p.L, p.n2max, p.N, wb.WEST_FULL)
    assert w.n_g == p.n_full
    w.set_vloc(torch.from_numpy(np.ascontiguousarray(p.vloc)).cuda())
    if with_kb:
        w.set_kb(torch.from_numpy(np.ascontiguousarray(p.beta)).cuda(), p.dcoef)
    rng = np.random.Generator(np.random.PCG64(96))
    c = rng.standard_normal((3, p.n_full)) + 1j * rng.standard_normal((3, p.n_full))
    x = torch.from_numpy(c).cuda()
    r = w.fft3d(+1, x)
    assert relmax(r.cpu().numpy(), oham.to_real_space(c, p.fft_idx, p.N)) < TOL
    assert relmax(w.fft3d(-1, r).cpu().numpy(), c) < TOL
    y = w.h_apply(x).cpu().numpy()
    ref = oham.apply_h(c, p.miller, p.L, p.N, p.vloc, p.beta if with_kb else None, p.dcoef if with_kb else None)
    assert relmax(y, ref) < TOL
    w.close()


def test_fp64_pipe_yardstick_runs_and_shows_one_shared_pipe():
    """west_probe_fp64_pipes: DMMA-only, DFMA-only and mixed launches all finish, report the flop counts west.h
    states, and the mixed rate does not exceed the better single-kind rate by more than 10 % - DMMA and DFMA share one pipe on B200."""
    import paper_2203_05623_b200 as wb
    p = oracle_problem.build("cfg1")
    w = wb.West(p.L, p.n2max, p.N, wb.WEST_FULL)
    rate = {}
    for mode, nd in ((1, 16), (2, 0), (3, 8)):
        ms, fd, ff = w.probe_fp64_pipes(mode, nd, iters=4000)
        assert ms > 0
        assert fd == ((148.0 * nd * 4000 * 8 * 512) if mode & 1 else 0.0) and ff == ((148.0 * (16 - nd) * 4000 * 8 * 4 * 64) if mode & 2 else 0.0)
        rate[mode] = (fd + ff) / ms
    assert rate[3] < 1.10 * max(rate[1], rate[2])
    with pytest.raises(wb.WestError):
        w.probe_fp64_pipes(0, 8)
    w.close()
