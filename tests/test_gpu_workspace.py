"""GPU checks of the workspace contract of include/west.h ("the caller allocates every device buffer including the
workspace; the library never allocates or frees in a hot call") and of the perturbation sub-blocks a small workspace forces."""
import ctypes as C

import numpy as np
import pytest

import oracle_problem
from gpu_common import make_west, random_vectors, relmax
from oracle import chi0 as ochi0

pytestmark = pytest.mark.gpu


def _free_bytes():
    import torch
    torch.cuda.synchronize()
    return torch.cuda.mem_get_info()[0]          # cudaMemGetInfo: what the DRIVER has free (not torch's cache)


def test_caller_workspace_means_no_allocation_in_the_hot_call():
    """Config-2-size cell (72^3 grid, 9139 Gamma plane waves, 128 states, 256 projectors), 8 perturbations: with a caller workspace
    of west_workspace_bytes the call leaves the driver's free memory untouched and repeats to within the atomics west.h names."""
    import torch
    import paper_2203_05623_b200 as wb
    p = oracle_problem.build("cfg2", dense=False)
    w = wb.West(p.L, p.n2max, p.N, wb.WEST_GAMMA)
    dev = torch.device("cuda:0")
    w.set_vloc(torch.from_numpy(np.ascontiguousarray(p.vloc)).to(dev))
    w.set_kb(torch.from_numpy(np.ascontiguousarray(p.beta[:, p.half])).to(dev), p.dcoef)
    # inputs of THIS test need not be eigenvectors (it checks memory behaviour and repeatability, not parity): orthonormalised
    # smooth random orbitals, "eigenvalues" = their Rayleigh quotients' order of magnitude
    rng = np.random.Generator(np.random.PCG64(77))
    n_occ = p.n_occ
    c = (rng.standard_normal((n_occ, w.n_g)) + 1j * rng.standard_normal((n_occ, w.n_g))) * np.exp(-0.5 * p.g2[p.half])
    c[:, 0] = c[:, 0].real
    y = np.concatenate([c.real * np.sqrt(2.0), c.imag * np.sqrt(2.0)], axis=1)
    y[:, 0] /= np.sqrt(2.0)
    y[:, w.n_g] = 0.0
    q, _ = np.linalg.qr(y.T)
    y = q.T
    y[:, 0] *= np.sqrt(2.0)
    psi = (y[:, :w.n_g] + 1j * y[:, w.n_g:]) / np.sqrt(2.0)
    eps = np.linspace(-0.5, 0.3, n_occ)
    w.set_states(torch.from_numpy(np.ascontiguousarray(psi)).to(dev), eps)
    n_pert = 8
    dV = torch.from_numpy(np.ascontiguousarray(p.dV[:n_pert])).to(dev)
    dn = torch.empty((1, n_pert, p.N, p.N, p.N), dtype=torch.float64, device=dev)
    need = w.workspace_bytes(wb.binding.WEST_OP_CHI0, n_pert, 1)
    assert need > 4 * 16 * w.n_g * n_pert * n_occ          # at least the four vector sets
    ws = torch.empty(need, dtype=torch.uint8, device=dev)
    w.set_workspace(ws)
    kw = dict(tol=1e-6, max_iter=8, alpha_pv=2.0, dn=dn, want_stats=False)
    w.chi0_apply(dV, [0.0], **kw)                              # first call: kernel attributes, module load
    a = dn.clone()
    held = w.device_bytes()
    f0 = _free_bytes()
    w.chi0_apply(dV, [0.0], **kw)
    f1 = _free_bytes()
    w.chi0_apply(dV, [0.0], **kw)
    f2 = _free_bytes()
    assert f0 == f1 == f2                                      # no cudaMalloc / cudaFree between the probes (driver-level free memory)
    assert w.device_bytes() == held
    # repeatable up to the FP64 atomics of the dn accumulation and the split-K GEMMs (west.h "Determinism")
    assert relmax(dn.cpu().numpy(), a.cpu().numpy()) < 1e-9           # (8 CG iterations on non-eigenvector inputs amplify the last-bit differences)
    # a workspace that is too small for even one perturbation is refused, nothing is allocated behind the caller's back
    small = torch.empty(1 << 20, dtype=torch.uint8, device=dev)
    w.set_workspace(small)
    with pytest.raises(wb.WestError) as e:
        w.chi0_apply(dV, [0.0], **kw)
    assert e.value.code == wb.binding.WEST_EWORKSPACE
    with pytest.raises(wb.WestError) as e:
        w.h_apply(torch.zeros((64, w.n_g), dtype=torch.complex128, device=dev))
    assert e.value.code == wb.binding.WEST_EWORKSPACE
    assert w.device_bytes() == held
    # h_apply with exactly its own size
    x = torch.zeros((64, w.n_g), dtype=torch.complex128, device=dev)
    w.set_workspace(torch.empty(w.workspace_bytes(wb.binding.WEST_OP_H_APPLY, 64), dtype=torch.uint8, device=dev))
    w.h_apply(x)
    w.set_workspace(None)
    w.close()


@pytest.mark.parametrize("name,omegas,solver", [("mini2", [0.0], 0), ("mini3", [0.05, 5.0], 0), ("mini3", [0.0, 0.6947], 1)])
def test_sub_blocks_forced_by_a_small_workspace_give_the_same_answer(name, omegas, solver):
    """A workspace sized for 2 (then 1) perturbations makes the library walk the 4-6 perturbations in sub-blocks; dn and dpsi must
    equal the oracle's sum over states exactly as the one-block run does."""
    import torch
    import paper_2203_05623_b200 as wb
    B = wb.binding
    p = oracle_problem.build(name)
    w, sel = make_west(p)
    dV = torch.from_numpy(np.ascontiguousarray(p.dV)).cuda()
    n_pert = dV.shape[0]
    ref = ochi0.chi0_sum_over_states(p.eps, p.U, p.n_occ, p.dV, omegas, p.miller, p.L, p.N)
    op = B.WEST_OP_CHI0_MULTISHIFT if solver == 1 else (B.WEST_OP_CHI0_IW if max(omegas) > 0 else B.WEST_OP_CHI0)
    full, dpsi_full, st = w.chi0_apply(dV, omegas, tol=1e-12, max_iter=3000, alpha_pv=p.alpha, solver=solver, want_dpsi=True)
    assert st["rc"] == 0 and st["n_sub_blocks"] == 1
    for fit in (2, 1):
        ws = torch.empty(w.workspace_bytes(op, fit, len(omegas)), dtype=torch.uint8, device="cuda")
        w.set_workspace(ws)
        dn, dpsi, st = w.chi0_apply(dV, omegas, tol=1e-12, max_iter=3000, alpha_pv=p.alpha, solver=solver, want_dpsi=True)
        assert st["rc"] == 0 and st["n_unconverged"] == 0
        assert st["n_sub_blocks"] == (n_pert + fit - 1) // fit
        assert relmax(dn.cpu().numpy(), ref) < 1e-9
        assert relmax(dn.cpu().numpy(), full.cpu().numpy()) < 1e-10
        assert relmax(dpsi.cpu().numpy(), dpsi_full.cpu().numpy()) < 1e-9
        w.set_workspace(None)
    w.close()


def test_alpha_below_the_band_width_is_refused_and_the_default_is_per_orbital():
    import torch
    import paper_2203_05623_b200 as wb
    p = oracle_problem.build("mini2")
    w, _ = make_west(p)
    dV = torch.from_numpy(np.ascontiguousarray(p.dV[:2])).cuda()
    width = float(p.eps[p.n_occ - 1] - p.eps[0])
    with pytest.raises(wb.WestError) as e:
        w.chi0_apply(dV, [0.0], alpha_pv=0.5 * width)
    assert e.value.code == wb.binding.WEST_EINVAL
    ref = ochi0.chi0_sum_over_states(p.eps, p.U, p.n_occ, p.dV[:2], [0.0], p.miller, p.L, p.N)
    dn0, _, st0 = w.chi0_apply(dV, [0.0], tol=1e-12, alpha_pv=0.0, check_every=1)         # per-orbital alpha_v (west.h)
    dn1, _, st1 = w.chi0_apply(dV, [0.0], tol=1e-12, alpha_pv=p.alpha, check_every=1)     # the oracle's constant 2 W
    assert st0["rc"] == 0 and relmax(dn0.cpu().numpy(), ref) < 1e-9 and relmax(dn1.cpu().numpy(), ref) < 1e-9
    assert 0 < st0["iters_min"] <= st0["iters"] and st0["n_h_apply"] <= st1["n_h_apply"] * 1.05
    w.close()


def test_stats_free_call_reports_non_convergence():
    import torch
    import paper_2203_05623_b200 as wb
    p = oracle_problem.build("mini2")
    w, _ = make_west(p)
    dV = torch.from_numpy(np.ascontiguousarray(p.dV[:2])).cuda()
    _, _, st = w.chi0_apply(dV, [0.0], tol=1e-12, max_iter=3, alpha_pv=p.alpha, want_stats=False)
    assert st["rc"] == wb.WEST_NOTCONVERGED
    _, _, st = w.chi0_apply(dV, [0.0], tol=1e-12, max_iter=500, alpha_pv=p.alpha, want_stats=False)
    assert st["rc"] == 0
    w.close()


def test_multishift_history_workspace_sizes():
    """WEST_OP_CHI0_MULTISHIFT_HIST is the size that holds the full 128-slot Krylov ring for the whole block; WEST_OP_CHI0_MULTISHIFT (the
    minimum) still runs - as sub-blocks or with the per-shift recurrences - and both give the sum over states; no allocation in either."""
    import torch
    import paper_2203_05623_b200 as wb
    B = wb.binding
    p = oracle_problem.build("mini3")
    w, sel = make_west(p)
    omegas = [0.0, 0.05, 5.0]
    dV = torch.from_numpy(np.ascontiguousarray(p.dV)).cuda()
    n_pert = dV.shape[0]
    ref = ochi0.chi0_sum_over_states(p.eps, p.U, p.n_occ, p.dV, omegas, p.miller, p.L, p.N)
    big = w.workspace_bytes(B.WEST_OP_CHI0_MULTISHIFT_HIST, n_pert, len(omegas))
    small = w.workspace_bytes(B.WEST_OP_CHI0_MULTISHIFT, n_pert, len(omegas))
    assert big > small > 0
    dn = torch.empty((len(omegas), n_pert, p.N, p.N, p.N), dtype=torch.float64, device="cuda")
    for need, slots in ((big, 128), (small, None)):
        ws = torch.empty(need, dtype=torch.uint8, device="cuda")
        w.set_workspace(ws)
        kw = dict(tol=1e-12, max_iter=3000, alpha_pv=p.alpha, solver=1, dn=dn)
        w.chi0_apply(dV, omegas, **kw)
        held, f0 = w.device_bytes(), _free_bytes()
        _, _, st = w.chi0_apply(dV, omegas, **kw)
        assert _free_bytes() == f0 and w.device_bytes() == held
        assert st["rc"] == 0 and st["n_unconverged"] == 0
        if slots is not None:
            assert st["ms_history_slots"] == slots and st["n_sub_blocks"] == 1
        assert relmax(dn.cpu().numpy(), ref) < 1e-9
        w.set_workspace(None)
    w.close()
