"""GPU parity, part 2: west_chi0_apply against the sum-over-states oracle (Eq. 10-11)."""
import numpy as np
import pytest

import oracle_problem
from gpu_common import make_west, relmax
from oracle import chi0 as ochi0
from oracle import gsphere as ogs

pytestmark = pytest.mark.gpu
TOL = 1e-9


def _run(name, precision=None, tol_cg=1e-12, alpha=None, precond=1, solver=0, omegas=None, max_iter=500, n_defl=0, cg_kernel=0, ms_history=0, want_dpsi=True):
    import torch
    import paper_2203_05623_b200 as wb
    p = oracle_problem.build(name)
    w, sel = make_west(p)
    w.set_cg_kernel(cg_kernel)
    w.set_ms_history(ms_history)
    if n_defl:
        w.set_deflation(torch.from_numpy(np.ascontiguousarray(p.U[:, p.n_occ:p.n_occ + n_defl].T[:, sel])).cuda(), p.eps[p.n_occ:p.n_occ + n_defl])
    dV = torch.from_numpy(np.ascontiguousarray(p.dV)).cuda()
    prec = wb.WEST_FP64 if precision is None else precision
    om = p.omegas if omegas is None else omegas
    dn, dpsi, st = w.chi0_apply(dV, om, tol=tol_cg, max_iter=max_iter, alpha_pv=p.alpha if alpha is None else alpha,
                                precond=precond, precision=prec, want_dpsi=want_dpsi, n_occ=p.n_occ, solver=solver)
    ref_dn, ref_dpsi = ochi0.chi0_sum_over_states(p.eps, p.U, p.n_occ, p.dV, om, p.miller, p.L, p.N, return_dpsi=True)
    w.close()
    return p, sel, dn.cpu().numpy(), dpsi.cpu().numpy() if want_dpsi else None, st, ref_dn, ref_dpsi


def _check_dpsi(p, sel, dpsi, ref_dpsi, tol):
    if p.gamma:
        # [w][i][v][2][n_g]: Re and Im parts of dpsi(r) as two real functions -> dpsi(G) = R(G) + i I(G) on the full sphere
        full = ogs.expand_half_to_full(dpsi[..., 0, :], p.miller) + 1j * ogs.expand_half_to_full(dpsi[..., 1, :], p.miller)
        assert relmax(full, ref_dpsi) < tol
    else:
        assert relmax(dpsi, ref_dpsi) < tol


def test_chi0_cfg1_full_complex():
    p, sel, dn, dpsi, st, ref_dn, ref_dpsi = _run("cfg1")
    assert st["rc"] == 0 and st["n_unconverged"] == 0 and st["resid_max"] <= 1e-12
    assert relmax(dn, ref_dn) < TOL
    _check_dpsi(p, sel, dpsi, ref_dpsi, TOL)


def test_chi0_mini2_gamma():
    p, sel, dn, dpsi, st, ref_dn, ref_dpsi = _run("mini2")
    assert st["rc"] == 0 and st["n_unconverged"] == 0
    assert relmax(dn, ref_dn) < TOL
    _check_dpsi(p, sel, dpsi, ref_dpsi, TOL)
    assert np.max(np.abs(dpsi[..., 1, :])) == 0.0          # omega = 0: dpsi is a real function


def test_chi0_mini3_imaginary_frequencies():
    p, sel, dn, dpsi, st, ref_dn, ref_dpsi = _run("mini3")
    assert st["rc"] == 0 and st["n_unconverged"] == 0
    for w in range(len(p.omegas)):
        assert relmax(dn[w], ref_dn[w]) < TOL
    _check_dpsi(p, sel, dpsi, ref_dpsi, TOL)


def test_chi0_mini4_mixed_precision():
    import paper_2203_05623_b200 as wb
    p, sel, dn, dpsi, st, ref_dn, ref_dpsi = _run("mini4", precision=wb.WEST_MIXED, tol_cg=1e-6)
    assert relmax(dn, ref_dn) < 1e-4                        # north_star: 1e-4 for the mixed path
    assert relmax(dn, ref_dn) > 1e-11


def test_chi0_alpha_and_preconditioner_do_not_change_the_result():
    p, sel, dn0, _, st0, ref_dn, _ = _run("mini2")
    _, _, dn1, _, st1, _, _ = _run("mini2", alpha=3.0 * p.alpha, precond=0)
    assert relmax(dn1, ref_dn) < TOL and relmax(dn1, dn0) < TOL
    assert st1["iters"] >= st0["iters"]                    # the preconditioner only changes the iteration count


def test_chi0_not_converged_status():
    import torch
    import paper_2203_05623_b200 as wb
    p = oracle_problem.build("cfg1")
    w, _ = make_west(p)
    dV = torch.from_numpy(np.ascontiguousarray(p.dV)).cuda()
    dn, _, st = w.chi0_apply(dV, [0.0], tol=1e-14, max_iter=3, alpha_pv=p.alpha)
    assert st["rc"] == wb.WEST_NOTCONVERGED and st["n_unconverged"] > 0 and st["iters"] == 3
    w.close()


def test_chi0_multishift_all_frequencies_from_one_krylov_sequence():
    """solver = 1: omega = 0 and three imaginary frequencies from one unpreconditioned CG sequence."""
    omegas = [0.0, 0.05, 0.6947, 5.0]
    p, sel, dn, dpsi, st, ref_dn, ref_dpsi = _run("mini3", solver=1, omegas=omegas, max_iter=2000)
    assert st["rc"] == 0 and st["n_unconverged"] == 0
    for w in range(len(omegas)):
        assert relmax(dn[w], ref_dn[w]) < TOL
    _check_dpsi(p, sel, dpsi, ref_dpsi, TOL)
    # one H*psi per column and iteration serves all four frequencies
    assert st["n_h_apply"] <= st["iters"] * p.n_occ * len(p.dV)


@pytest.mark.parametrize("slots", [-1, 2, 3, 7, 32, 128])
@pytest.mark.parametrize("want_dpsi", [True, False])
def test_chi0_multishift_krylov_history_and_per_shift_recurrences_agree(slots, want_dpsi):
    """west_set_ms_history: the shifted solutions contracted from a ring of seed residuals (ring sizes that wrap after every iteration,
    every second, every sixth, a few times, never) and the per-shift vector recurrences (-1) all reach the sum over states (Eq. 10-11
    with the i omega shift) within the same 1e-9, with the same iteration count; the carry vectors of a wrapping
    ring and the Re-only contraction (no dpsi requested) are covered."""
    omegas = [0.0, 0.05, 0.6947, 5.0]
    p, sel, dn, dpsi, st, ref_dn, ref_dpsi = _run("mini3", solver=1, omegas=omegas, max_iter=2000, ms_history=slots, want_dpsi=want_dpsi)
    assert st["rc"] == 0 and st["n_unconverged"] == 0
    assert st["ms_history_slots"] == (0 if slots < 0 else slots)
    for w in range(len(omegas)):
        assert relmax(dn[w], ref_dn[w]) < TOL
    if want_dpsi:
        _check_dpsi(p, sel, dpsi, ref_dpsi, TOL)
    _, _, dn0, _, st0, _, _ = _run("mini3", solver=1, omegas=omegas, max_iter=2000, ms_history=-1, want_dpsi=False)
    assert st0["iters"] == st["iters"] and st0["n_h_apply"] == st["n_h_apply"]
    assert relmax(dn, dn0) < 1e-11
    assert (st["n_hist_passes"] > 0) == (slots >= 0) and (st["n_shift_updates"] > 0) == (slots < 0)


def test_chi0_multishift_history_hits_the_iteration_cap_cleanly():
    """max_iter below convergence: WEST_NOTCONVERGED, partial sums written (finite), the ring sized by max_iter + 1."""
    import paper_2203_05623_b200 as wb
    p, sel, dn, _, st, ref_dn, _ = _run("mini3", solver=1, omegas=[0.0, 0.5], max_iter=9, want_dpsi=False)
    assert st["rc"] == wb.WEST_NOTCONVERGED and st["n_unconverged"] > 0 and st["iters"] == 9 and st["ms_history_slots"] == 10
    assert np.all(np.isfinite(dn))
    _, _, dn0, _, st0, _, _ = _run("mini3", solver=1, omegas=[0.0, 0.5], max_iter=9, want_dpsi=False, ms_history=-1)
    assert relmax(dn, dn0) < 1e-11


@pytest.mark.parametrize("name,solver,omegas", [("cfg1", 0, None), ("mini2", 0, None), ("mini3", 0, None), ("mini3", 1, [0.0, 0.05, 5.0])])
def test_chi0_with_deflated_conduction_states(name, solver, omegas):
    """west_set_deflation: same result as without (parity against the sum over states), fewer iterations."""
    p, sel, dn0, _, st0, ref_dn, ref_dpsi = _run(name, solver=solver, omegas=omegas, max_iter=2000)
    p, sel, dn, dpsi, st, ref_dn, ref_dpsi = _run(name, solver=solver, omegas=omegas, max_iter=2000, n_defl=12)
    assert st["rc"] == 0 and st["n_unconverged"] == 0
    assert relmax(dn, ref_dn) < TOL
    _check_dpsi(p, sel, dpsi, ref_dpsi, TOL)
    # at omega = 0 the smallest eigenvalue of the operator is the gap and deflation must help; large omega already lifts the spectrum
    assert st["iters"] <= st0["iters"] and (omegas is not None or name == "mini3" or st["iters"] < st0["iters"])


@pytest.mark.parametrize("name", ["cfg1", "mini2"])
@pytest.mark.parametrize("which", [1, 2])
def test_chi0_other_cg_kernels(name, which):
    """west_set_cg_kernel(1): the streaming vector kernel (the one cfg 5 and the COCG pairs use); (2): the column split over a 2-CTA
    cluster, on cells where the default is the column-resident kernel; same parity bar against the sum over states (Eq. 10-11),
    same iteration count."""
    p, sel, dn, dpsi, st, ref_dn, ref_dpsi = _run(name, cg_kernel=which, omegas=[0.0])
    assert st["rc"] == 0 and st["n_unconverged"] == 0
    assert relmax(dn, ref_dn) < 1e-9
    _check_dpsi(p, sel, dpsi, ref_dpsi, 1e-9)
    _, _, dn0, _, st0, _, _ = _run(name, cg_kernel=0, omegas=[0.0])
    assert st0["iters"] == st["iters"]
    assert relmax(dn, dn0) < 1e-12


@pytest.mark.parametrize("name,omegas", [("cfg1", None), ("mini2", None), ("mini3", [0.0, 0.6947]), ("mini48", None)])
def test_chi0_block_cg_same_answer_fewer_h_applications(name, omegas):
    """solver = 2 (second half): the perturbations of one orbital share one Krylov space.  Same parity bar against the
    sum over states (Eq. 10-11); at omega > 0 (mini3's second frequency) the call falls back to COCG; H*psi count below solver 0's."""
    p, sel, dn, dpsi, st, ref_dn, ref_dpsi = _run(name, solver=2, omegas=omegas)
    assert st["rc"] == 0 and st["n_unconverged"] == 0 and st["resid_max"] <= 1e-12
    for w in range(dn.shape[0]):
        assert relmax(dn[w], ref_dn[w]) < TOL
    _check_dpsi(p, sel, dpsi, ref_dpsi, TOL)
    _, _, dn0, _, st0, _, _ = _run(name, solver=0, omegas=omegas)
    assert relmax(dn, dn0) < TOL
    assert st["n_h_apply"] < st0["n_h_apply"]
    assert 0 < st["iters_min"] <= st["iters"]


def test_chi0_block_cg_mixed_precision_and_deflation():
    import paper_2203_05623_b200 as wb
    p, sel, dn, dpsi, st, ref_dn, ref_dpsi = _run("mini4", precision=wb.WEST_MIXED, tol_cg=1e-6, solver=2)
    assert st["rc"] == 0 and relmax(dn, ref_dn) < 1e-4
    p, sel, dn, dpsi, st, ref_dn, ref_dpsi = _run("mini2", solver=2, n_defl=12)
    assert st["rc"] == 0 and st["n_unconverged"] == 0 and relmax(dn, ref_dn) < TOL


def test_chi0_block_cg_degenerate_blocks():
    """Linearly dependent and zero right-hand sides inside one block (the rank-revealing solve must drop them), and a block of one."""
    import torch
    p = oracle_problem.build("mini2")
    w, _ = make_west(p)
    N = p.N
    dV = np.concatenate([p.dV[:2], 2.0 * p.dV[:1] - 0.5 * p.dV[1:2], np.full((1, N, N, N), 0.3), p.dV[:1]])     # rank 2 of 5, one zero response
    ref = ochi0.chi0_sum_over_states(p.eps, p.U, p.n_occ, dV, [0.0], p.miller, p.L, p.N)
    dn, _, st = w.chi0_apply(torch.from_numpy(np.ascontiguousarray(dV)).cuda(), [0.0], tol=1e-12, alpha_pv=p.alpha, solver=2)
    assert st["rc"] == 0 and st["n_unconverged"] == 0
    assert relmax(dn.cpu().numpy(), ref) < TOL and np.max(np.abs(dn[0, 3].cpu().numpy())) < 1e-12 * np.max(np.abs(ref))
    dn1, _, st1 = w.chi0_apply(torch.from_numpy(np.ascontiguousarray(dV[:1])).cuda(), [0.0], tol=1e-12, alpha_pv=p.alpha, solver=2)
    assert st1["rc"] == 0 and relmax(dn1.cpu().numpy()[0, 0], ref[0, 0]) < TOL
    w.close()
