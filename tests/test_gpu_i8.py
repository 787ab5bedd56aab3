"""GPU parity of WEST_FP64_I8 (include/west.h): the KB / P_v projector GEMMs of H*psi as error-free int8-slice products on the INT8
tensor path (tcgen05 kind::i8).  Same bars as WEST_FP64: H*psi against the oracle's dense H, chi0*dV against the sum over
states (Eq. 10-11), 1e-9; and against the DMMA path of the same library far below that."""
import numpy as np
import pytest

import oracle_problem
from gpu_common import make_west, random_vectors, relmax
from oracle import chi0 as ochi0
from oracle import hamiltonian as oham

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("name,n_vec", [("cfg1", 5), ("mini2", 7), ("mini48", 130)])
def test_h_apply_i8_vs_dense_h_and_vs_dmma(name, n_vec):
    import torch
    import paper_2203_05623_b200 as wb
    p = oracle_problem.build(name)
    w, sel = make_west(p, with_states=False)
    c, c_full = random_vectors(p, n_vec, seed=31)
    x = torch.from_numpy(np.ascontiguousarray(c)).cuda()
    y64 = w.h_apply(x, precision=wb.WEST_FP64).cpu().numpy()
    y8 = w.h_apply(x, precision=wb.WEST_FP64_I8).cpu().numpy()
    H = oham.dense_h(p.miller, p.L, p.N, p.vloc, p.beta, p.dcoef)
    ref = (H @ c_full.T).T[:, sel]
    assert relmax(y64, ref) < 1e-12
    assert relmax(y8, ref) < 1e-12
    assert relmax(y8, y64) < 1e-13
    w.close()


@pytest.mark.parametrize("name,omegas,solver", [("cfg1", None, 0), ("mini2", None, 0), ("mini3", None, 0), ("mini3", [0.0, 0.05, 5.0], 1), ("mini2", None, 2)])
def test_chi0_i8_matches_the_sum_over_states(name, omegas, solver):
    import torch
    import paper_2203_05623_b200 as wb
    p = oracle_problem.build(name)
    w, sel = make_west(p)
    dV = torch.from_numpy(np.ascontiguousarray(p.dV)).cuda()
    om = p.omegas if omegas is None else omegas
    dn, dpsi, st = w.chi0_apply(dV, om, tol=1e-12, max_iter=3000, alpha_pv=p.alpha, precision=wb.WEST_FP64_I8, solver=solver)
    ref = ochi0.chi0_sum_over_states(p.eps, p.U, p.n_occ, p.dV, om, p.miller, p.L, p.N)
    assert st["rc"] == 0 and st["n_unconverged"] == 0
    assert relmax(dn.cpu().numpy(), ref) < 1e-9
    dn64, _, st64 = w.chi0_apply(dV, om, tol=1e-12, max_iter=3000, alpha_pv=p.alpha, solver=solver)
    assert relmax(dn.cpu().numpy(), dn64.cpu().numpy()) < 1e-10
    assert abs(st["iters"] - st64["iters"]) <= 1
    w.close()


def test_h_apply_i8_cfg2_size():
    """72^3 grid, 9139 Gamma plane waves, 256 projectors: 300 vectors (ragged tile tail), against the DMMA path and, for four of them,
    the oracle's matrix-free H."""
    import torch
    import paper_2203_05623_b200 as wb
    p = oracle_problem.build("cfg2", dense=False)
    w = wb.West(p.L, p.n2max, p.N, wb.WEST_GAMMA)
    w.set_vloc(torch.from_numpy(np.ascontiguousarray(p.vloc)).cuda())
    w.set_kb(torch.from_numpy(np.ascontiguousarray(p.beta[:, p.half])).cuda(), p.dcoef)
    c, c_full = random_vectors(p, 300, seed=32)
    x = torch.from_numpy(np.ascontiguousarray(c)).cuda()
    y64 = w.h_apply(x, precision=wb.WEST_FP64).cpu().numpy()
    y8 = w.h_apply(x, precision=wb.WEST_FP64_I8).cpu().numpy()
    assert relmax(y8, y64) < 1e-13
    for v in (0, 127, 128, 299):
        ref = oham.apply_h(c_full[v], p.miller, p.L, p.N, p.vloc, p.beta, p.dcoef)[p.half]
        assert relmax(y8[v], ref) < 1e-12
    w.close()


@pytest.mark.parametrize("name", ["mini2", "mini48"])
def test_chi0_i8_six_slices_at_a_loose_tolerance(name):
    """west.h: with tol >= 1e-9 the int8 path cuts every operand row into 6 slices (2^-42 of the row maxima).  The solve must behave as
    the DMMA solve at the same tolerance: same iteration count (+-1), both within the tolerance's reach of the sum over states, and close
    to each other far below it."""
    import torch
    import paper_2203_05623_b200 as wb
    p = oracle_problem.build(name)
    w, sel = make_west(p)
    dV = torch.from_numpy(np.ascontiguousarray(p.dV)).cuda()
    ref = ochi0.chi0_sum_over_states(p.eps, p.U, p.n_occ, p.dV, [0.0], p.miller, p.L, p.N)
    dn8, _, st8 = w.chi0_apply(dV, [0.0], tol=1e-8, max_iter=500, alpha_pv=p.alpha, precision=wb.WEST_FP64_I8, check_every=1)
    dn64, _, st64 = w.chi0_apply(dV, [0.0], tol=1e-8, max_iter=500, alpha_pv=p.alpha, check_every=1)
    assert st8["rc"] == 0 and st64["rc"] == 0 and abs(st8["iters"] - st64["iters"]) <= 1
    e8, e64 = relmax(dn8.cpu().numpy(), ref), relmax(dn64.cpu().numpy(), ref)
    assert e8 < 1e-6 and e64 < 1e-6
    assert relmax(dn8.cpu().numpy(), dn64.cpu().numpy()) < 1e-7
    w.close()
