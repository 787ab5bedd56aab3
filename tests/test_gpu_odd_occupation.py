"""WEST_GAMMA with an ODD number of occupied orbitals (reading R15: the library appends one zero orbital internally; spin channels
often have odd counts).  chi0 (PCG, COCG, multi-shift), dpsi in the caller's layout, Lanczos chains and brakets against the oracle."""
import numpy as np
import pytest

import oracle_problem
from gpu_common import relmax
from oracle import chi0 as ochi0
from oracle import gsphere as ogs
from oracle import lanczos as olz

pytestmark = pytest.mark.gpu


def _west(p, n_occ):
    import torch
    import paper_2203_05623_b200 as wb
    w = wb.West(p.L, p.n2max, p.N, wb.WEST_GAMMA)
    w.set_vloc(torch.from_numpy(np.ascontiguousarray(p.vloc)).cuda())
    w.set_kb(torch.from_numpy(np.ascontiguousarray(p.beta[:, p.half])).cuda(), p.dcoef)
    w.set_states(torch.from_numpy(np.ascontiguousarray(p.U[:, :n_occ].T[:, p.half])).cuda(), p.eps[:n_occ])
    return w


@pytest.mark.parametrize("name,n_occ,omegas,solver", [("mini2", 13, [0.0], 0), ("mini2", 7, [0.0, 0.6], 0), ("tinyg", 5, [0.05, 0.5, 2.0], 1),
                                                      ("tinyg", 1, [0.0], 0)])
def test_chi0_with_an_odd_number_of_orbitals(name, n_occ, omegas, solver):
    import torch
    p = oracle_problem.build(name)
    w = _west(p, n_occ)
    alpha = ochi0.default_alpha(p.eps, n_occ)
    dV = torch.from_numpy(p.dV[:3]).cuda()
    dn, dpsi, st = w.chi0_apply(dV, omegas, tol=1e-12, max_iter=3000, alpha_pv=alpha, solver=solver, want_dpsi=True, n_occ=n_occ)
    ref_dn, ref_dpsi = ochi0.chi0_sum_over_states(p.eps, p.U, n_occ, p.dV[:3], omegas, p.miller, p.L, p.N, return_dpsi=True)
    assert st["rc"] == 0 and st["n_unconverged"] == 0
    assert not torch.isnan(dn).any()
    assert relmax(dn.cpu().numpy(), ref_dn) < 1e-9
    d = dpsi.cpu().numpy()                                         # [w][i][n_occ][2][n_g], the caller's n_occ
    assert d.shape[2] == n_occ
    full = ogs.expand_half_to_full(d[..., 0, :], p.miller) + 1j * ogs.expand_half_to_full(d[..., 1, :], p.miller)
    assert relmax(full, ref_dpsi) < 1e-9
    w.close()


def test_lanczos_with_an_odd_number_of_orbitals():
    import torch
    p = oracle_problem.build("mini2")
    n_occ, n_steps, n_pert = 7, 12, 3
    w = _west(p, n_occ)
    phi = np.ascontiguousarray(p.dV[:n_pert])
    a, b, nrm, br = w.lanczos(torch.from_numpy(phi).cuda(), n_steps, n_occ, want_brakets=True)
    q1, nrm_ref = olz.start_vectors(p.U[:, :n_occ], phi, p.fft_idx, p.N)
    ar, brf, brak = olz.chains_with_brakets(lambda y: p.H @ y, q1, n_steps)
    assert a.shape == (n_pert, n_occ, n_steps) and br.shape == (n_occ, n_steps, n_pert, n_pert)
    assert relmax(nrm.cpu().numpy(), nrm_ref) < 1e-12
    assert relmax(a.cpu().numpy(), ar) < 1e-9
    assert relmax(b.cpu().numpy(), brf) < 1e-9
    assert np.max(np.abs(br.cpu().numpy() - brak.real)) < 1e-9
    w.close()
