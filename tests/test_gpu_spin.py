"""Spin-polarised chi0*dV (N_spin = 2) through the C ABI against oracle.chi0.chi0_spin_polarised:
one context per channel (its own V_loc^sigma and orbitals), occupation 1, the second call accumulating into the first call's dn."""
import numpy as np
import pytest

import oracle_problem
import synth
from gpu_common import relmax
from oracle import chi0 as ochi0
from oracle import hamiltonian as oham

pytestmark = pytest.mark.gpu


def _channels(p, occs):
    """Per channel: (eps, U, n_occ, vloc) from the dense oracle eigensystem of h^sigma = T + V_loc +- B + V_NL."""
    B = synth.spin_splitting_field(p.cfg)
    out = []
    for sgn, n_occ in zip((+1, -1), occs):
        vloc = p.vloc + sgn * B
        H = oham.dense_h(p.miller, p.L, p.N, vloc, p.beta, p.dcoef)
        eps, U = oham.eigensystem(H, p.miller, real_orbitals=p.gamma)
        out.append((eps, U, n_occ, vloc))
    return out


def _contexts(p, ch):
    import torch
    import paper_2203_05623_b200 as wb
    sel = p.half if p.gamma else np.arange(p.n_full)
    ws = []
    for eps, U, n_occ, vloc in ch:
        w = wb.West(p.L, p.n2max, p.N, wb.WEST_GAMMA if p.gamma else wb.WEST_FULL)
        w.set_vloc(torch.from_numpy(np.ascontiguousarray(vloc)).cuda())
        w.set_kb(torch.from_numpy(np.ascontiguousarray(p.beta[:, sel])).cuda(), p.dcoef)
        w.set_states(torch.from_numpy(np.ascontiguousarray(U[:, :n_occ].T[:, sel])).cuda(), eps[:n_occ])
        ws.append(w)
    return ws


@pytest.mark.parametrize("name,occs,omegas", [("cfg1", (9, 7), [0.0]), ("mini2", (16, 16), [0.0, 0.5]), ("mini2", (22, 14), [0.0])])
def test_spin_polarised_chi0_matches_the_oracle(name, occs, omegas):
    import torch
    import paper_2203_05623_b200 as wb
    p = oracle_problem.build(name)
    ch = _channels(p, occs)
    ref = ochi0.chi0_spin_polarised([c[:3] for c in ch], p.dV, omegas, p.miller, p.L, p.N)
    ws = _contexts(p, ch)
    alphas = [ochi0.default_alpha(c[0], c[2]) for c in ch]
    dV = torch.from_numpy(p.dV).cuda()
    dn, stats = wb.West.chi0_apply_spin(ws, dV, omegas, tol=1e-12, max_iter=2000, alpha_pv=alphas)
    assert all(st["rc"] == 0 and st["n_unconverged"] == 0 for st in stats)
    assert relmax(dn.cpu().numpy(), ref) < 1e-9
    # each channel alone, occupation 1, equals half of the same context's unpolarised (occupation 2) answer
    a, _, _ = ws[0].chi0_apply(dV, omegas, tol=1e-12, max_iter=2000, alpha_pv=alphas[0], occupation=1.0)
    b, _, _ = ws[0].chi0_apply(dV, omegas, tol=1e-12, max_iter=2000, alpha_pv=alphas[0])
    assert relmax((2 * a).cpu().numpy(), b.cpu().numpy()) < 1e-12
    for w in ws:
        w.close()


def test_identical_channels_reduce_to_the_unpolarised_result_and_bad_options_are_refused():
    import torch
    import paper_2203_05623_b200 as wb
    from gpu_common import make_west
    p = oracle_problem.build("mini2")
    w, _ = make_west(p)
    dV = torch.from_numpy(p.dV[:2]).cuda()
    unpol, _, _ = w.chi0_apply(dV, [0.0], tol=1e-12, alpha_pv=p.alpha)
    both, _ = wb.West.chi0_apply_spin([w, w], dV, [0.0], tol=1e-12, alpha_pv=p.alpha)
    assert relmax(both.cpu().numpy(), unpol.cpu().numpy()) < 1e-13
    with pytest.raises(wb.WestError) as e:
        w.chi0_apply(dV, [0.0], occupation=3.0)
    assert e.value.code == wb.binding.WEST_EINVAL
    w.close()
