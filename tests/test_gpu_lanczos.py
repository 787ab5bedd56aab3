"""GPU parity of west_lanczos (Eq. 15-19) against oracle/lanczos.py."""
import numpy as np
import pytest

import oracle_problem
from gpu_common import make_west, relmax
from oracle import hamiltonian as oham
from oracle import lanczos as olz

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("name,n_steps", [("cfg1", 20), ("mini2", 30)])
def test_lanczos_chains_and_brakets(name, n_steps):
    import torch
    p = oracle_problem.build(name)
    w, sel = make_west(p)
    n_pert = 3
    phi = np.ascontiguousarray(p.dV[:n_pert])
    a, b, nrm, br = w.lanczos(torch.from_numpy(phi).cuda(), n_steps, p.n_occ, want_brakets=p.gamma)
    q1, nrm_ref = olz.start_vectors(p.U[:, :p.n_occ], phi, p.fft_idx, p.N)
    apply_H = lambda y: p.H @ y
    assert relmax(nrm.cpu().numpy(), nrm_ref) < 1e-12
    if p.gamma:
        ar, brf, brak = olz.chains_with_brakets(apply_H, q1, n_steps)
        got = br.cpu().numpy()                                   # [i][l][n][m], real for real functions
        assert np.max(np.abs(brak.imag)) < 1e-10
        assert np.max(np.abs(got - brak.real)) < 1e-9
    else:
        ar = np.zeros((n_pert, p.n_occ, n_steps)); brf = np.zeros_like(ar)
        for m in range(n_pert):
            for i in range(p.n_occ):
                ar[m, i], brf[m, i] = olz.chain(apply_H, q1[m, i], n_steps)
    assert relmax(a.cpu().numpy(), ar) < 1e-9
    assert relmax(b.cpu().numpy(), brf) < 1e-9
    w.close()


def test_lanczos_cfg2_size_sampled_chains():
    """Config-2 size (72^3, 9139 plane waves) with library-generated orbitals CHECKED by the oracle (as in test_gpu_cfg5.py): sampled
    chains against the oracle's matrix-free recurrence on the same start vectors."""
    import torch
    import synth
    import paper_2203_05623_b200 as wb
    from paper_2203_05623_b200 import eigs
    from oracle import gsphere as ogs
    p = oracle_problem.build("cfg2", dense=False)
    w = wb.West(p.L, p.n2max, p.N, wb.WEST_GAMMA)
    dev = torch.device("cuda:0")
    w.set_vloc(torch.from_numpy(np.ascontiguousarray(p.vloc)).to(dev))
    w.set_kb(torch.from_numpy(np.ascontiguousarray(p.beta[:, p.half])).to(dev), p.dcoef)
    eps, psi, res = eigs.lowest_states(w, p.n_occ, tol=1e-9)
    w.set_states(psi, eps[:p.n_occ])
    n_pert, L = 4, 30
    phi = np.ascontiguousarray(p.dV[:n_pert])
    a, b, nrm, br = w.lanczos(torch.from_numpy(phi).to(dev), L, p.n_occ, want_brakets=True)
    U = ogs.expand_half_to_full(psi.cpu().numpy(), p.miller).T
    apply_H = lambda y: oham.apply_h(y, p.miller, p.L, p.N, p.vloc, p.beta, p.dcoef)
    for m, i in ((0, 0), (3, 127), (2, 64)):
        q1, n1 = olz.start_vectors(U[:, i:i + 1], phi[m:m + 1], p.fft_idx, p.N)
        ar, brf = olz.chain(apply_H, q1[0, 0], L)
        assert abs(float(nrm[m, i]) - n1[0, 0]) < 1e-12 * n1[0, 0]
        assert relmax(a[m, i].cpu().numpy(), ar) < 1e-9 and relmax(b[m, i].cpu().numpy(), brf) < 1e-9
    # braket of step 0 is the Gram matrix of the start vectors of one orbital
    q1, _ = olz.start_vectors(U[:, 5:6], phi, p.fft_idx, p.N)
    G = (np.conj(q1[:, 0]) @ q1[:, 0].T).real
    assert np.max(np.abs(br[5, 0].cpu().numpy() - G)) < 1e-10
    w.close()
