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


def _diag_ctx():
    import paper_2203_05623_b200 as wb
    return wb.West(10.0, 25, 24, wb.WEST_FULL)


def _check_diag(alpha, beta, d, U, tol=1e-12):
    """Against oracle.lanczos.eig_tridiagonal: what is unique (eigenvalues; the spectral sum of Eq. 19) is compared, the rest
    (orthonormal eigenvectors of T, sign convention) is checked for validity; eigenvectors themselves only when the spectrum is simple."""
    for c in range(alpha.shape[0]):
        T = olz.tridiagonal(alpha[c], beta[c])
        scale = max(np.max(np.abs(T)), 1e-300)
        d_ref, U_ref = olz.eig_tridiagonal(alpha[c], beta[c])
        assert np.max(np.abs(d[c] - d_ref)) < tol * scale * len(d_ref)
        assert np.all(np.diff(d[c]) >= 0)
        assert np.max(np.abs(U[c].T @ U[c] - np.eye(len(d_ref)))) < 1e-12
        assert np.max(np.abs(T @ U[c] - U[c] * d[c][None, :])) < 1e-12 * scale * len(d_ref)
        assert np.all(U[c][0] >= 0)
        if len(d_ref) > 1 and np.min(np.diff(d_ref)) > 1e-3 * scale:
            # the sign rule binds only where the first component is not at rounding level; elsewhere compare up to the sign
            fixed = np.abs(U_ref[0]) > 1e-8
            assert np.max(np.abs(U[c][:, fixed] - U_ref[:, fixed])) < 1e-9
            sgn = np.sign(np.sum(U[c] * U_ref, axis=0))
            assert np.max(np.abs(U[c] * sgn[None, :] - U_ref)) < 1e-9
        for z in (0.3j, 0.1 + 2.0j):
            x = (U[c] * U[c][0][None, :]) @ (1.0 / (d[c] - z))
            assert np.max(np.abs(x - olz.resolvent_column(alpha[c], beta[c], z))) < 1e-11


@pytest.mark.parametrize("n", [1, 2, 7, 30, 33, 64])
def test_tridiagonal_eigensolver_random_and_special_matrices(n):
    import torch
    rng = np.random.Generator(np.random.PCG64(100 + n))
    n_chain = 37
    alpha = rng.standard_normal((n_chain, n))
    beta = np.abs(rng.standard_normal((n_chain, n))) + 0.05
    alpha[0], beta[0] = 0.3, 0.7                                   # Toeplitz: closed-form spectrum
    if n > 4:
        beta[1, n // 2] = 0.0                                      # reducible: two independent blocks
        alpha[2] = 1.0; beta[2] = 1e-9                             # nearly diagonal, clustered eigenvalues
        beta[3] *= 1e3; alpha[3] *= 1e-3                           # badly scaled
    w = _diag_ctx()
    d, U, sw = w.lanczos_diag(torch.from_numpy(alpha).cuda(), torch.from_numpy(beta).cuda(), want_sweeps=True)
    assert int(sw.min()) >= 0
    d, U = d.cpu().numpy(), U.cpu().numpy()
    if n > 4:
        # row 1 is reducible: first components of the second block's eigenvectors are exactly zero, the sign rule does not bind
        keep = [c for c in range(n_chain) if c != 1]
        T = olz.tridiagonal(alpha[1], beta[1])
        assert np.max(np.abs(np.sort(np.linalg.eigvalsh(T)) - d[1])) < 1e-12 * n
        assert np.max(np.abs(T @ U[1] - U[1] * d[1][None, :])) < 1e-12 * n
    else:
        keep = list(range(n_chain))
    _check_diag(alpha[keep], beta[keep], d[keep], U[keep])
    k = np.arange(1, n + 1)
    assert np.max(np.abs(d[0] - np.sort(0.3 + 1.4 * np.cos(k * np.pi / (n + 1))))) < 1e-13 * n
    w.close()


def test_tridiagonal_eigensolver_on_real_chains_and_errors():
    """alpha, beta of oracle chains (cfg 1, 30 steps, where orthogonality is already lost and Ritz values cluster) as the input of both sides."""
    import torch
    import paper_2203_05623_b200 as wb
    p = oracle_problem.build("cfg1")
    q1, _ = olz.start_vectors(p.U[:, :p.n_occ], p.dV[:2], p.fft_idx, p.N)
    ab = [olz.chain(lambda y: p.H @ y, q1[m, i], 30) for m in range(2) for i in range(p.n_occ)]
    alpha = np.array([x[0] for x in ab]); beta = np.array([x[1] for x in ab])
    w = _diag_ctx()
    d, U = w.lanczos_diag(torch.from_numpy(alpha).cuda(), torch.from_numpy(beta).cuda())
    _check_diag(alpha, beta, d.cpu().numpy(), U.cpu().numpy())
    with pytest.raises(wb.WestError) as e:
        w.lanczos_diag(torch.zeros((2, 65), dtype=torch.float64, device="cuda"), torch.zeros((2, 65), dtype=torch.float64, device="cuda"))
    assert e.value.code == wb.binding.WEST_EINVAL
    d0, U0 = w.lanczos_diag(torch.zeros((0, 30), dtype=torch.float64, device="cuda"), torch.zeros((0, 30), dtype=torch.float64, device="cuda"))
    assert d0.shape == (0, 30) and U0.shape == (0, 30, 30)
    w.close()


def test_lanczos_fp32_operand_brakets():
    """WEST_MIXED: the braket Gram blocks of Eq. 19 / Fig. 4 with FP32 (TF32 hi + lo) operands on the tcgen05 path - the FP32 payload of
    Fig. 5c as an operand format.  FP32-class agreement with the oracle's FP64 brakets; the chains themselves run the
    mixed H*psi and agree to its tolerance."""
    import torch
    import paper_2203_05623_b200 as wb
    p = oracle_problem.build("mini2")
    w, sel = make_west(p)
    n_pert, n_steps = 5, 12
    phi = np.ascontiguousarray(p.dV[:n_pert])
    a, b, nrm, br = w.lanczos(torch.from_numpy(phi).cuda(), n_steps, p.n_occ, want_brakets=True, precision=wb.WEST_MIXED)
    a64, b64, _, br64 = w.lanczos(torch.from_numpy(phi).cuda(), n_steps, p.n_occ, want_brakets=True)
    q1, _ = olz.start_vectors(p.U[:, :p.n_occ], phi, p.fft_idx, p.N)
    ar, brf, brak = olz.chains_with_brakets(lambda y: p.H @ y, q1, n_steps)
    got = br.cpu().numpy()
    assert np.max(np.abs(br64.cpu().numpy() - brak.real)) < 1e-9
    # step 0 is the Gram matrix of the start vectors: pure operand-format error (no mixed H*psi yet)
    assert 1e-12 < np.max(np.abs(got[:, 0] - brak.real[:, 0])) < 5e-6
    assert np.max(np.abs(got - brak.real)) < 1e-4
    assert relmax(a.cpu().numpy(), ar) < 1e-4
    w.close()
