"""Lanczos chains of the wfreq step, Eq. 15-18, one chain per (perturbation m, orbital i), step by step.

    q^0 = 0,  q^1 = psi_i phi_m                                  (Eq. 16; reading R16: normalised, the norm is returned)
    alpha^l   = <q^l | h | q^l>                                   (Eq. 17)
    beta^{l+1} = || (h - alpha^l) q^l - beta^l q^{l-1} ||          (Eq. 18)
    q^{l+1}   = [(h - alpha^l) q^l - beta^l q^{l-1}] / beta^{l+1}  (Eq. 15)
and the brakets <q^1_{n i} | q^l_{m i}> of Eq. 19 (the GEMM of Fig. 4).
Plain textbook recurrence, no re-orthogonalisation (the paper's Eq. 15 has none).  Test infrastructure, like the rest of oracle/.
Pins (tests/test_oracle_lanczos.py): Lanczos relation against the dense H, moment matching e1^T T^k e1 = <q1|H^k|q1> for k < 2L,
exhaustion of an exactly 5-dimensional Krylov space, and the resolvent identity behind Eq. 19.
"""
import numpy as np

from . import hamiltonian as ham


def start_vectors(U_occ, phi, fft_idx, N):
    """q1[m, i, :] = (phi_m psi_i)(G) on the sphere, normalised; returns q1, norms.  U_occ[n_g, n_occ], phi[n_pert, N, N, N] real."""
    u = ham.to_real_space(U_occ.T, fft_idx, N)                       # [n_occ, N, N, N]
    q1 = np.stack([ham.to_g_space(phi[m][None] * u, fft_idx) for m in range(len(phi))])
    nrm = np.sqrt(np.sum(np.abs(q1) ** 2, axis=-1))
    return q1 / nrm[..., None], nrm


def chain(apply_H, q1, n_steps, keep_vectors=False):
    """One chain.  Returns alpha[n_steps], beta[n_steps] (beta[l] = beta^{l+2}, the norm computed in step l) and, if asked, the
    vectors q^1 .. q^{n_steps}."""
    alpha, beta = np.zeros(n_steps), np.zeros(n_steps)
    q_prev = np.zeros_like(q1)
    q = q1.copy()
    b_prev = 0.0
    Q = [q.copy()] if keep_vectors else None
    for l in range(n_steps):
        hq = apply_H(q)
        a = np.vdot(q, hq).real
        w = hq - a * q - b_prev * q_prev
        b = np.linalg.norm(w)
        alpha[l], beta[l] = a, b
        q_prev, q, b_prev = q, w / b, b
        if keep_vectors and l + 1 < n_steps:
            Q.append(q.copy())
    return (alpha, beta, np.array(Q)) if keep_vectors else (alpha, beta)


def chains_with_brakets(apply_H, q1, n_steps):
    """All chains of q1[n_pert, n_occ, n_g]; brakets[i, l, n, m] = <q^1_{n i} | q^{l+1}_{m i}>."""
    n_pert, n_occ, _ = q1.shape
    alpha = np.zeros((n_pert, n_occ, n_steps))
    beta = np.zeros((n_pert, n_occ, n_steps))
    brak = np.zeros((n_occ, n_steps, n_pert, n_pert), dtype=np.complex128)
    for i in range(n_occ):
        Qs = []
        for m in range(n_pert):
            alpha[m, i], beta[m, i], Q = chain(apply_H, q1[m, i], n_steps, keep_vectors=True)
            Qs.append(Q)                                             # [n_steps, n_g]
        Qs = np.array(Qs)                                            # [m, l, g]
        brak[i] = np.einsum("ng,mlg->lnm", np.conj(q1[:, i]), Qs)
    return alpha, beta, brak


def tridiagonal(alpha, beta):
    """T_L with alpha on the diagonal and beta^2..beta^L on the off-diagonals (beta[l] = beta^{l+2})."""
    L = len(alpha)
    T = np.diag(alpha)
    for l in range(L - 1):
        T[l, l + 1] = T[l + 1, l] = beta[l]
    return T


def eig_tridiagonal(alpha, beta):
    """d^{l'} and U^{l l'} of Eq. 19: eigenvalues (ascending) and orthonormal eigenvectors (columns) of the tridiagonal
    matrix with alpha^l on the diagonal and beta^l on the sub- and super-diagonal, T = U diag(d) U^T.  LAPACK through numpy.linalg.eigh
    is the step; the sign of each eigenvector is fixed by U[0, l'] >= 0 (the first component of an eigenvector of an unreduced
    tridiagonal matrix is never zero), which is what makes U unique when the eigenvalues are simple."""
    T = tridiagonal(np.asarray(alpha, dtype=np.float64), np.asarray(beta, dtype=np.float64))
    d, U = np.linalg.eigh(T)
    U = U * np.where(U[0] < 0, -1.0, 1.0)[None, :]
    return d, U


def resolvent_column(alpha, beta, z):
    """x = (T - z)^{-1} e_1 by a dense solve: the vector Eq. 19 evaluates as x_l = sum_l' U^{l l'} U^{1 l'} / (d^{l'} - z)."""
    T = tridiagonal(np.asarray(alpha, dtype=np.float64), np.asarray(beta, dtype=np.float64)).astype(np.complex128)
    e1 = np.zeros(len(alpha), dtype=np.complex128); e1[0] = 1.0
    return np.linalg.solve(T - z * np.eye(len(alpha)), e1)
