"""Pins of oracle/lanczos.py (Eq. 15-19) against the dense Hamiltonian and textbook Lanczos identities."""
import numpy as np

import oracle_problem as op
from oracle import lanczos as olz


def _setup():
    p = op.build("cfg1")
    q1, nrm = olz.start_vectors(p.U[:, :p.n_occ], p.dV[:2], p.fft_idx, p.N)
    return p, q1, nrm


def test_lanczos_relation_and_orthonormality_with_dense_h():
    p, q1, _ = _setup()
    H = p.H
    L = 12
    a, b, Q = olz.chain(lambda y: H @ y, q1[1, 3], L, keep_vectors=True)
    T = olz.tridiagonal(a, b)
    # H Q_L = Q_L T_L + beta^{L+1} q^{L+1} e_L^T  (rows of Q are the vectors)
    lhs = (H @ Q.T)
    rhs = Q.T @ T
    resid = lhs - rhs
    assert np.max(np.abs(resid[:, :L - 1])) < 1e-12
    assert abs(np.linalg.norm(resid[:, L - 1]) - b[L - 1]) < 1e-12
    G = Q.conj() @ Q.T
    assert np.max(np.abs(G - np.eye(L))) < 1e-10


def test_moment_matching():
    p, q1, _ = _setup()
    H = p.H
    L = 6
    a, b = olz.chain(lambda y: H @ y, q1[0, 0], L)
    T = olz.tridiagonal(a, b)
    v = q1[0, 0].copy()
    e = np.zeros(L); e[0] = 1.0
    for k in range(2 * L):                                   # e1^T T^k e1 = <q1|H^k|q1> for k = 0 .. 2L-1
        lhs = e @ np.linalg.matrix_power(T, k) @ e
        rhs = np.vdot(q1[0, 0], v).real
        assert abs(lhs - rhs) < 1e-9 * max(1.0, abs(rhs)), k
        v = H @ v


def test_exhaustion_of_a_five_dimensional_krylov_space():
    p, _, _ = _setup()
    c = np.array([0.5, -0.3, 0.7, 0.2, 0.4])
    idx = [1, 4, 9, 20, 33]
    q = p.U[:, idx] @ c
    q /= np.linalg.norm(q)
    a, b = olz.chain(lambda y: p.H @ y, q, 5)
    assert b[4] < 1e-7 * b[0]                                 # the sixth vector vanishes (up to rounding amplified by 1/beta)
    ritz = np.linalg.eigvalsh(olz.tridiagonal(a, b))
    assert np.max(np.abs(ritz - p.eps[idx])) < 1e-9


def test_resolvent_identity_behind_eq19():
    # <q1|(H - z)^-1|q1> = [(T - z)^-1]_11 exactly once the Krylov space is exhausted, and converges with L otherwise
    p, q1, _ = _setup()
    z = -1.0 + 0.7j
    q = q1[1, 0]
    exact = np.vdot(q, np.linalg.solve(p.H - z * np.eye(p.n_full), q))
    errs = []
    for L in (4, 8, 16, 32):
        a, b = olz.chain(lambda y: p.H @ y, q, L)
        T = olz.tridiagonal(a, b)
        errs.append(abs(np.linalg.inv(T - z * np.eye(L))[0, 0] - exact))
    assert errs[-1] < 1e-6 and errs[-1] < errs[1] < errs[0]


def test_brakets_first_step_is_the_gram_matrix_of_the_start_vectors():
    p, q1, _ = _setup()
    a, b, br = olz.chains_with_brakets(lambda y: p.H @ y, q1[:, :2], 3)
    for i in range(2):
        G = np.conj(q1[:, i]) @ q1[:, i].T
        assert np.max(np.abs(br[i, 0] - G)) < 1e-13
        assert np.allclose(np.diag(br[i, 1]), 0.0, atol=1e-12)      # q^2 is orthogonal to q^1


def test_eig_tridiagonal_closed_form_reconstruction_and_resolvent():
    """Toeplitz tridiagonal (a on the diagonal, b beside it): d_k = a + 2 b cos(k pi/(n+1)), U_lk = sqrt(2/(n+1)) sin(l k pi/(n+1));
    then a real chain: T = U d U^T, orthonormality, sign convention, and the spectral sum of Eq. 19 against a dense solve."""
    n, a, b = 9, 0.3, -0.7
    d, U = olz.eig_tridiagonal(np.full(n, a), np.full(n, b))
    k = np.arange(1, n + 1)
    d_ref = np.sort(a + 2 * b * np.cos(k * np.pi / (n + 1)))
    assert np.max(np.abs(d - d_ref)) < 1e-13
    # eigenvector of d = a + 2 b cos(k pi/(n+1)) is sin(l k pi/(n+1)); compare through the projector (sign-free)
    order = np.argsort(a + 2 * b * np.cos(k * np.pi / (n + 1)))
    V = np.sqrt(2.0 / (n + 1)) * np.sin(np.outer(k, k) * np.pi / (n + 1))[:, order]
    assert np.max(np.abs(np.abs(U) - np.abs(V))) < 1e-12
    assert np.all(U[0] >= 0)
    p, q1, _ = _setup()
    al, be = olz.chain(lambda y: p.H @ y, q1[0, 2], 14)
    d, U = olz.eig_tridiagonal(al, be)
    T = olz.tridiagonal(al, be)
    assert np.max(np.abs(U @ np.diag(d) @ U.T - T)) < 1e-12
    assert np.max(np.abs(U.T @ U - np.eye(14))) < 1e-12
    for z in (0.4j, -0.2 + 1.5j):
        x = (U * U[0][None, :]) @ (1.0 / (d - z))
        assert np.max(np.abs(x - olz.resolvent_column(al, be, z))) < 1e-11
