"""The iterative route of the paper, step by step, for sizes where the dense oracle does not fit.

"A preconditioned conjugate gradient method is used to solve equation 10".  The paper states
neither the preconditioner, the alpha P_v shift nor the threshold; the readings are A3-A5 and A7 of
SURVEY.md 8(c) / DESIGN.md:

    operator   A_v = H - eps_v - i omega + alpha P_v            (A3)
    M_v(G)     = 1 / max(1, |G|^2 / (1.35 <psi_v|T|psi_v>))      (A4)
    stop       ||r||_2 / ||b||_2 <= tol per column               (A5)
    i omega    COCG: textbook PCG with the unconjugated bilinear form (x, y) = sum_G x(-G) y(G)   (A7)

These are textbook recurrences (Hestenes-Stiefel PCG; van der Vorst-Melissen COCG) written in their usual
order with no blocking or fusion.  tests/test_oracle_iterative.py pins them to chi0.chi0_sum_over_states
(the plain definition) and to the true residual recomputed with the dense matrix.

``lowest_states`` produces the occupied orbitals (inputs of Eq. 10) for cells whose dense matrix is too
large to diagonalise in a test: LOBPCG (scipy, a library eigensolver) on the matrix-free apply_h in the
real cos/sin representation, accepted only if every eigen-residual passes the stated threshold.
"""
import numpy as np
import scipy.sparse.linalg as spla

from . import gsphere
from . import hamiltonian as ham


def kinetic_expectation(U_occ, g2):
    """<psi_v|T|psi_v> for columns of U_occ[n_g, n_v]."""
    return np.real(np.sum(np.conj(U_occ) * (g2[:, None] * U_occ), axis=0))


def preconditioner(g2, tk_v):
    return 1.0 / np.maximum(1.0, g2 / (1.35 * tk_v))


def pcg_sternheimer(apply_H, U_occ, eps_v, v, b, g2, alpha, tol=1e-12, max_iter=500):
    """omega = 0: solve (H - eps_v + alpha P_v) x = -(1 - P_v) b for one column by PCG.  Returns x, iters, relres."""
    Pv = lambda y: U_occ @ (U_occ.conj().T @ y)
    A = lambda y: apply_H(y) - eps_v * y + alpha * Pv(y)
    Mdiag = preconditioner(g2, kinetic_expectation(U_occ, g2)[v])
    rhs = -(b - Pv(b))
    x = np.zeros_like(rhs)
    r = rhs.copy()
    z = Mdiag * r
    p = z.copy()
    rz = np.vdot(r, z).real
    bnorm = np.linalg.norm(rhs)
    if bnorm == 0.0:
        return x, 0, 0.0
    it = 0
    while it < max_iter and np.linalg.norm(r) > tol * bnorm:
        Ap = A(p)
        a = rz / np.vdot(p, Ap).real
        x = x + a * p
        r = r - a * Ap
        z = Mdiag * r
        rz_new = np.vdot(r, z).real
        p = z + (rz_new / rz) * p
        rz = rz_new
        it += 1
    return x, it, np.linalg.norm(r) / bnorm


def cocg_sternheimer(apply_H, U_occ, eps_v, v, b, g2, minus, alpha, omega, tol=1e-12, max_iter=500):
    """i omega: solve (H - eps_v - i omega + alpha P_v) x = -(1 - P_v) b by COCG with (x, y) = sum_G x(-G) y(G).

    Valid when H and P_v are real-symmetric in real space (real V_loc, real-in-r projectors, real orbitals)."""
    Pv = lambda y: U_occ @ (U_occ.conj().T @ y)
    A = lambda y: apply_H(y) - (eps_v + 1j * omega) * y + alpha * Pv(y)
    bil = lambda x, y: np.sum(x[minus] * y)
    Mdiag = preconditioner(g2, kinetic_expectation(U_occ, g2)[v])
    rhs = -(b - Pv(b))
    x = np.zeros_like(rhs)
    r = rhs.copy()
    z = Mdiag * r
    p = z.copy()
    rz = bil(r, z)
    bnorm = np.linalg.norm(rhs)
    if bnorm == 0.0:
        return x, 0, 0.0
    it = 0
    while it < max_iter and np.linalg.norm(r) > tol * bnorm:
        Ap = A(p)
        a = rz / bil(p, Ap)
        x = x + a * p
        r = r - a * Ap
        z = Mdiag * r
        rz_new = bil(r, z)
        p = z + (rz_new / rz) * p
        rz = rz_new
        it += 1
    return x, it, np.linalg.norm(r) / bnorm


def lowest_states(n_states, miller, L, N, vloc, beta, dcoef, tol=1e-9, max_iter=400, n_guard=None, seed=7):
    """Lowest n_states eigenpairs of H as REAL orbitals (c(-G) = conj c(G)), by LOBPCG in the cos/sin basis.

    Works on half-sphere real coordinates y (length n_g_full): y -> c (complex, full sphere) -> apply_h -> back.
    Returns eps[n_states], U[n_g_full, n_states], max eigen-residual; raises if the residual exceeds tol*10."""
    m = np.asarray(miller)
    n_g = len(m)
    minus = gsphere.index_of_minus(m)
    half = np.nonzero(gsphere.half_sphere_mask(m))[0]
    i0 = [i for i in half if minus[i] == i]
    assert len(i0) == 1
    pos = np.array([i for i in half if minus[i] != i])
    neg = minus[pos]
    zero = i0[0]
    s = 1.0 / np.sqrt(2.0)
    n_pos = len(pos)

    def to_c(Y):                                   # Y[n_g, k] real -> C[k, n_g] complex
        Y = np.asarray(Y)
        C = np.zeros((Y.shape[1], n_g), dtype=np.complex128)
        C[:, zero] = Y[0]
        a, bb = Y[1:1 + n_pos].T, Y[1 + n_pos:].T
        C[:, pos] = s * (a - 1j * bb)
        C[:, neg] = s * (a + 1j * bb)
        return C

    def to_y(C):                                   # inverse of to_c for real functions
        Y = np.empty((n_g, C.shape[0]))
        Y[0] = C[:, zero].real
        Y[1:1 + n_pos] = (np.sqrt(2.0) * C[:, pos].real).T
        Y[1 + n_pos:] = (-np.sqrt(2.0) * C[:, pos].imag).T
        return Y

    def matmat(Y):
        Y = Y.reshape(n_g, -1)
        return to_y(ham.apply_h(to_c(Y), m, L, N, vloc, beta, dcoef))

    g2 = gsphere.g2_of(m, L)
    g2y = np.concatenate([[g2[zero]], g2[pos], g2[pos]])
    prec = 1.0 / np.maximum(1.0, g2y)              # Teter-like diagonal; affects iterations only

    n_guard = max(8, n_states // 8) if n_guard is None else n_guard
    k = n_states + n_guard
    rng = np.random.Generator(np.random.PCG64(seed))
    X = rng.standard_normal((n_g, k)) * prec[:, None]
    Aop = spla.LinearOperator((n_g, n_g), matvec=matmat, matmat=matmat, dtype=np.float64)
    Mop = spla.LinearOperator((n_g, n_g), matvec=lambda y: prec * y.reshape(-1),
                              matmat=lambda Y: prec[:, None] * Y, dtype=np.float64)
    w, V = spla.lobpcg(Aop, X, M=Mop, tol=tol * 0.1, maxiter=max_iter, largest=False)
    order = np.argsort(w)[:n_states]
    w, V = w[order], V[:, order]
    U = to_c(V).T
    R = ham.apply_h(U.T, m, L, N, vloc, beta, dcoef).T - U * w[None, :]
    res = float(np.max(np.linalg.norm(R, axis=0)))
    if not res < 10.0 * tol:
        raise RuntimeError(f"lowest_states: eigen-residual {res:.3e} above {10 * tol:.1e}")
    return w, U, res
