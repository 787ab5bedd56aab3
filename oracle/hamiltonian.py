"""Steps a2-a6: the Kohn-Sham-like Hamiltonian H = T + V_loc + V_NL in the plane-wave basis.

"the kinetic operator and the local potential are applied in the reciprocal or direct space,
respectively ... at least two FFTs (one forward and one backward) are required at every application
of the KS Hamiltonian" (dual-space technique).  Eq. 1 names the terms;
here they are synthetic (readings A10/A12): T(G) = |G|^2 (Ry), V_loc a real grid function,
V_NL = sum_k |beta_k> D_k <beta_k| (Kleinman-Bylander).

Conventions (A10): G->r is unscaled with exp(+i G.r); r->G carries 1/N^3 and exp(-i G.r).
Coefficients c(G) are normalised sum_G |c|^2 = 1, so psi(r) = u(r)/sqrt(Omega) with u = to_real_space(c).

Two independent statements of the same operator live here on purpose:
  dense_h      - the matrix, by index arithmetic on the DFT of the grid array V_loc
  apply_h      - matrix-free, through scipy.fft (pocketfft; the library FFT is a step, not the oracle)
tests/test_oracle_hamiltonian.py checks one against the other and both against closed forms.
"""
import numpy as np
import scipy.fft as sfft

from . import gsphere


def scatter(c, fft_idx, N):
    """Sphere coefficients [..., n_g] -> zero-padded grid [..., N, N, N]."""
    c = np.asarray(c)
    grid = np.zeros(c.shape[:-1] + (N * N * N,), dtype=np.complex128)
    grid[..., fft_idx] = c
    return grid.reshape(c.shape[:-1] + (N, N, N))


def gather(grid, fft_idx):
    g = np.asarray(grid)
    N = g.shape[-1]
    return g.reshape(g.shape[:-3] + (N * N * N,))[..., fft_idx]


def to_real_space(c, fft_idx, N):
    """u(r_j) = sum_G c(G) exp(+i G.r_j), unscaled."""
    return sfft.ifftn(scatter(c, fft_idx, N), axes=(-3, -2, -1), workers=-1) * float(N) ** 3


def to_g_space(f, fft_idx):
    """c(G) = (1/N^3) sum_j f(r_j) exp(-i G.r_j), truncated to the sphere."""
    N = f.shape[-1]
    return gather(sfft.fftn(f, axes=(-3, -2, -1), workers=-1), fft_idx) / float(N) ** 3


def dense_h(miller, L, N, vloc, beta, dcoef):
    """H[n, n'] = |G_n|^2 delta_nn' + Vt[(n - n') mod N] + sum_k beta_k(n) D_k conj(beta_k(n')),
    Vt = fftn(V_loc)/N^3 (the DFT of the grid array itself, so the matrix IS the dual-space operator)."""
    m = np.asarray(miller, dtype=np.int64)
    n_g = len(m)
    vt = np.fft.fftn(vloc) / float(N) ** 3
    d = (m[:, None, :] - m[None, :, :]) % N
    H = vt[d[..., 0], d[..., 1], d[..., 2]].astype(np.complex128)
    H[np.arange(n_g), np.arange(n_g)] += gsphere.g2_of(m, L)
    if beta is not None and len(beta):
        b = np.asarray(beta)
        H += (b.T * np.asarray(dcoef)[None, :]) @ np.conj(b)
    return H


def apply_h(c, miller, L, N, vloc, beta, dcoef):
    """Matrix-free H c for c[..., n_g] (full-sphere coefficients)."""
    c = np.asarray(c, dtype=np.complex128)
    idx = gsphere.fft_index(miller, N)
    out = gsphere.g2_of(miller, L) * c
    out = out + to_g_space(vloc * to_real_space(c, idx, N), idx)
    if beta is not None and len(beta):
        b = np.asarray(beta)
        proj = c @ np.conj(b).T                      # <beta_k | c>
        out = out + (proj * np.asarray(dcoef)) @ b
    return out


def real_basis(miller):
    """Unitary Q (n_g x n_g) from plane waves to the cos/sin basis of real functions (reading A6):
    column for G = 0 is |0>; for each G in the open half sphere the pair (|G> + |-G>)/sqrt2 and
    (|G> - |-G>)/(i sqrt2).  Q^H H Q is real symmetric when V_loc and the projectors are real in r-space."""
    m = np.asarray(miller)
    n_g = len(m)
    minus = gsphere.index_of_minus(m)
    half = np.nonzero(gsphere.half_sphere_mask(m))[0]
    Q = np.zeros((n_g, n_g), dtype=np.complex128)
    col = 0
    s = 1.0 / np.sqrt(2.0)
    for i in half:
        j = minus[i]
        if i == j:
            Q[i, col] = 1.0
            col += 1
        else:
            Q[i, col] = s
            Q[j, col] = s
            col += 1
            Q[i, col] = -1j * s
            Q[j, col] = 1j * s
            col += 1
    assert col == n_g
    return Q


def eigensystem(H, miller=None, real_orbitals=False):
    """Step 3 of SURVEY.md 8(c): eigh(H) -> eps ascending, columns U.

    With real_orbitals (Gamma mode, reading A6) the diagonalisation is done in the cos/sin basis so every
    eigenvector is a real function of r whatever the degeneracies are."""
    if not real_orbitals:
        eps, U = np.linalg.eigh(H)
        return eps, U
    Q = real_basis(miller)
    Hr = Q.conj().T @ H @ Q
    assert np.max(np.abs(Hr.imag)) < 1e-9 * max(1.0, np.max(np.abs(Hr.real))), "H is not real in r-space"
    eps, Y = np.linalg.eigh(np.ascontiguousarray(Hr.real))
    return eps, Q @ Y
