"""PDEP: leading eigenpairs of the symmetrised static response chi0bar = v^1/2 chi0(omega = 0) v^1/2 (Eq. 9),
as its plain definition: the dense matrix in the basis of real potentials on the wavefunction sphere, then LAPACK eigh.

A real potential is phi(r) = sum_G c(G) exp(i G.r) with c(-G) = conj c(G) and no G = 0 term; its real coordinates are
y = (sqrt2 Re c(G), sqrt2 Im c(G)) over the open half sphere, so that <phi, phi'> = sum_G conj(c) c' = y.y'.  v(G) = 8 pi / |G|^2 (Rydberg
units, e^2 = 2).  chi0 acts through oracle.chi0.chi0_sum_over_states (itself pinned in tests/test_oracle_chi0.py):
    chi0bar[y', y] = < phi_y' , v^1/2 P_S [ chi0 ( v^1/2 phi_y ) ] >,   P_S = truncation of the density response to the sphere.
Test infrastructure, like the rest of oracle/.  Pins (tests/test_oracle_pdep.py): symmetry, negative semi-definiteness, agreement of one
column with a finite-field derivative is inherited from chi0's own pins.
"""
import numpy as np

from . import chi0 as ochi0
from . import gsphere as ogs
from . import hamiltonian as ham


def real_basis_size(miller):
    half = np.nonzero(ogs.half_sphere_mask(miller))[0]
    return 2 * (len(half) - 1)


def coeffs_from_y(y, miller):
    """y[..., 2(n_half-1)] -> half-sphere coefficients [..., n_half] (c(0) = 0)."""
    half = np.nonzero(ogs.half_sphere_mask(miller))[0]
    n = len(half) - 1
    c = np.zeros(y.shape[:-1] + (n + 1,), dtype=np.complex128)
    c[..., 1:] = (y[..., :n] + 1j * y[..., n:]) / np.sqrt(2.0)
    return c


def y_from_coeffs(c):
    return np.concatenate([np.sqrt(2.0) * c[..., 1:].real, np.sqrt(2.0) * c[..., 1:].imag], axis=-1)


def sqrt_coulomb(miller, L):
    """v^1/2 on the half sphere (0 at G = 0)."""
    half = np.nonzero(ogs.half_sphere_mask(miller))[0]
    g2 = ogs.g2_of(miller[half], L)
    out = np.zeros(len(half))
    out[1:] = np.sqrt(8.0 * np.pi / g2[1:])
    return out


def apply_chi0bar(c_half, eps, U, n_occ, miller, L, N):
    """chi0bar applied to potentials given by half-sphere coefficients c_half[n, n_half]; returns the same representation."""
    idx = ogs.fft_index(miller, N)
    half = np.nonzero(ogs.half_sphere_mask(miller))[0]
    sv = sqrt_coulomb(miller, L)
    full = ogs.expand_half_to_full(c_half * sv, miller)
    dV = ham.to_real_space(full, idx, N)
    assert np.max(np.abs(dV.imag)) < 1e-10 * max(1.0, np.max(np.abs(dV.real)))
    dn = ochi0.chi0_sum_over_states(eps, U, n_occ, np.ascontiguousarray(dV.real), [0.0], miller, L, N)[0]
    return ham.to_g_space(dn, idx)[:, half] * sv


def dense_chi0bar(eps, U, n_occ, miller, L, N):
    n = real_basis_size(miller)
    out = y_from_coeffs(apply_chi0bar(coeffs_from_y(np.eye(n), miller), eps, U, n_occ, miller, L, N))
    return out.T            # column j = image of basis vector j


def pdep_eigenpairs(eps, U, n_occ, miller, L, N, n_pdep):
    M = dense_chi0bar(eps, U, n_occ, miller, L, N)
    lam, Y = np.linalg.eigh(0.5 * (M + M.T))
    return lam[:n_pdep], Y[:, :n_pdep], M
