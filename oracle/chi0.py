"""Steps a1, a7-a10 as their plain definition: chi0 * dV by the sum over states.

The method (Eq. 10: (h - eps_i) P_c dpsi_i^j = -P_c v_j psi_i, solved by preconditioned CG,
PAPER.md:121; Eq. 11: dn_j = sum_sigma sum_i [psi_i^* dpsi_i^j + c.c.]) reaches exactly, up to
rounding, the textbook sum over empty states that it was designed to avoid (Adler-Wiser).
So the oracle is that sum, written out:

    b_iv   = gather(fftn(dV_i * u_v) / N^3)                     (dV_i psi_v in the plane-wave basis)
    dpsi_iv = - sum_{c > N_v} psi_c <psi_c | b_iv> / (eps_c - eps_v - i omega)
    dn_i(r) = (4 / Omega) Re sum_v conj(u_v(r)) du_iv(r)         (spin-unpolarised: 2 spins x 2 for the c.c.)

``sternheimer_dense`` is the brute-force cross-check: build A = H - (eps_v + i omega) + alpha P_v densely and
call numpy.linalg.solve on the right-hand side -P_c b (reading A3: alpha P_v changes nothing in the solution).
"""
import numpy as np

from . import gsphere
from . import hamiltonian as ham


def rhs_vectors(U_occ, dV, fft_idx, N):
    """b[i, v, :] = (dV_i psi_v)(G) on the sphere.  U_occ[n_g, n_v] columns; dV[n_p, N, N, N] real."""
    u = ham.to_real_space(U_occ.T, fft_idx, N)                    # [n_v, N, N, N]
    return np.stack([ham.to_g_space(dV[i][None] * u, fft_idx) for i in range(len(dV))])


def chi0_sum_over_states(eps, U, n_occ, dV, omegas, miller, L, N, return_dpsi=False, occupation=2.0):
    """dn[w, i, N, N, N] (real, e/bohr^3) for every frequency omega_w >= 0 (imaginary axis) and perturbation i.
    occupation: electrons per orbital, 2 for a spin-unpolarised system, 1 for ONE channel of a spin-polarised one (the sum over
    sigma of Eq. 11); the prefactor is occupation x 2 (c.c.) / Omega."""
    idx = gsphere.fft_index(miller, N)
    vol = float(L) ** 3
    Uo, Uc = U[:, :n_occ], U[:, n_occ:]
    eo, ec = eps[:n_occ], eps[n_occ:]
    b = rhs_vectors(Uo, dV, idx, N)                               # [n_p, n_v, n_g]
    u_occ = ham.to_real_space(Uo.T, idx, N)                       # [n_v, N, N, N]
    M = np.einsum("gc,pvg->pvc", np.conj(Uc), b)                  # <psi_c | b_iv>
    dn = np.zeros((len(omegas), len(dV), N, N, N))
    dpsi_all = np.zeros((len(omegas), len(dV), n_occ, U.shape[0]), dtype=np.complex128) if return_dpsi else None
    for w, om in enumerate(omegas):
        denom = ec[None, :] - eo[:, None] - 1j * om               # [n_v, n_c]
        coef = -M / denom[None]
        dpsi = np.einsum("gc,pvc->pvg", Uc, coef)                 # [n_p, n_v, n_g]
        if return_dpsi:
            dpsi_all[w] = dpsi
        for i in range(len(dV)):
            du = ham.to_real_space(dpsi[i], idx, N)
            dn[w, i] = (2.0 * occupation / vol) * np.real(np.sum(np.conj(u_occ) * du, axis=0))
    return (dn, dpsi_all) if return_dpsi else dn


def default_alpha(eps, n_occ):
    """Reading A3: alpha = 2 (eps_Nv - eps_1), floored at 0.01 Ry."""
    return max(2.0 * float(eps[n_occ - 1] - eps[0]), 0.01)


def sternheimer_dense(H, eps, U, n_occ, dV, omega, alpha, miller, L, N, return_dpsi=False, occupation=2.0):
    """Brute force: for each (i, v) solve (H - eps_v - i omega + alpha P_v) x = -P_c b_iv with LAPACK."""
    idx = gsphere.fft_index(miller, N)
    vol = float(L) ** 3
    Uo = U[:, :n_occ]
    Pv = Uo @ Uo.conj().T
    b = rhs_vectors(Uo, dV, idx, N)
    u_occ = ham.to_real_space(Uo.T, idx, N)
    n_g = H.shape[0]
    dn = np.zeros((len(dV), N, N, N))
    dpsi = np.zeros((len(dV), n_occ, n_g), dtype=np.complex128)
    for v in range(n_occ):
        A = H - (eps[v] + 1j * omega) * np.eye(n_g) + alpha * Pv
        rhs = -(b[:, v, :] - b[:, v, :] @ Pv.T)                   # -(1 - P_v) b, rows are vectors
        x = np.linalg.solve(A, rhs.T).T                           # [n_p, n_g]
        dpsi[:, v, :] = x
    for i in range(len(dV)):
        du = ham.to_real_space(dpsi[i], idx, N)
        dn[i] = (2.0 * occupation / vol) * np.real(np.sum(np.conj(u_occ) * du, axis=0))
    return (dn, dpsi) if return_dpsi else dn


def chi0_spin_polarised(channels, dV, omegas, miller, L, N):
    """N_spin = 2 (Tables 3, 5, 7 list N_spin): each channel sigma has its own h^sigma, hence its own
    (eps, U, n_occ) = channels[sigma]; Eq. 10 is solved per channel with P_c^sigma, and Eq. 11 sums the channels, each orbital
    holding one electron:  dn = sum_sigma (2 / Omega) Re sum_v conj(u_v^sigma) du_v^sigma."""
    dn = 0.0
    for eps, U, n_occ in channels:
        dn = dn + chi0_sum_over_states(eps, U, n_occ, dV, omegas, miller, L, N, occupation=1.0)
    return dn


def dn_from_dpsi(U_occ, dpsi, miller, L, N):
    """Eq. 11 alone: dn(r) = (4/Omega) Re sum_v conj(u_v) du_v for dpsi[n_v, n_g]."""
    idx = gsphere.fft_index(miller, N)
    u = ham.to_real_space(U_occ.T, idx, N)
    du = ham.to_real_space(dpsi, idx, N)
    return (4.0 / float(L) ** 3) * np.real(np.sum(np.conj(u) * du, axis=0))


def response_matrix(dV, dn, L):
    """M_ij = <dV_j, dn_i> = (Omega / N^3) sum_r dV_j(r) dn_i(r), in Ry (reading A9)."""
    N = dV.shape[-1]
    return (float(L) ** 3 / float(N) ** 3) * np.einsum("jxyz,ixyz->ij", dV, dn)
