"""Pins for oracle/chi0.py (steps a1, a7-a10: Eq. 10-11).  CPU only.

Three independent routes to the same dn must agree: the sum over states (the definition), a dense LAPACK
solve of the Sternheimer equation, and the finite-field derivative of the ground-state density (PAPER.md:112:
"the linear variation of the electron density may be computed using either linear response or a finite-field
method").  A free-electron case is checked against a ten-line Lindhard sum written here from scratch.
"""
import numpy as np

import oracle_problem as op
from oracle import chi0 as ochi0
from oracle import gsphere as ogs
from oracle import hamiltonian as oham


def _relmax(a, b):
    return np.max(np.abs(a - b)) / np.max(np.abs(b))


def test_sum_over_states_equals_dense_sternheimer_and_alpha_independence():
    p = op.build("cfg1")
    dV = p.dV[:2]
    for om in (0.0, 0.05, 1.0):
        sos, dpsi_sos = ochi0.chi0_sum_over_states(p.eps, p.U, p.n_occ, dV, [om], p.miller, p.L, p.N, return_dpsi=True)
        for alpha in (0.5, 3.0):
            dn, dpsi = ochi0.sternheimer_dense(p.H, p.eps, p.U, p.n_occ, dV, om, alpha, p.miller, p.L, p.N, return_dpsi=True)
            assert _relmax(dn, sos[0]) < 1e-11
            assert _relmax(dpsi, dpsi_sos[0]) < 1e-10
            # solution lies in the conduction space: P_v dpsi = 0
            Uo = p.U[:, : p.n_occ]
            assert np.max(np.abs(dpsi @ np.conj(Uo))) < 1e-11


def test_finite_field_derivative_of_the_density():
    """dn = d n[V_loc + lambda dV] / d lambda at lambda = 0, n(r) = (2/Omega) sum_v |u_v(r)|^2."""
    p = op.build("cfg1")
    dV = p.dV[1]
    lam = 2e-4

    def density(vloc):
        H = oham.dense_h(p.miller, p.L, p.N, vloc, p.beta, p.dcoef)
        _, U = np.linalg.eigh(H)
        u = oham.to_real_space(U[:, : p.n_occ].T, p.fft_idx, p.N)
        return (2.0 / p.L ** 3) * np.sum(np.abs(u) ** 2, axis=0)

    ff = (density(p.vloc + lam * dV) - density(p.vloc - lam * dV)) / (2 * lam)
    dn = ochi0.chi0_sum_over_states(p.eps, p.U, p.n_occ, dV[None], [0.0], p.miller, p.L, p.N)[0, 0]
    assert _relmax(dn, ff) < 2e-6


def test_free_electron_lindhard_sum():
    """V = 0, D = 0, closed shells N_v in {1, 7, 19}: dV = 2 v cos(q.r) gives
    dn(r) = -(4 v / Omega) cos(q.r) sum_{k occ} sum_{+-} [k +- q empty] / (|k +- q|^2 - |k|^2) (2 pi / L)^-2 ..."""
    L, N, n2max = 10.0, 24, 25
    m = ogs.enumerate_sphere(n2max)
    idx = ogs.fft_index(m, N)
    zero = np.zeros((N, N, N))
    H = oham.dense_h(m, L, N, zero, None, None)
    eps, U = np.linalg.eigh(H)
    q = np.array([2, 1, 0])
    v = 0.05
    j = np.arange(N)
    phase = 2 * np.pi * (q[0] * j[:, None, None] + q[1] * j[None, :, None] + q[2] * j[None, None, :]) / N
    dV = 2 * v * np.cos(phase)
    for n_occ in (1, 7, 19):
        dn = ochi0.chi0_sum_over_states(eps, U, n_occ, dV[None], [0.0], m, L, N)[0, 0]
        # independent Lindhard loop over integer k-vectors
        order = np.argsort(np.sum(m.astype(int) ** 2, axis=1), kind="stable")
        occ = {tuple(int(x) for x in m[i]) for i in order[:n_occ]}
        s = 0.0
        for k in occ:
            for sign in (+1, -1):
                kq = tuple(int(k[a] + sign * q[a]) for a in range(3))
                if kq not in occ:
                    s += 1.0 / ((2 * np.pi / L) ** 2 * (sum(x * x for x in kq) - sum(x * x for x in k)))
        ref = -(4.0 * v / L ** 3) * s * np.cos(phase)
        assert _relmax(dn, ref) < 1e-11


def test_response_matrix_symmetry_negativity_monotonicity_and_charge():
    p = op.build("mini3")
    dV = p.dV
    oms = [0.0] + p.omegas
    dn = ochi0.chi0_sum_over_states(p.eps, p.U, p.n_occ, dV, oms, p.miller, p.L, p.N)
    prev = None
    for w in range(len(oms)):
        M = ochi0.response_matrix(dV, dn[w], p.L)
        assert np.max(np.abs(M - M.T)) < 1e-12 * np.max(np.abs(M))
        ev = np.linalg.eigvalsh(0.5 * (M + M.T))
        assert ev.max() < 0                                   # negative definite
        if prev is not None:
            assert np.all(np.diag(-M) < np.diag(-prev))        # -M decreases with omega
        prev = M
        assert np.max(np.abs(dn[w].sum(axis=(1, 2, 3)))) < 1e-10 * np.max(np.abs(dn[w])) * p.N ** 3


def test_constant_perturbation_gives_no_response_and_linearity():
    p = op.build("cfg1")
    const = np.full((1, p.N, p.N, p.N), 0.3)
    dn = ochi0.chi0_sum_over_states(p.eps, p.U, p.n_occ, const, [0.0, 0.7], p.miller, p.L, p.N)
    ref = ochi0.chi0_sum_over_states(p.eps, p.U, p.n_occ, p.dV[:2], [0.0, 0.7], p.miller, p.L, p.N)
    assert np.max(np.abs(dn)) < 1e-12 * np.max(np.abs(ref)) * 3
    comb = (2.0 * p.dV[0] - 0.5 * p.dV[1])[None]
    dnc = ochi0.chi0_sum_over_states(p.eps, p.U, p.n_occ, comb, [0.0, 0.7], p.miller, p.L, p.N)
    assert _relmax(dnc[:, 0], 2.0 * ref[:, 0] - 0.5 * ref[:, 1]) < 1e-12


def test_eq11_is_real_and_dn_from_dpsi_matches():
    p = op.build("cfg1")
    dn, dpsi = ochi0.chi0_sum_over_states(p.eps, p.U, p.n_occ, p.dV[:1], [0.3], p.miller, p.L, p.N, return_dpsi=True)
    Uo = p.U[:, : p.n_occ]
    u = oham.to_real_space(Uo.T, p.fft_idx, p.N)
    du = oham.to_real_space(dpsi[0, 0], p.fft_idx, p.N)
    eq11 = (2.0 / p.L ** 3) * np.sum(np.conj(u) * du + np.conj(du) * u, axis=0)    # sum over 2 spins of [psi* dpsi + c.c.]
    assert np.max(np.abs(eq11.imag)) < 1e-15 * np.max(np.abs(eq11.real))
    assert _relmax(eq11.real, dn[0, 0]) < 1e-14
    assert _relmax(ochi0.dn_from_dpsi(Uo, dpsi[0, 0], p.miller, p.L, p.N), dn[0, 0]) < 1e-14


def _spin_channels(p, n_occ_up=None, n_occ_dn=None):
    import synth
    B = synth.spin_splitting_field(p.cfg)
    ch = []
    for sgn, n_occ in ((+1, n_occ_up or p.n_occ), (-1, n_occ_dn or p.n_occ)):
        H = oham.dense_h(p.miller, p.L, p.N, p.vloc + sgn * B, p.beta, p.dcoef)
        eps, U = np.linalg.eigh(H)
        ch.append((eps, U, n_occ, H))
    return B, ch


def test_spin_polarised_finite_field_derivative_and_limits():
    """N_spin = 2: dn = d/d lambda of n(r) = (1/Omega) sum_sigma sum_v |u_v^sigma|^2 with h^sigma = T + V_loc +- B + lambda dV + V_NL,
    different occupations in the two channels; identical channels reduce to the unpolarised result; an empty channel adds nothing."""
    p = op.build("cfg1")
    dV = p.dV[1]
    B, ch = _spin_channels(p, n_occ_up=p.n_occ + 1, n_occ_dn=p.n_occ - 1)
    lam = 2e-4

    def density(lmb):
        n = 0.0
        for sgn, n_occ in ((+1, p.n_occ + 1), (-1, p.n_occ - 1)):
            H = oham.dense_h(p.miller, p.L, p.N, p.vloc + sgn * B + lmb * dV, p.beta, p.dcoef)
            _, U = np.linalg.eigh(H)
            u = oham.to_real_space(U[:, :n_occ].T, p.fft_idx, p.N)
            n = n + (1.0 / p.L ** 3) * np.sum(np.abs(u) ** 2, axis=0)
        return n

    ff = (density(lam) - density(-lam)) / (2 * lam)
    dn = ochi0.chi0_spin_polarised([c[:3] for c in ch], dV[None], [0.0], p.miller, p.L, p.N)[0, 0]
    assert _relmax(dn, ff) < 5e-6
    # per channel: dense Sternheimer solve with that channel's own H and projector
    for eps, U, n_occ, H in ch:
        a = ochi0.chi0_sum_over_states(eps, U, n_occ, dV[None], [0.3], p.miller, p.L, p.N, occupation=1.0)[0]
        b = ochi0.sternheimer_dense(H, eps, U, n_occ, dV[None], 0.3, 1.7, p.miller, p.L, p.N, occupation=1.0)
        assert _relmax(b, a) < 1e-11
    same = ochi0.chi0_spin_polarised([(p.eps, p.U, p.n_occ)] * 2, dV[None], [0.0, 0.5], p.miller, p.L, p.N)
    unpol = ochi0.chi0_sum_over_states(p.eps, p.U, p.n_occ, dV[None], [0.0, 0.5], p.miller, p.L, p.N)
    assert _relmax(same, unpol) < 1e-13
    one = ochi0.chi0_spin_polarised([ch[0][:3], (ch[1][0], ch[1][1], 0)], dV[None], [0.0], p.miller, p.L, p.N)
    up = ochi0.chi0_sum_over_states(*ch[0][:3], dV[None], [0.0], p.miller, p.L, p.N, occupation=1.0)
    assert _relmax(one, up) < 1e-14
