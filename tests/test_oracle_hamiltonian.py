"""Pins for oracle/hamiltonian.py (steps a2-a6).  CPU only."""
import numpy as np

import oracle_problem as op
from oracle import gsphere as ogs
from oracle import hamiltonian as oham


def test_delta_in_g_is_a_plane_wave_and_scaling():
    N, L = 24, 10.0
    m = ogs.enumerate_sphere(25)
    idx = ogs.fft_index(m, N)
    k = int(np.nonzero((m == np.array([2, -1, 3])).all(axis=1))[0][0])
    c = np.zeros(len(m), dtype=complex)
    c[k] = 1.0
    u = oham.to_real_space(c, idx, N)
    j = np.arange(N)
    pw = (np.exp(2j * np.pi * 2 * j / N)[:, None, None] * np.exp(-2j * np.pi * j / N)[None, :, None]
          * np.exp(2j * np.pi * 3 * j / N)[None, None, :])
    assert np.max(np.abs(u - pw)) < 1e-13           # e^{+iG.r}, unscaled
    back = oham.to_g_space(u, idx)
    assert np.max(np.abs(back - c)) < 1e-14         # 1/N^3 on the way back: round trip is the identity


def test_round_trip_and_parseval():
    N = 24
    m = ogs.enumerate_sphere(25)
    idx = ogs.fft_index(m, N)
    rng = np.random.default_rng(1)
    c = rng.standard_normal((3, len(m))) + 1j * rng.standard_normal((3, len(m)))
    u = oham.to_real_space(c, idx, N)
    assert np.max(np.abs(oham.to_g_space(u, idx) - c)) < 1e-13
    assert np.allclose(np.sum(np.abs(u) ** 2, axis=(1, 2, 3)) / N ** 3, np.sum(np.abs(c) ** 2, axis=1), rtol=1e-13)


def test_dense_is_hermitian_and_time_reversal_symmetric():
    p = op.build("cfg1")
    assert np.max(np.abs(p.H - p.H.conj().T)) < 1e-14
    Hm = p.H[np.ix_(p.minus, p.minus)]
    assert np.max(np.abs(Hm - p.H.conj())) < 1e-14  # H(-G,-G') = conj H(G,G'): H is real in r-space


def test_dense_equals_matrix_free():
    for name in ("cfg1", "mini2"):
        p = op.build(name)
        rng = np.random.default_rng(2)
        c = rng.standard_normal((4, p.n_full)) + 1j * rng.standard_normal((4, p.n_full))
        a = c @ p.H.T
        b = oham.apply_h(c, p.miller, p.L, p.N, p.vloc, p.beta, p.dcoef)
        assert np.max(np.abs(a - b)) < 1e-12 * np.max(np.abs(a))


def test_special_cases_kinetic_only_and_constant_potential():
    p = op.build("cfg1")
    rng = np.random.default_rng(3)
    c = rng.standard_normal(p.n_full) + 1j * rng.standard_normal(p.n_full)
    zero = np.zeros_like(p.vloc)
    assert np.array_equal(oham.apply_h(c, p.miller, p.L, p.N, zero, None, None), p.g2 * c)
    H0 = oham.dense_h(p.miller, p.L, p.N, zero, None, None)
    assert np.array_equal(H0, np.diag(p.g2).astype(complex))
    const = zero + 0.37
    y = oham.apply_h(c, p.miller, p.L, p.N, const, None, None)
    assert np.max(np.abs(y - (p.g2 + 0.37) * c)) < 1e-13
    # free-electron levels of the empty box: eigenvalues are (2 pi / L)^2 |n|^2 with the right multiplicities
    eps = np.linalg.eigvalsh(H0)
    ref = np.sort((2 * np.pi / p.L) ** 2 * np.sum(p.miller.astype(float) ** 2, axis=1))
    assert np.allclose(eps, ref, atol=1e-12)


def test_projector_term_matches_its_definition_elementwise():
    p = op.build("cfg1")
    zero = np.zeros_like(p.vloc)
    Hnl = oham.dense_h(p.miller, p.L, p.N, zero, p.beta, p.dcoef) - np.diag(p.g2)
    i, j = 17, 401
    want = sum(p.beta[k, i] * p.dcoef[k] * np.conj(p.beta[k, j]) for k in range(len(p.beta)))
    assert abs(Hnl[i, j] - want) < 1e-15


def test_eigenpairs_residual_orthonormality_and_real_orbitals():
    for name in ("cfg1", "mini2"):
        p = op.build(name)
        U = p.U[:, : p.n_occ + 4]
        R = p.H @ U - U * p.eps[None, : p.n_occ + 4]
        assert np.max(np.abs(R)) < 1e-11
        assert np.max(np.abs(U.conj().T @ U - np.eye(U.shape[1]))) < 1e-12
        assert p.gap > 0.02
        if p.gamma:
            u = oham.to_real_space(U.T, p.fft_idx, p.N)
            assert np.max(np.abs(u.imag)) < 1e-12 * np.max(np.abs(u.real))
            assert np.max(np.abs(U[p.minus] - np.conj(U))) < 1e-12
