"""Pins for oracle/iterative.py: the paper's PCG route against the plain definition.  CPU only."""
import numpy as np

import oracle_problem as op
from oracle import chi0 as ochi0
from oracle import hamiltonian as oham
from oracle import iterative as oit


def test_pcg_matches_sum_over_states_and_true_residual():
    p = op.build("cfg1")
    Uo = p.U[:, : p.n_occ]
    b = ochi0.rhs_vectors(Uo, p.dV[:1], p.fft_idx, p.N)[0]
    _, dpsi = ochi0.chi0_sum_over_states(p.eps, p.U, p.n_occ, p.dV[:1], [0.0], p.miller, p.L, p.N, return_dpsi=True)
    apply_H = lambda y: oham.apply_h(y, p.miller, p.L, p.N, p.vloc, p.beta, p.dcoef)
    Pv = Uo @ Uo.conj().T
    for v in (0, 3, p.n_occ - 1):
        x, it, rel = oit.pcg_sternheimer(apply_H, Uo, p.eps[v], v, b[v], p.g2, p.alpha, tol=1e-12)
        assert 5 < it < 200 and rel <= 1e-12
        A = p.H - p.eps[v] * np.eye(p.n_full) + p.alpha * Pv
        rhs = -(b[v] - Pv @ b[v])
        assert np.linalg.norm(A @ x - rhs) / np.linalg.norm(rhs) < 1e-10
        assert np.max(np.abs(x - dpsi[0, 0, v])) / np.max(np.abs(dpsi[0, 0, v])) < 1e-9


def test_cocg_matches_sum_over_states_at_imaginary_frequency():
    p = op.build("mini3")
    Uo = p.U[:, : p.n_occ]
    b = ochi0.rhs_vectors(Uo, p.dV[:1], p.fft_idx, p.N)[0]
    apply_H = lambda y: oham.apply_h(y, p.miller, p.L, p.N, p.vloc, p.beta, p.dcoef)
    for om in (0.05, 5.0):
        _, dpsi = ochi0.chi0_sum_over_states(p.eps, p.U, p.n_occ, p.dV[:1], [om], p.miller, p.L, p.N, return_dpsi=True)
        for v in (0, p.n_occ - 1):
            x, it, rel = oit.cocg_sternheimer(apply_H, Uo, p.eps[v], v, b[v], p.g2, p.minus, p.alpha, om, tol=1e-12)
            assert it < 300 and rel <= 1e-12
            assert np.max(np.abs(x - dpsi[0, 0, v])) / np.max(np.abs(dpsi[0, 0, v])) < 1e-9


def test_lowest_states_agree_with_dense_eigh():
    p = op.build("mini2")
    eps, U, res = oit.lowest_states(p.n_occ, p.miller, p.L, p.N, p.vloc, p.beta, p.dcoef, tol=1e-9)
    assert res < 1e-8
    assert np.max(np.abs(eps - p.eps[: p.n_occ])) < 1e-10
    # same occupied subspace: projector difference
    Uo = p.U[:, : p.n_occ]
    S = Uo.conj().T @ U
    assert abs(np.linalg.svd(S, compute_uv=False).min() - 1.0) < 1e-8
    assert np.max(np.abs(U[p.minus] - np.conj(U))) < 1e-12     # real orbitals
