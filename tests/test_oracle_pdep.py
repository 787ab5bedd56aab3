"""Pins of oracle/pdep.py: chi0bar is symmetric and negative semi-definite, its quadratic form is the response-matrix
element of oracle.chi0 (a different code path), and v^1/2 has the closed form 8 pi / G^2."""
import numpy as np

import oracle_problem as op
from oracle import chi0 as ochi0
from oracle import gsphere as ogs
from oracle import hamiltonian as oham
from oracle import pdep as opd


def test_dense_chi0bar_is_symmetric_negative_and_consistent_with_the_response_matrix():
    p = op.build("tinyg")
    lam, Y, M = opd.pdep_eigenpairs(p.eps, p.U, p.n_occ, p.miller, p.L, p.N, 6)
    assert np.max(np.abs(M - M.T)) < 1e-10 * np.max(np.abs(M))
    assert lam[0] < 0 and np.max(np.linalg.eigvalsh(0.5 * (M + M.T))) < 1e-10
    # y^T M y = <dV, dn> / Omega with dV = v^1/2 phi_y, by oracle.chi0.response_matrix (grid sums instead of sphere sums)
    rng = np.random.default_rng(3)
    y = rng.standard_normal(M.shape[0])
    c = opd.coeffs_from_y(y[None], p.miller) * opd.sqrt_coulomb(p.miller, p.L)
    dV = oham.to_real_space(ogs.expand_half_to_full(c, p.miller), p.fft_idx, p.N).real
    dn = ochi0.chi0_sum_over_states(p.eps, p.U, p.n_occ, np.ascontiguousarray(dV), [0.0], p.miller, p.L, p.N)[0]
    quad = ochi0.response_matrix(dV, dn, p.L)[0, 0] / p.L ** 3
    assert abs(y @ M @ y - quad) < 1e-10 * abs(quad)


def test_sqrt_coulomb_closed_form():
    p = op.build("tinyg", dense=False)
    sv = opd.sqrt_coulomb(p.miller, p.L)
    half = p.miller[p.half]
    k = np.argmax((half == [0, 0, 1]).all(axis=1))
    assert abs(sv[k] ** 2 - 8 * np.pi / (2 * np.pi / p.L) ** 2) < 1e-12 and sv[0] == 0.0
