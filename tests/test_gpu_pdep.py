"""GPU parity of the PDEP Davidson shell against the dense chi0bar of oracle/pdep.py."""
import numpy as np
import pytest

import oracle_problem
from gpu_common import make_west
from oracle import pdep as opd

pytestmark = pytest.mark.gpu


def test_pdep_eigenpairs_match_the_dense_oracle():
    from paper_2203_05623_b200 import pdep as gp
    p = oracle_problem.build("tinyg")
    n_pdep = 6
    lam_ref, Y_ref, M = opd.pdep_eigenpairs(p.eps, p.U, p.n_occ, p.miller, p.L, p.N, n_pdep + 2)
    w, sel = make_west(p)
    lam, C, res, n_app = gp.pdep(w, n_pdep, p.n_occ, p.alpha, tol=1e-8, tol_cg=1e-12)
    assert np.max(res) < 1e-8
    assert np.max(np.abs(lam - lam_ref[:n_pdep])) < 1e-8 * abs(lam_ref[0])
    # eigenvectors: the computed potentials, in the oracle's real coordinates, span the oracle's leading invariant subspace
    Yg = opd.y_from_coeffs(C.cpu().numpy())                           # [n_pdep, dim]
    gap = lam_ref[n_pdep] - lam_ref[n_pdep - 1]
    assert gap > 1e-6 * abs(lam_ref[0])
    P = Yg @ Y_ref[:, :n_pdep]
    assert np.max(np.abs(P @ P.T - np.eye(n_pdep))) < 1e-6
    # far fewer chi0*dV applications than the dimension of the space (the point of PDEP)
    assert n_app < M.shape[0] // 2
    w.close()
