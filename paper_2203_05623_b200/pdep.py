"""PDEP shell around the hot path (widening row SURVEY 8(f)-3): the leading eigenpairs of the symmetrised
static response chi0bar = v^1/2 chi0(omega = 0) v^1/2 by block Davidson - trial potentials in, `west_chi0_apply` for every new
vector, Rayleigh-Ritz on a matrix of at most (4 N_PDEP)^2 (torch.linalg.eigh, i.e. cuSOLVER, as the paper does), residual expansion.

Potentials live on the wavefunction sphere as real functions without a G = 0 term, i.e. exactly the WEST_GAMMA vector storage, so the
transforms are `west_fft3d`; v(G) = 8 pi / |G|^2 in Rydberg units.  Outer algebra only (small dense matrices, orthogonalisation): torch.
"""
import math

import numpy as np
import torch

from .binding import WEST_GAMMA


class Chi0Bar:
    def __init__(self, west, n_occ, alpha_pv, tol_cg=1e-10, max_iter=500):
        assert west.mode == WEST_GAMMA, "PDEP shell is implemented for WEST_GAMMA (real orbitals)"
        self.w, self.n_occ, self.alpha, self.tol, self.max_iter = west, n_occ, alpha_pv, tol_cg, max_iter
        _, _, _, g2 = west.gsphere()
        sv = np.zeros(west.n_g)
        sv[1:] = np.sqrt(8.0 * np.pi / g2[1:])
        self.sv = torch.from_numpy(sv).cuda()
        sw = torch.full((2 * west.n_g,), math.sqrt(2.0), dtype=torch.float64, device="cuda")
        sw[0] = 0.0
        sw[1] = 0.0                                   # no G = 0 component in a PDEP potential
        self.sw = sw
        self.isw = torch.where(sw > 0, 1.0 / sw.clamp_min(1e-300), torch.zeros_like(sw))
        self.n_applied = 0

    def to_c(self, Y):
        return torch.view_as_complex((Y * self.isw).reshape(Y.shape[0], -1, 2).contiguous())

    def to_y(self, C):
        return torch.view_as_real(C).reshape(C.shape[0], -1) * self.sw

    def apply(self, Y):
        """chi0bar on real-coordinate rows Y[n, 2 n_g] (Euclidean inner product = real-space inner product of the potentials)."""
        C = self.to_c(Y) * self.sv
        dV = self.w.fft3d(+1, C.contiguous())
        dn, _, st = self.w.chi0_apply(dV, [0.0], tol=self.tol, max_iter=self.max_iter, alpha_pv=self.alpha, check_every=1)
        if st["rc"] != 0:
            raise RuntimeError("chi0_apply did not converge inside the PDEP shell: %s" % st)
        out = self.w.fft3d(-1, dn[0].contiguous()) * self.sv
        self.n_applied += Y.shape[0]
        return self.to_y(out)

    def random(self, n, seed):
        g = torch.Generator(device="cuda").manual_seed(seed)
        Y = torch.randn((n, 2 * self.w.n_g), dtype=torch.float64, device="cuda", generator=g)
        return Y * (self.sw > 0)


def _orthonormalise(Ynew, V):
    """Two-pass Gram-Schmidt of the rows of Ynew against the rows of V, then QR among themselves; drops numerically dependent rows."""
    for _ in range(2):
        if V is not None and V.shape[0]:
            Ynew = Ynew - (Ynew @ V.T) @ V
    Q, R = torch.linalg.qr(Ynew.T)
    keep = torch.abs(torch.diagonal(R)) > 1e-10 * torch.abs(torch.diagonal(R)).max()
    return Q.T[keep].contiguous()


def pdep(west, n_pdep, n_occ, alpha_pv, tol=1e-6, max_outer=60, max_basis=None, tol_cg=1e-10, seed=5, verbose=False):
    """Lowest n_pdep eigenpairs of chi0bar.  Returns eigenvalues [n_pdep] (numpy), eigenpotentials as half-sphere coefficients
    [n_pdep][n_g] (CUDA c128, c(0) = 0, orthonormal), residual norms, and the number of chi0*dV applications used."""
    op = Chi0Bar(west, n_occ, alpha_pv, tol_cg)
    max_basis = 4 * n_pdep if max_basis is None else max_basis
    V = _orthonormalise(op.random(n_pdep, seed), None)
    AV = op.apply(V)
    lam = res = None
    for outer in range(max_outer):
        H = V @ AV.T
        th, S = torch.linalg.eigh(0.5 * (H + H.T))
        U = S[:, :n_pdep].T @ V                      # Ritz vectors of the most negative eigenvalues
        AU = S[:, :n_pdep].T @ AV
        lam = th[:n_pdep]
        R = AU - lam[:, None] * U
        res = torch.linalg.norm(R, dim=1)
        if verbose:
            print("pdep outer %d  basis %d  max residual %.3e  lambda_0 %.6f" % (outer, V.shape[0], float(res.max()), float(lam[0])))
        if float(res.max()) < tol:
            break
        if V.shape[0] + n_pdep > max_basis:          # restart from the Ritz vectors (at most 4 N_PDEP)
            V, AV = U.contiguous(), AU.contiguous()
        T = _orthonormalise(R[res >= tol], V)
        if T.shape[0] == 0:
            break
        V = torch.cat([V, T])
        AV = torch.cat([AV, op.apply(T)])
    H = V @ AV.T
    th, S = torch.linalg.eigh(0.5 * (H + H.T))
    U = S[:, :n_pdep].T @ V
    return th[:n_pdep].cpu().numpy(), op.to_c(U), res.cpu().numpy(), op.n_applied
