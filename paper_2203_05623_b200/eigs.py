"""Occupied orbitals for cells whose dense H cannot be diagonalised: Chebyshev-filtered subspace iteration on the GPU.

Set-up code (untimed, outside the hot path): the inputs psi_i, eps_i of Eq. 10 must be eigenvectors of the
same H the library applies, so they are produced THROUGH ``west_h_apply``.  torch supplies QR / small eigh only.
In WEST_GAMMA mode vectors are real functions stored on the half sphere; the iteration runs in the real coordinates
y = sqrt(w) * (re, im) in which the real-space inner product is Euclidean (w = 2, except G = 0: re 1, im 0).
"""
import math

import torch

from .binding import WEST_GAMMA


class _Space:
    def __init__(self, west):
        self.w = west
        self.gamma = west.mode == WEST_GAMMA
        if self.gamma:
            sw = torch.full((2 * west.n_g,), math.sqrt(2.0), dtype=torch.float64, device="cuda")
            sw[0] = 1.0
            sw[1] = 0.0
            self.sw = sw
            self.isw = torch.where(sw > 0, 1.0 / sw.clamp_min(1e-300), torch.zeros_like(sw))

    def to_x(self, Y):          # Y [n, dim] -> complex coefficients [n, n_g]
        if self.gamma:
            return torch.view_as_complex((Y * self.isw).reshape(Y.shape[0], -1, 2).contiguous())
        return Y.contiguous()

    def to_y(self, X):
        if self.gamma:
            return torch.view_as_real(X).reshape(X.shape[0], -1) * self.sw
        return X

    def H(self, Y):
        return self.to_y(self.w.h_apply(self.to_x(Y)))

    def random(self, n, seed):
        g = torch.Generator(device="cuda").manual_seed(seed)
        if self.gamma:
            Y = torch.randn((n, 2 * self.w.n_g), dtype=torch.float64, device="cuda", generator=g)
            Y[:, 1] = 0.0
            return Y
        re = torch.randn((n, self.w.n_g), dtype=torch.float64, device="cuda", generator=g)
        im = torch.randn((n, self.w.n_g), dtype=torch.float64, device="cuda", generator=g)
        return torch.complex(re, im)

    def gram(self, A, B):
        return A.conj() @ B.T if not self.gamma else A @ B.T


def _upper_bound(sp, steps=12, seed=11):
    """Safe upper bound of the spectrum from a short Lanczos run (largest Ritz value + residual norm)."""
    v = sp.random(1, seed)
    v = v / torch.linalg.norm(v)
    alphas, betas = [], []
    v_prev = torch.zeros_like(v)
    beta = 0.0
    for _ in range(steps):
        wv = sp.H(v) - beta * v_prev
        a = float(torch.real(torch.sum(v.conj() * wv)))
        wv = wv - a * v
        beta = float(torch.linalg.norm(wv))
        alphas.append(a)
        betas.append(beta)
        if beta < 1e-12:
            break
        v_prev, v = v, wv / beta
    k = len(alphas)
    T = torch.zeros((k, k), dtype=torch.float64)
    for i in range(k):
        T[i, i] = alphas[i]
        if i + 1 < k:
            T[i, i + 1] = T[i + 1, i] = betas[i]
    return float(torch.linalg.eigvalsh(T)[-1]) + betas[-1]


def lowest_states(west, n_states, n_guard=None, tol=1e-10, degree=16, max_outer=200, seed=7, verbose=False):
    """Lowest n_states eigenpairs of the H held by ``west`` (needs set_vloc / set_kb).  Returns eps [n], psi [n][n_g] (CUDA,
    c128, orthonormal over the full sphere), max residual norm."""
    sp = _Space(west)
    n_guard = max(8, n_states // 8) if n_guard is None else n_guard
    k = n_states + n_guard
    ub = _upper_bound(sp) * 1.01 + 0.1
    Y = sp.random(k, seed)
    Q, _ = torch.linalg.qr(Y.T)
    Y = Q.T.contiguous()
    HY = sp.H(Y)
    Hs = sp.gram(Y, HY)
    th, S = torch.linalg.eigh(0.5 * (Hs + Hs.conj().T))
    Y = (S.T.to(Y.dtype) @ Y) if sp.gamma else (S.conj().T @ Y)
    res = float("inf")
    for outer in range(max_outer):
        a0, a = float(th[0]), float(th[-1])
        a = max(a, a0 + 1e-3)
        e, cc = (ub - a) / 2.0, (ub + a) / 2.0
        sigma = e / (a0 - cc)
        sigma1 = sigma
        Y0 = Y
        Y1 = (sp.H(Y0) - cc * Y0) * (sigma1 / e)
        for _ in range(2, degree + 1):
            sigma2 = 1.0 / (2.0 / sigma1 - sigma)
            Y2 = (sp.H(Y1) - cc * Y1) * (2.0 * sigma2 / e) - (sigma * sigma2) * Y0
            Y0, Y1, sigma = Y1, Y2, sigma2
        Q, _ = torch.linalg.qr(Y1.T)
        Y = Q.T.contiguous()
        if sp.gamma:
            Y[:, 1] = 0.0
        HY = sp.H(Y)
        Hs = sp.gram(Y, HY)
        th, S = torch.linalg.eigh(0.5 * (Hs + Hs.conj().T))
        St = S.T.to(Y.dtype) if sp.gamma else S.conj().T
        Y = St @ Y
        HY = St @ HY
        R = HY[:n_states] - th[:n_states, None].to(Y.dtype) * Y[:n_states]
        res = float(torch.linalg.norm(R, dim=1).max())
        if verbose:
            print("chefsi outer %d  residual %.3e  eps[0]=%.6f eps[n-1]=%.6f" % (outer, res, float(th[0]), float(th[n_states - 1])))
        if res < tol:
            break
    psi = sp.to_x(Y[:n_states].contiguous()).contiguous()
    return th[:n_states + 1].cpu().numpy().copy(), psi, res
