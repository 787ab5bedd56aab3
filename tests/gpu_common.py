"""Test helper (not a test): hands an oracle-side Problem (tests/oracle_problem.py) to the CUDA library."""
import numpy as np


def relmax(a, b):
    """relative max-norm error max|a-b| / max|b|"""
    a = np.asarray(a)
    b = np.asarray(b)
    d = np.max(np.abs(b))
    return float(np.max(np.abs(a - b)) / (d if d > 0 else 1.0))


def make_west(p, with_states=True, with_kb=True):
    import torch
    import paper_2203_05623_b200 as wb

    mode = wb.WEST_GAMMA if p.gamma else wb.WEST_FULL
    w = wb.West(p.L, p.n2max, p.N, mode)
    sel = p.half if p.gamma else np.arange(p.n_full)
    assert w.n_g == len(sel)
    dev = torch.device("cuda:0")
    w.set_vloc(torch.from_numpy(np.ascontiguousarray(p.vloc)).to(dev))
    if with_kb and len(p.beta):
        w.set_kb(torch.from_numpy(np.ascontiguousarray(p.beta[:, sel])).to(dev), p.dcoef)
    if with_states:
        psi = np.ascontiguousarray(p.U[:, :p.n_occ].T[:, sel])
        w.set_states(torch.from_numpy(psi).to(dev), p.eps[:p.n_occ])
    return w, sel


def random_vectors(p, n_vec, seed):
    """Random coefficient vectors in the storage of the problem's mode, plus their full-sphere expansion (oracle side)."""
    from oracle import gsphere as ogs
    rng = np.random.Generator(np.random.PCG64(seed))
    if p.gamma:
        c = rng.standard_normal((n_vec, len(p.half))) + 1j * rng.standard_normal((n_vec, len(p.half)))
        c[:, 0] = c[:, 0].real
        return c, ogs.expand_half_to_full(c, p.miller)
    c = rng.standard_normal((n_vec, p.n_full)) + 1j * rng.standard_normal((n_vec, p.n_full))
    return c, c
