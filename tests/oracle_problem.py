"""Test helper (not a test): assemble one workload for the ORACLE side from synth/ + oracle/.

Everything a parity test hands to the CUDA path as *input* comes out of here: the synthetic potentials and
projectors (synth/), and the occupied orbitals / eigenvalues (oracle eigensolver: they are inputs of Eq. 10,
PAPER.md:116).  Nothing here ever comes from the CUDA path.
"""
import functools

import numpy as np

import synth
from oracle import chi0 as ochi0
from oracle import gsphere as ogs
from oracle import hamiltonian as oham


class Problem:
    pass


@functools.lru_cache(maxsize=8)
def build(name, dense=True):
    cfg = synth.get_config(name)
    p = Problem()
    p.cfg = cfg
    p.L, p.N, p.n2max = cfg["L"], cfg["N"], cfg["n2max"]
    p.miller = ogs.enumerate_sphere(cfg["n2max"])            # full sphere, always
    p.n_full = len(p.miller)
    p.fft_idx = ogs.fft_index(p.miller, p.N)
    p.minus = ogs.index_of_minus(p.miller)
    p.half = np.nonzero(ogs.half_sphere_mask(p.miller))[0]
    p.g2 = ogs.g2_of(p.miller, p.L)
    p.atoms = synth.atoms_for(cfg)
    p.vloc = synth.vloc_for(cfg, p.atoms)
    p.beta, p.dcoef = synth.kb_projectors(p.miller, p.L, p.atoms, 0.8, cfg["projectors"])
    p.n_occ = cfg["n_occ"]
    p.gamma = cfg["mode"] == "gamma"
    if dense:
        p.H = oham.dense_h(p.miller, p.L, p.N, p.vloc, p.beta, p.dcoef)
        p.eps, p.U = oham.eigensystem(p.H, p.miller, real_orbitals=p.gamma)
        p.gap = float(p.eps[p.n_occ] - p.eps[p.n_occ - 1])
        p.alpha = ochi0.default_alpha(p.eps, p.n_occ)
    p.dV = synth.perturbations(cfg)
    p.omegas = list(cfg["omegas"])
    return p
