"""Seeded synthetic inputs for the chi0*dV hot path (arXiv 2203.05623, Eq. 10-11).

This package holds ONLY input recipes: cell/config tables, smooth random fields,
atom positions, model potentials and Gaussian Kleinman-Bylander projectors.
It contains none of the method's arithmetic (no G-sphere enumeration, no
Hamiltonian application, no FFT of wavefunctions, no Sternheimer solve): callers
pass in the Miller indices they enumerated themselves.  It is the one module the
CPU oracle (``oracle/``) and the CUDA path (``paper_2203_05623_b200/``) share.
"""
from .configs import CONFIGS, get_config, seed_for  # noqa: F401
from .fields import (  # noqa: F401
    make_rng,
    smooth_field,
    random_positions,
    diamond_positions,
    epm_vloc,
    kb_projectors,
    perturbations,
    vloc_for,
    atoms_for,
    dense_grid,
    spin_splitting_field,
)
