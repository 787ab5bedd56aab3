"""Workload table: the five BASELINE.json configs plus reduced ("mini") shapes.

Every entry is integers and literals only, so the G-sphere is defined without
floating point (SURVEY.md section 8(c) reading A2): ``n2max = floor(E_cut L^2 / 4 pi^2)``
is stored, not recomputed.  E_cut L^2/(4 pi^2) for the shapes used here:
cfg1 25.33, mini 66.53, cfg2-4 266.13, cfg5 1064.51 (all far from an integer).

mode: "full"  = complex orbitals on the full sphere (config 1, "FP64 complex")
      "gamma" = real orbitals, half-sphere storage (configs 2-5, "Gamma plane waves")
"""
import math

_OMEGA8 = [0.05 * 100.0 ** (k / 7.0) for k in range(8)]          # 0.05 .. 5 Ry, log-spaced
_OMEGA4 = [0.05 * 100.0 ** (k / 3.0) for k in range(4)]          # 0.05 .. 5 Ry, log-spaced

CONFIGS = {
    # BASELINE.json configs[0]
    "cfg1": dict(cfg=1, L=10.0, ecut=10.0, n2max=25, N=24, mode="full", lattice="random", n_atoms=2,
                 projectors="s", n_occ=8, n_pert=4, omegas=[0.0], vloc="random", precision="fp64"),
    # config-1 cell with real orbitals (Gamma storage): small enough for a dense chi0 matrix in the PDEP oracle
    "tinyg": dict(cfg=11, L=10.0, ecut=10.0, n2max=25, N=24, mode="gamma", lattice="random", n_atoms=2,
                  projectors="s", n_occ=8, n_pert=4, omegas=[0.0], vloc="random", precision="fp64"),
    # reduced Si-like cell: one diamond cell, everything else as configs 2-4
    "mini2": dict(cfg=12, L=10.25, ecut=25.0, n2max=66, N=36, mode="gamma", lattice="diamond", ncell=1,
                  n_atoms=8, projectors="sp", n_occ=16, n_pert=6, omegas=[0.0], vloc="epm", precision="fp64"),
    "mini3": dict(cfg=12, L=10.25, ecut=25.0, n2max=66, N=36, mode="gamma", lattice="diamond", ncell=1,
                  n_atoms=8, projectors="sp", n_occ=16, n_pert=4, omegas=[0.05, 0.6947, 5.0], vloc="epm",
                  precision="fp64"),
    "mini4": dict(cfg=12, L=10.25, ecut=25.0, n2max=66, N=36, mode="gamma", lattice="diamond", ncell=1,
                  n_atoms=8, projectors="sp", n_occ=16, n_pert=6, omegas=[0.0], vloc="epm", precision="mixed"),
    # same mini cell but on a 48^3 grid and with full-sphere complex storage (second FFT size, full mode)
    "mini48": dict(cfg=13, L=10.25, ecut=25.0, n2max=66, N=48, mode="full", lattice="diamond", ncell=1,
                   n_atoms=8, projectors="sp", n_occ=16, n_pert=3, omegas=[0.0], vloc="epm", precision="fp64"),
    # BASELINE.json configs[1..4]
    "cfg2": dict(cfg=2, L=20.5, ecut=25.0, n2max=266, N=72, mode="gamma", lattice="diamond", ncell=2,
                 n_atoms=64, projectors="sp", n_occ=128, n_pert=64, omegas=[0.0], vloc="epm", precision="fp64"),
    "cfg3": dict(cfg=2, L=20.5, ecut=25.0, n2max=266, N=72, mode="gamma", lattice="diamond", ncell=2,
                 n_atoms=64, projectors="sp", n_occ=128, n_pert=64, omegas=_OMEGA8, vloc="epm", precision="fp64"),
    "cfg4": dict(cfg=2, L=20.5, ecut=25.0, n2max=266, N=72, mode="gamma", lattice="diamond", ncell=2,
                 n_atoms=64, projectors="sp", n_occ=128, n_pert=128, omegas=[0.0], vloc="epm", precision="mixed"),
    "cfg5": dict(cfg=5, L=41.0, ecut=25.0, n2max=1064, N=144, mode="gamma", lattice="diamond", ncell=4,
                 n_atoms=512, projectors="sp", n_occ=1024, n_pert=256, pert_batch=16,
                 omegas=[0.0] + _OMEGA4, vloc="epm", precision="fp64"),
}


def get_config(name):
    c = dict(CONFIGS[name])
    c["name"] = name
    # consistency of the stored integer with the float recipe it came from
    assert c["n2max"] == int(math.floor(c["ecut"] * c["L"] ** 2 / (4.0 * math.pi ** 2))), name
    n_max = int(math.isqrt(c["n2max"]))
    assert c["N"] >= 4 * n_max + 1, "grid must hold products of two sphere-limited functions alias-free"
    c["n_max"] = n_max
    c["n_proj"] = c["n_atoms"] * (4 if c["projectors"] == "sp" else 1)
    return c


def seed_for(cfg_id, k):
    """Seeds 1000*cfg + k.  k: 0 V_loc noise, 1 atom positions, 2.. dV stream, 98 spin splitting field, 99 random test vectors."""
    return 1000 * int(cfg_id) + int(k)
