"""Seeded input recipes ("Synthetic inputs").

Stand-ins for the paper's Si supercells (Table 5) and SG15 ONCV
pseudopotentials, which are not available offline.  Nothing in this
file is part of the method being tested: it only manufactures arrays.

Units: Rydberg atomic units (hbar^2/2m = 1, kinetic energy |G|^2 Ry), lengths in bohr.
Grids are [ix][iy][iz], z fastest; G = (2 pi / L) n.
"""
import numpy as np
from scipy.interpolate import PchipInterpolator

from .configs import seed_for


def make_rng(cfg_id, k):
    return np.random.Generator(np.random.PCG64(seed_for(cfg_id, k)))


def _grid_n(N):
    """Signed integer frequencies of an N-point periodic grid, FFT order."""
    n = np.arange(N)
    return np.where(n < (N + 1) // 2, n, n - N)


def smooth_field(N, L, sigma, rms, rng):
    """White normal noise on the N^3 grid, Gaussian-filtered in G-space by exp(-sigma^2 G^2 / 2),
    mean removed, rescaled to the requested rms.  Real, shape (N, N, N)."""
    w = rng.standard_normal((N, N, N))
    n = _grid_n(N).astype(np.float64) * (2.0 * np.pi / L)
    g2 = n[:, None, None] ** 2 + n[None, :, None] ** 2 + n[None, None, :] ** 2
    f = np.fft.ifftn(np.fft.fftn(w) * np.exp(-0.5 * sigma * sigma * g2)).real
    f -= f.mean()
    f *= rms / np.sqrt(np.mean(f * f))
    return np.ascontiguousarray(f)


def random_positions(n_atoms, L, rng):
    return rng.uniform(0.0, L, size=(n_atoms, 3))


_DIAMOND_BASIS = np.array(
    [[0, 0, 0], [0, 2, 2], [2, 0, 2], [2, 2, 0], [1, 1, 1], [1, 3, 3], [3, 1, 3], [3, 3, 1]], dtype=np.float64
) / 4.0


def diamond_positions(ncell, a, disp_sigma, rng):
    """ncell^3 conventional 8-atom diamond cells of side a, plus N(0, disp_sigma) displacements."""
    pos = []
    for i in range(ncell):
        for j in range(ncell):
            for k in range(ncell):
                pos.append((_DIAMOND_BASIS + np.array([i, j, k], dtype=np.float64)) * a)
    pos = np.concatenate(pos, axis=0)
    pos = pos + rng.normal(0.0, disp_sigma, size=pos.shape)
    return pos


# (q^2 in (2 pi / a)^2, v in Ry).  The three middle points are the textbook empirical-pseudopotential
# form factors of silicon (V3, V8, V11); the end points are this repo's choice.
_EPM_Q2 = np.array([0.0, 3.0, 8.0, 11.0, 16.0, 24.0])
_EPM_V = np.array([-0.8, -0.21, 0.04, 0.08, 0.0, 0.0])
_EPM = PchipInterpolator(_EPM_Q2, _EPM_V, extrapolate=False)


def epm_vloc(N, L, positions, a):
    """V_loc(G) = v(|G|^2) * (1/N_at) sum_a exp(-i G.tau_a), G = 0 term dropped, on the N^3 grid; returns V(r) real."""
    n = _grid_n(N).astype(np.float64)
    q = n * (a / L)                                   # in units of 2 pi / a
    q2 = q[:, None, None] ** 2 + q[None, :, None] ** 2 + q[None, None, :] ** 2
    v = np.nan_to_num(_EPM(np.minimum(q2, _EPM_Q2[-1])), nan=0.0)
    v[q2 >= _EPM_Q2[-1]] = 0.0
    v[0, 0, 0] = 0.0
    g = n * (2.0 * np.pi / L)
    sf = np.zeros((N, N, N), dtype=np.complex128)
    for tau in positions:
        ex = np.exp(-1j * g * tau[0])
        ey = np.exp(-1j * g * tau[1])
        ez = np.exp(-1j * g * tau[2])
        sf += ex[:, None, None] * ey[None, :, None] * ez[None, None, :]
    sf /= len(positions)
    vg = v * sf
    vr = np.fft.ifftn(vg) * float(N) ** 3             # V(r) = sum_G V(G) exp(+i G.r)
    assert np.max(np.abs(vr.imag)) < 1e-10 * max(1.0, np.max(np.abs(vr.real)))
    return np.ascontiguousarray(vr.real)


def kb_projectors(miller, L, positions, sigma=0.8, projectors="sp", d_s=0.5, d_p=-0.25):
    """Gaussian Kleinman-Bylander projectors on a caller-supplied list of Miller triples.

    beta_s(G)   ~ exp(-sigma^2 G^2 / 2) exp(-i G.tau)
    beta_p,m(G) ~ -i G_m exp(-sigma^2 G^2 / 2) exp(-i G.tau),  m = x, y, z
    each normalised to sum_G |beta|^2 = 1 over the supplied set.  Returns (beta[n_proj][n_g] c128, d[n_proj]).
    Order: atom-major, then s, px, py, pz.
    """
    m = np.asarray(miller, dtype=np.float64)
    g = m * (2.0 * np.pi / L)
    g2 = np.sum(g * g, axis=1)
    env = np.exp(-0.5 * sigma * sigma * g2)
    rows, d = [], []
    for tau in positions:
        phase = np.exp(-1j * (g @ tau))
        b = env * phase
        rows.append(b / np.sqrt(np.sum(np.abs(b) ** 2)))
        d.append(d_s)
        if projectors == "sp":
            for ax in range(3):
                b = -1j * g[:, ax] * env * phase
                rows.append(b / np.sqrt(np.sum(np.abs(b) ** 2)))
                d.append(d_p)
    return np.ascontiguousarray(np.array(rows, dtype=np.complex128)), np.array(d, dtype=np.float64)


def atoms_for(cfg):
    rng = make_rng(cfg["cfg"], 1)
    if cfg["lattice"] == "random":
        return random_positions(cfg["n_atoms"], cfg["L"], rng)
    a = cfg["L"] / cfg["ncell"]
    return diamond_positions(cfg["ncell"], a, 0.10, rng)


def vloc_for(cfg, positions):
    if cfg["vloc"] == "random":
        return smooth_field(cfg["N"], cfg["L"], 1.0, 0.5, make_rng(cfg["cfg"], 0))
    return epm_vloc(cfg["N"], cfg["L"], positions, cfg["L"] / cfg["ncell"])


def perturbations(cfg, n_pert=None, first=0):
    """dV_i = smooth_field(sigma = 1 bohr, rms 0.1 Ry), one seeded stream per perturbation index."""
    n_pert = cfg["n_pert"] if n_pert is None else n_pert
    out = np.empty((n_pert, cfg["N"], cfg["N"], cfg["N"]), dtype=np.float64)
    for i in range(n_pert):
        out[i] = smooth_field(cfg["N"], cfg["L"], 1.0, 0.1, make_rng(cfg["cfg"], 2 + first + i))
    return out


def dense_grid(n, n_batch=1, seed=7000):
    """Complex standard-normal data on an n^3 grid, [n_batch][n][n][n] complex128: the input of the dense FFT benchmark
    (Fig. 3: the paper times transforms of wavefunction-like data whose values do not matter for the timing)."""
    rng = np.random.Generator(np.random.PCG64(seed + n))
    x = rng.standard_normal((n_batch, n, n, n)) + 1j * rng.standard_normal((n_batch, n, n, n))
    return np.ascontiguousarray(x)


def spin_splitting_field(cfg):
    """B(r) of the spin-polarised workload (N_spin = 2): V_up = V_loc + B, V_down = V_loc - B with B a smooth
    field (sigma 1.5 bohr, rms 0.03 Ry, seed stream 98); both channels keep n_occ orbitals, so both keep a gap."""
    return smooth_field(cfg["N"], cfg["L"], 1.5, 0.03, make_rng(cfg["cfg"], 98))
