"""Step a0: the plane-wave sphere and its index maps, by brute force.

"retains only the Fourier components that correspond to a chosen kinetic energy cutoff"
(FFTXlib).  Readings A1/A2 of SURVEY.md 8(c) / DESIGN.md: inclusion is the integer test
|n|^2 <= n2max; order is ascending lexicographic in the signed triple (n_x, n_y, n_z); the Gamma half
sphere is {0} U {first non-zero component positive}.
"""
import numpy as np


def enumerate_sphere(n2max):
    """All integer triples with n_x^2+n_y^2+n_z^2 <= n2max, lexicographic in signed (n_x, n_y, n_z). int32 [n_g][3]."""
    n_max = 0
    while (n_max + 1) ** 2 <= n2max:
        n_max += 1
    out = []
    for nx in range(-n_max, n_max + 1):
        for ny in range(-n_max, n_max + 1):
            for nz in range(-n_max, n_max + 1):
                if nx * nx + ny * ny + nz * nz <= n2max:
                    out.append((nx, ny, nz))
    return np.array(out, dtype=np.int32).reshape(-1, 3)


def fft_index(miller, N):
    """Linear index of G on the [ix][iy][iz] grid, ix = n_x mod N (z fastest). int32."""
    m = np.asarray(miller, dtype=np.int64)
    ix, iy, iz = m[:, 0] % N, m[:, 1] % N, m[:, 2] % N
    return ((ix * N + iy) * N + iz).astype(np.int32)


def half_sphere_mask(miller):
    """True for G = 0 and for triples whose first non-zero component is positive."""
    m = np.asarray(miller)
    first = np.where(m[:, 0] != 0, m[:, 0], np.where(m[:, 1] != 0, m[:, 1], m[:, 2]))
    return first >= 0


def index_of_minus(miller):
    """For each G in the list, the position of -G in the same list (dictionary lookup, not arithmetic)."""
    m = np.asarray(miller)
    where = {tuple(int(x) for x in t): i for i, t in enumerate(m)}
    return np.array([where[(-int(t[0]), -int(t[1]), -int(t[2]))] for t in m], dtype=np.int32)


def g2_of(miller, L):
    """|G|^2 in Ry, G = (2 pi / L) n."""
    m = np.asarray(miller, dtype=np.float64)
    return (2.0 * np.pi / L) ** 2 * np.sum(m * m, axis=1)


def expand_half_to_full(c_half, miller_full):
    """Half-sphere coefficients of a real function -> full sphere via c(-G) = conj c(G).

    c_half[..., n_half] is ordered like the half-sphere rows of miller_full (which, in lexicographic
    order, are its contiguous tail starting at G = 0)."""
    mask = half_sphere_mask(miller_full)
    minus = index_of_minus(miller_full)
    idx_half = np.nonzero(mask)[0]
    full = np.zeros(c_half.shape[:-1] + (len(miller_full),), dtype=np.complex128)
    full[..., idx_half] = c_half
    full[..., minus[idx_half]] = np.conj(c_half)
    # G = 0 is its own partner and must be real for a real function
    return full


def restrict_full_to_half(c_full, miller_full):
    return c_full[..., np.nonzero(half_sphere_mask(miller_full))[0]]
