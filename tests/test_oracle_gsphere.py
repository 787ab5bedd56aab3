"""Pins for oracle/gsphere.py (step a0).  CPU only."""
import math
import os

import numpy as np

from oracle import gsphere as ogs

HERE = os.path.dirname(os.path.abspath(__file__))


def _count_by_shells(n2max):
    """Independent count: sum over n_x, n_y of the number of integers n_z with n_z^2 <= rest (closed form per column)."""
    nm = math.isqrt(n2max)
    tot = 0
    for nx in range(-nm, nm + 1):
        for ny in range(-nm, nm + 1):
            rest = n2max - nx * nx - ny * ny
            if rest >= 0:
                tot += 2 * math.isqrt(rest) + 1
    return tot


def test_counts_of_the_five_configs():
    # values fixed by the integer definition |n|^2 <= n2max: 515 / 2301 / 18277 / 145405
    for n2max, full in ((25, 515), (66, 2301), (266, 18277)):
        m = ogs.enumerate_sphere(n2max)
        assert len(m) == full == _count_by_shells(n2max)
        assert int(np.sum(ogs.half_sphere_mask(m))) == (full + 1) // 2
    assert _count_by_shells(1064) == 145405


def test_continuum_limit():
    for n2max in (25, 266, 1064):
        assert abs(_count_by_shells(n2max) / (4.0 / 3.0 * math.pi * n2max ** 1.5) - 1.0) < 0.03


def test_order_is_lexicographic_and_half_is_tail():
    m = ogs.enumerate_sphere(66)
    keys = [tuple(int(x) for x in t) for t in m]
    assert keys == sorted(keys)
    assert len(set(keys)) == len(keys)
    assert np.all(np.sum(m.astype(np.int64) ** 2, axis=1) <= 66)
    mask = ogs.half_sphere_mask(m)
    n_half = int(mask.sum())
    assert np.array_equal(np.nonzero(mask)[0], np.arange(len(m) - n_half, len(m)))
    assert tuple(m[len(m) - n_half]) == (0, 0, 0)


def test_minus_map_is_the_reversal_involution():
    m = ogs.enumerate_sphere(25)
    minus = ogs.index_of_minus(m)
    assert np.array_equal(minus[minus], np.arange(len(m)))
    assert np.array_equal(m[minus], -m)
    # lexicographic order is reversed by negation
    assert np.array_equal(minus, np.arange(len(m))[::-1])


def test_fft_index_wraps_negative_frequencies():
    N = 24
    m = ogs.enumerate_sphere(25)
    idx = ogs.fft_index(m, N)
    assert len(np.unique(idx)) == len(idx)
    # decode and compare with numpy's own frequency table
    freq = np.rint(np.fft.fftfreq(N) * N).astype(int)
    ix, iy, iz = idx // (N * N), (idx // N) % N, idx % N
    assert np.array_equal(freq[ix], m[:, 0]) and np.array_equal(freq[iy], m[:, 1]) and np.array_equal(freq[iz], m[:, 2])


def test_expand_restrict_roundtrip_gives_real_function():
    N = 24
    m = ogs.enumerate_sphere(25)
    rng = np.random.default_rng(0)
    n_half = (len(m) + 1) // 2
    c = rng.standard_normal(n_half) + 1j * rng.standard_normal(n_half)
    c[0] = c[0].real
    full = ogs.expand_half_to_full(c, m)
    assert np.array_equal(ogs.restrict_full_to_half(full, m), c)
    grid = np.zeros(N ** 3, dtype=complex)
    grid[ogs.fft_index(m, N)] = full
    f = np.fft.ifftn(grid.reshape(N, N, N))
    assert np.max(np.abs(f.imag)) < 1e-17 + 1e-15 * np.max(np.abs(f.real))


def test_paper_table5_plane_wave_counts():
    """PAPER.md:319-326 (Table 5).  E_cut = 16 Ry, cubic n x n x n Si supercells, a = 10.2612 bohr (not stated in
    the paper): a full-sphere count reproduces 3 of the 4 printed N_PW exactly and all within 0.2 %."""
    a = 10.2612
    exact = 0
    with open(os.path.join(HERE, "golden", "table5_npw.txt")) as f:
        rows = [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]
    assert len(rows) == 4
    for n, _natom, _nel, ecut, npw in rows:
        L = int(n) * a
        n2max = int(math.floor(float(ecut) * L * L / (4.0 * math.pi ** 2)))
        cnt = _count_by_shells(n2max)
        if int(n) == 3:
            assert cnt == len(ogs.enumerate_sphere(n2max))
        assert abs(cnt - int(npw)) / int(npw) < 2e-3
        exact += cnt == int(npw)
        # the half-sphere (Gamma trick) count is off by a factor two: the paper's N_PW is the full sphere
        assert abs((cnt + 1) // 2 - int(npw)) / int(npw) > 0.4
    assert exact >= 3
