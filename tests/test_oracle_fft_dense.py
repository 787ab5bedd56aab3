"""Pins of oracle/fft_dense.py (the dense C2C 3D DFT of Fig. 3) against the definition written as plain loops,
closed forms, DFT theorems and numpy's library FFT."""
import cmath
import itertools

import numpy as np
import pytest

import synth
from oracle import fft_dense as ofd


def _loops(x, sign):
    n = x.shape[0]
    X = np.zeros((n, n, n), dtype=complex)
    for kx, ky, kz in itertools.product(range(n), repeat=3):
        s = 0j
        for rx, ry, rz in itertools.product(range(n), repeat=3):
            s += x[rx, ry, rz] * cmath.exp(sign * 2j * cmath.pi * (kx * rx + ky * ry + kz * rz) / n)
        X[kx, ky, kz] = s
    return X


@pytest.mark.parametrize("n", [3, 4])
@pytest.mark.parametrize("sign", [1, -1])
def test_against_plain_python_triple_loop(n, sign):
    x = synth.dense_grid(n, 1, seed=11)[0]
    assert np.max(np.abs(ofd.dft3(x, sign) - _loops(x, sign))) < 1e-12
    ks = [(0, 0, 0), (1, 2, n - 1), (n - 1, 0, 1)]
    got = ofd.dft3_at(x, sign, ks)
    ref = _loops(x, sign)
    assert np.max(np.abs(got - np.array([ref[k] for k in ks]))) < 1e-12


@pytest.mark.parametrize("sign", [1, -1])
def test_delta_gives_plane_wave_and_plane_wave_gives_delta(sign):
    n = 12
    r0 = (5, 0, 7)                                  # asymmetric in the three axes: a transposed axis fails here
    x = np.zeros((n, n, n), dtype=complex); x[r0] = 1.0
    k = np.arange(n)
    pw = np.exp(sign * 2j * np.pi * (k[:, None, None] * r0[0] + k[None, :, None] * r0[1] + k[None, None, :] * r0[2]) / n)
    assert np.max(np.abs(ofd.dft3(x, sign) - pw)) < 1e-12
    q = (2, 9, 4)
    w = np.exp(-sign * 2j * np.pi * (k[:, None, None] * q[0] + k[None, :, None] * q[1] + k[None, None, :] * q[2]) / n)
    X = ofd.dft3(w, sign)                           # exp(-sign ..q.r) transforms to n^3 delta(k - q)
    expect = np.zeros((n, n, n), dtype=complex); expect[q] = n ** 3
    assert np.max(np.abs(X - expect)) < 1e-9


def test_parseval_shift_and_inverse():
    n = 10
    x = synth.dense_grid(n, 1, seed=3)[0]
    X = ofd.dft3(x, -1)
    assert abs(np.sum(np.abs(X) ** 2) - n ** 3 * np.sum(np.abs(x) ** 2)) < 1e-8 * n ** 3 * np.sum(np.abs(x) ** 2)
    back = ofd.dft3(X, +1) / n ** 3
    assert np.max(np.abs(back - x)) < 1e-12
    s = (1, 3, 6)                                   # shift theorem: x(r - s) -> X(k) exp(sign 2 pi i k.s / n)
    xs = np.roll(x, s, axis=(0, 1, 2))
    k = np.arange(n)
    ph = np.exp(-2j * np.pi * (k[:, None, None] * s[0] + k[None, :, None] * s[1] + k[None, None, :] * s[2]) / n)
    assert np.max(np.abs(ofd.dft3(xs, -1) - X * ph)) < 1e-10


@pytest.mark.parametrize("n", [7, 16, 24])
def test_against_numpy_fft_library(n):
    x = synth.dense_grid(n, 2, seed=5)
    assert np.max(np.abs(ofd.dft3(x, -1) - np.fft.fftn(x, axes=(1, 2, 3)))) < 1e-9
    assert np.max(np.abs(ofd.dft3(x, +1) - np.fft.ifftn(x, axes=(1, 2, 3)) * n ** 3)) < 1e-9
    ks = [(1, 2, 3), (n - 1, n - 2, 0)]
    assert np.max(np.abs(ofd.dft3_at(x[1], -1, ks) - np.array([np.fft.fftn(x[1])[k] for k in ks]))) < 1e-9
