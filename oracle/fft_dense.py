"""Dense complex-to-complex 3D DFT on an n^3 cubic grid: the operation timed in Fig. 3 (one FP64 or FP32 C2C
FFT on a 128^3 or 256^3 grid, data resident on the device).  Test infrastructure, like the rest of oracle/.

Definition (unnormalised, sign = +1 or -1; the paper fixes neither, reading R17: both signs, no scaling, like the library call it times):

    X[k_x, k_y, k_z] = sum_{r_x, r_y, r_z} x[r_x, r_y, r_z] exp(sign 2 pi i (k_x r_x + k_y r_y + k_z r_z) / n)

`dft3` is that sum written out: the n x n matrix F[k, r] = exp(sign 2 pi i k r / n) contracted with each axis in turn (the triple sum
factorises exactly; no fast algorithm, no library FFT, complex128 throughout, exponent reduced mod n in integers so that the matrix
entries are exact to rounding).  `dft3_at` evaluates single outputs X[k] by the full triple sum, for sampled checks at sizes where the
matrix form is slow.  Pins (tests/test_oracle_fft_dense.py): pure-Python triple loop at n = 3 and 4, delta <-> plane wave closed
forms, Parseval, the shift theorem, inverse = conj-sign / n^3, and agreement with numpy.fft (a library routine for the same
definition) on random input at composite and prime n.
"""
import numpy as np


def dft_matrix(n, sign):
    """F[k, r] = exp(sign 2 pi i k r / n), the phase index k r reduced mod n in integer arithmetic."""
    if sign not in (1, -1):
        raise ValueError("sign must be +1 or -1")
    kr = np.outer(np.arange(n), np.arange(n)) % n
    ang = 2.0 * np.pi * kr / n
    return np.cos(ang) + 1j * sign * np.sin(ang)


def dft3(x, sign):
    """X = the definition above for x[n, n, n] (any leading batch axes allowed), complex128."""
    x = np.asarray(x, dtype=np.complex128)
    n = x.shape[-1]
    if x.shape[-3:] != (n, n, n):
        raise ValueError("cubic grids only")
    F = dft_matrix(n, sign)
    y = np.einsum("ka,...abc->...kbc", F, x)        # sum over r_x
    y = np.einsum("kb,...abc->...akc", F, y)        # sum over r_y
    y = np.einsum("kc,...abc->...abk", F, y)        # sum over r_z
    return y


def dft3_at(x, sign, ks):
    """X[k] for each k = (k_x, k_y, k_z) in ks, each by the full n^3-term sum."""
    x = np.asarray(x, dtype=np.complex128)
    n = x.shape[-1]
    r = np.arange(n)
    out = np.empty(len(ks), dtype=np.complex128)
    for i, (kx, ky, kz) in enumerate(ks):
        ex = np.exp(sign * 2j * np.pi * ((kx * r) % n) / n)
        ey = np.exp(sign * 2j * np.pi * ((ky * r) % n) / n)
        ez = np.exp(sign * 2j * np.pi * ((kz * r) % n) / n)
        out[i] = ex @ ((x @ ez) @ ey)               # sum_z first, then y, then x
    return out
