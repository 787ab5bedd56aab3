"""CPU-only check of the DEVICE code of the pruned FFT (no GPU needed): the kernel phases of fft_kernels.cuh are functions of
(tid, nthreads), so tests/host/step_fft.cu steps K1 -> K2 -> K3 thread by thread on the host; the result (T + V_loc) c must
match the oracle's matrix-free H and the sphere order must match the oracle's enumeration bit for bit."""
import os
import shutil
import subprocess

import numpy as np
import pytest

from oracle import gsphere as ogs
from oracle import hamiltonian as oham

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
NVCC = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"


@pytest.fixture(scope="module")
def stepper(tmp_path_factory):
    if not os.path.exists(NVCC):
        pytest.skip("nvcc not available")
    exe = str(tmp_path_factory.mktemp("step") / "step_fft")
    r = subprocess.run([NVCC, "-O1", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-x", "cu", "-o", exe,
                        os.path.join(ROOT, "tests", "host", "step_fft.cu")], capture_output=True, text=True)
    assert r.returncode == 0, r.stderr[-2000:]
    return exe


@pytest.mark.parametrize("N,n2max,gamma,L,nvec,f32,tol", [
    (24, 25, 0, 10.0, 2, 0, 1e-13), (24, 25, 1, 10.0, 3, 0, 1e-13), (36, 66, 1, 10.25, 2, 0, 1e-13),
    (48, 66, 0, 10.25, 1, 0, 1e-13), (24, 25, 1, 10.0, 3, 1, 1e-5)])
@pytest.mark.parametrize("nb", [1, 2])
def test_stepped_device_code_matches_oracle(stepper, tmp_path, N, n2max, gamma, L, nvec, f32, tol, nb):
    rng = np.random.default_rng(5)
    m = ogs.enumerate_sphere(n2max)
    V = rng.standard_normal((N, N, N))
    if gamma:
        half = np.nonzero(ogs.half_sphere_mask(m))[0]
        X = rng.standard_normal((nvec, len(half))) + 1j * rng.standard_normal((nvec, len(half)))
        X[:, 0] = X[:, 0].real
        cfull = ogs.expand_half_to_full(X, m)
    else:
        half = np.arange(len(m))
        X = rng.standard_normal((nvec, len(m))) + 1j * rng.standard_normal((nvec, len(m)))
        cfull = X
    fin, fout = str(tmp_path / "in.bin"), str(tmp_path / "out.bin")
    with open(fin, "wb") as f:
        f.write(np.ascontiguousarray(X).astype(np.complex128).tobytes())
        f.write(V.tobytes())
    r = subprocess.run([stepper, str(N), str(n2max), str(gamma), str(L), str(nvec), str(f32), fin, fout, str(nb)], capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    raw = open(fout, "rb").read()
    ng = X.shape[1]
    Y = np.frombuffer(raw[:nvec * ng * 16], dtype=np.complex128).reshape(nvec, ng)
    mil = np.frombuffer(raw[nvec * ng * 16:], dtype=np.int32).reshape(-1, 3)
    assert np.array_equal(mil, m[half])
    ref = oham.apply_h(cfull, m, L, N, V, None, None)[:, half]
    assert np.max(np.abs(Y - ref)) / np.max(np.abs(ref)) < tol
