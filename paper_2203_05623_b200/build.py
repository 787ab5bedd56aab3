"""Builds paper_2203_05623_b200/libwest.so (the C-ABI library of include/west.h) with nvcc for sm_100a, in-tree.

    python -m paper_2203_05623_b200.build [--force]

No torch involvement: the library links only against the CUDA runtime.
"""
import concurrent.futures as cf
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
ROOT = os.path.dirname(HERE)
OBJ = os.path.join(ROOT, "build", "west_obj")
LIB = os.path.join(HERE, "libwest.so")

# (N1, N2, N, NW, MINB, CU, ZMINB, ZNT): N = N1*N2 grid size; LC = x lines per chunk in the plane kernel
# NW = warps per CTA of the plane kernel, MINB = resident CTAs per SM it is compiled for (register cap),
# CU = stick units per CTA of the z kernels (2 * CU * max(N1, N2) <= 256 threads)
# ZMINB = resident CTAs per SM the z-stick kernels are compiled for
# ZNT = threads per CTA of the z-stick kernels (2 * CU * max(N1, N2) <= ZNT)
# N = 144: four resident CTAs of 9 units instead of two of 10 (K1 3.67 -> 2.60 ms, K3 4.05 -> 3.32 ms per 1024 slots; sweep in profiles/r02_z_kernel_shapes.md)
FFT_SIZES = [(4, 6, 24, 4, 4, 20, 4, 256), (6, 6, 36, 4, 4, 20, 4, 256), (6, 8, 48, 6, 3, 16, 4, 256), (8, 9, 72, 12, 2, 14, 4, 256),
             (12, 12, 144, 12, 1, 9, 4, 224)]
K2H_SHAPES = {72: tuple(int(x) for x in os.environ.get("WEST_K2H_72", "6,3,2,1").split(",")),
              144: tuple(int(x) for x in os.environ.get("WEST_K2H_144", "12,1,1,1").split(","))}
# measured alternatives of the z-stick kernels' shape: WEST_Z_<N>="CU,ZMINB,ZNT" overrides the table entry of grid size N
for _i, _t in enumerate(FFT_SIZES):
    _v = os.environ.get("WEST_Z_%d" % _t[2])
    if _v:
        _cu, _zminb, _znt = (int(x) for x in _v.split(","))
        FFT_SIZES[_i] = _t[:5] + (_cu, _zminb, _znt)
# FP32 variant of the H*psi plane kernel (WEST_MIXED): (warps per CTA, resident CTAs per SM); absent = the FP64 shape
K2H32_SHAPES = {n: tuple(int(x) for x in os.environ["WEST_K2H32_%d" % n].split(",")) for n in (72, 144) if os.environ.get("WEST_K2H32_%d" % n)}
NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xcompiler", "-fPIC"]


def _nvcc():
    for p in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if p and (os.path.isabs(p) and os.path.exists(p) or not os.path.isabs(p)):
            return p
    raise RuntimeError("nvcc not found")


def _sources():
    out = [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC)) if f.endswith((".cu", ".cuh", ".h", ".hpp"))]
    out.append(os.path.join(ROOT, "include", "west.h"))
    out.append(os.path.abspath(__file__))
    return out


def up_to_date():
    if not os.path.exists(LIB):
        return False
    t = os.path.getmtime(LIB)
    return all(os.path.getmtime(s) <= t for s in _sources())


def _run(cmd):
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("command failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout, r.stderr))
    return r


def build(force=False, verbose=False):
    if not force and up_to_date():
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    nvcc = _nvcc()
    jobs = []
    for n1, n2, n, nw, minb, cu, zminb, znt in FFT_SIZES:
        o = os.path.join(OBJ, "fft_%d.o" % n)
        # shape of the H*psi plane kernel: (warps per CTA, resident CTAs per SM, warps per line group, items per thread and pass);
        # other N: the one-way variants' shape.  Measured alternatives: profiles/r02_k2_ilp.md
        k2h = K2H_SHAPES.get(n)
        extra = ["-DWEST_NW_H=%d" % k2h[0], "-DWEST_MINB_H=%d" % k2h[1], "-DWEST_GW_H=%d" % k2h[2], "-DWEST_NB_H=%d" % k2h[3]] if k2h else []
        k2h32 = K2H32_SHAPES.get(n)
        if k2h32:
            extra += ["-DWEST_NW_H32=%d" % k2h32[0], "-DWEST_MINB_H32=%d" % k2h32[1]]
        jobs.append((o, [nvcc] + NVCC_FLAGS + extra + ["-DWEST_N1=%d" % n1, "-DWEST_N2=%d" % n2, "-DWEST_NN=%d" % n, "-DWEST_NW=%d" % nw, "-DWEST_MINB=%d" % minb, "-DWEST_CU=%d" % cu, "-DWEST_ZMINB=%d" % zminb, "-DWEST_ZNT=%d" % znt,
                                               "-c", os.path.join(CSRC, "fft_n.cu"), "-o", o]))
    o = os.path.join(OBJ, "fft_dense.o")
    jobs.append((o, [nvcc] + NVCC_FLAGS + ["-c", os.path.join(CSRC, "fft_dense.cu"), "-o", o]))
    o = os.path.join(OBJ, "west.o")
    jobs.append((o, [nvcc] + NVCC_FLAGS + ["-c", os.path.join(CSRC, "west.cu"), "-o", o]))
    with cf.ThreadPoolExecutor(max_workers=min(8, len(jobs))) as ex:
        list(ex.map(lambda j: _run(j[1]), jobs))
    _run([nvcc, "-shared", "-o", LIB] + [j[0] for j in jobs] + ["-gencode", "arch=compute_100a,code=sm_100a"])
    if verbose:
        print("built", LIB)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
