// Internal launch interface between west.cu and the per-grid-size FFT translation units (fft_n.cu compiled once per N).
#pragma once
#include <cuda_runtime.h>
#include "fft_kernels.cuh"

struct K2Any {                 // K2Args<T> with untyped W / V
    void* W;
    const void* V;
    cx<double>* R;
    const cx<double>* ucache;
    const double* dV;
    double* dn;
    int n_uslots;
    int slot0;
    double fac;
};

struct FftOps {
    int N, N1, N2, CU, LC;
    int LC_H;      // lines per group of the H*psi plane kernel: fixes the V_loc layout (K2::vloc_index)
    // grid.y = slots in every launch; slot0 offsets are applied by the caller through pointer arithmetic / VecMap
    cudaError_t (*k1)(int f32, int gamma, int n_slots, cudaStream_t st, const WestGeom& g, VecMap vm, const cx<double>* X, void* W);
    cudaError_t (*k2)(int f32, int mode, int n_slots, cudaStream_t st, const WestGeom& g, const K2Any& a);
    cudaError_t (*k3)(int f32, int gamma, int n_slots, cudaStream_t st, const WestGeom& g, VecMap vm, const void* W, K3Epi e, cx<double>* Y);
};

const FftOps* west_fft_ops_24();
const FftOps* west_fft_ops_36();
const FftOps* west_fft_ops_48();
const FftOps* west_fft_ops_72();
const FftOps* west_fft_ops_144();
