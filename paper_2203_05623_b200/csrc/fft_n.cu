// Per-grid-size instantiation of the FFT kernels.  Compiled once per supported N with
//   -DWEST_N1=.. -DWEST_N2=.. -DWEST_NN=.. -DWEST_NW=.. -DWEST_MINB=.. -DWEST_CU=..
//   (N = N1*N2; NW = warps per CTA of the plane kernel, MINB = its resident CTAs per SM; CU = stick units per CTA in K1/K3)
#include "fft_ops.h"

#ifndef WEST_N1
#error "compile with -DWEST_N1 -DWEST_N2 -DWEST_NN -DWEST_NW -DWEST_MINB -DWEST_CU"
#endif
#ifndef WEST_MINB
#define WEST_MINB 1
#endif
#ifndef WEST_ZNT
#define WEST_ZNT 256
#endif
#ifndef WEST_NW_H
#define WEST_NW_H WEST_NW
#define WEST_MINB_H WEST_MINB
#endif
#ifndef WEST_NW_H32         // shape of the FP32 H*psi plane kernel (WEST_MIXED): half the shared memory per CTA, so more CTAs fit
#define WEST_NW_H32 WEST_NW_H
#define WEST_MINB_H32 WEST_MINB_H
#endif
#ifndef WEST_GW_H
#define WEST_GW_H 1         // warps per line group of the H*psi plane kernel (2 = warp pairs)
#endif
#ifndef WEST_NB_H
#define WEST_NB_H 1         // independent items per thread and pass of the H*psi plane kernel (K2's NB)
#endif

namespace {
constexpr int N1 = WEST_N1, N2 = WEST_N2, NN = N1 * N2, NW = WEST_NW, LPW = K2Cfg<N1, N2>::LPW;
// stick units per CTA: GAMMA runs two transforms per unit, so FULL takes twice as many units for the same 256 threads
template <bool GAMMA> struct CUof { static constexpr int v = GAMMA ? WEST_CU : 2 * WEST_CU; };

template <typename KernelT>
cudaError_t set_smem(KernelT k, size_t bytes) {
    if (bytes <= 48 * 1024) return cudaSuccess;
    return cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

template <typename T, bool GAMMA>
cudaError_t k1_t(int n_slots, cudaStream_t st, const WestGeom& g, VecMap vm, const cx<double>* X, void* W) {
    constexpr int CU = CUof<GAMMA>::v;
    using K = K1<T, N1, N2, GAMMA, CU>;
    auto kern = k1_g2r_z<T, N1, N2, GAMMA, CU>;
    cudaError_t e = set_smem(kern, K::smem_bytes);
    if (e != cudaSuccess) return e;
    dim3 grid((g.n_units + CU - 1) / CU, n_slots);
    kern<<<grid, WEST_ZNT, K::smem_bytes, st>>>(g, vm, X, reinterpret_cast<cx<T>*>(W));
    return cudaGetLastError();
}
template <typename T, bool GAMMA>
cudaError_t k3_t(int n_slots, cudaStream_t st, const WestGeom& g, VecMap vm, const void* W, K3Epi ep, cx<double>* Y) {
    constexpr int CU = CUof<GAMMA>::v;
    using K = K3<T, N1, N2, GAMMA, CU>;
    auto kern = k3_r2g_z<T, N1, N2, GAMMA, CU>;
    cudaError_t e = set_smem(kern, K::smem_bytes);
    if (e != cudaSuccess) return e;
    dim3 grid((g.n_units + CU - 1) / CU, n_slots);
    kern<<<grid, WEST_ZNT, K::smem_bytes, st>>>(g, vm, reinterpret_cast<const cx<T>*>(W), ep, Y);
    return cudaGetLastError();
}
template <typename T, int MODE>
cudaError_t k2_t(int n_slots, cudaStream_t st, const WestGeom& g, const K2Any& a) {
    // the H*psi variant may use a different CTA shape from the one-way variants (store / dn / load)
    constexpr int NWm = MODE == K2_H ? (sizeof(T) == 4 ? WEST_NW_H32 : WEST_NW_H) : NW;
    constexpr int MBm = MODE == K2_H ? (sizeof(T) == 4 ? WEST_MINB_H32 : WEST_MINB_H) : WEST_MINB;
    constexpr int GWm = MODE == K2_H ? WEST_GW_H : 1;
    constexpr int NBm = MODE == K2_H ? WEST_NB_H : 1;
    constexpr int LPG = K2Cfg<N1, N2, GWm, NBm>::LPW;
    using K = K2<T, N1, N2, MODE, LPG>;
    auto kern = k2_planes<T, N1, N2, MODE, NWm, MBm, GWm, NBm>;
    const size_t bytes = sizeof(cx<T>) * (size_t)((g.nr + (NWm / GWm) * LPG) * K::PITCH + 2 * NN);
    cudaError_t e = set_smem(kern, bytes);
    if (e != cudaSuccess) return e;
    K2Args<T> t;
    t.W = reinterpret_cast<cx<T>*>(a.W);
    t.V = reinterpret_cast<const T*>(a.V);
    t.R = a.R; t.ucache = a.ucache; t.dV = a.dV; t.dn = a.dn; t.n_uslots = a.n_uslots; t.slot0 = a.slot0; t.fac = a.fac;
    dim3 grid(NN, n_slots);
    kern<<<grid, NWm * 32, bytes, st>>>(g, t);
    return cudaGetLastError();
}

cudaError_t k1_entry(int f32, int gamma, int n_slots, cudaStream_t st, const WestGeom& g, VecMap vm, const cx<double>* X, void* W) {
    if (f32) return gamma ? k1_t<float, true>(n_slots, st, g, vm, X, W) : k1_t<float, false>(n_slots, st, g, vm, X, W);
    return gamma ? k1_t<double, true>(n_slots, st, g, vm, X, W) : k1_t<double, false>(n_slots, st, g, vm, X, W);
}
cudaError_t k3_entry(int f32, int gamma, int n_slots, cudaStream_t st, const WestGeom& g, VecMap vm, const void* W, K3Epi e, cx<double>* Y) {
    if (f32) return gamma ? k3_t<float, true>(n_slots, st, g, vm, W, e, Y) : k3_t<float, false>(n_slots, st, g, vm, W, e, Y);
    return gamma ? k3_t<double, true>(n_slots, st, g, vm, W, e, Y) : k3_t<double, false>(n_slots, st, g, vm, W, e, Y);
}
cudaError_t k2_entry(int f32, int mode, int n_slots, cudaStream_t st, const WestGeom& g, const K2Any& a) {
    if (f32) {
        if (mode == K2_H) return k2_t<float, K2_H>(n_slots, st, g, a);
        return cudaErrorInvalidValue;          // only the H*psi path has an FP32 variant
    }
    switch (mode) {
        case K2_H: return k2_t<double, K2_H>(n_slots, st, g, a);
        case K2_TOR: return k2_t<double, K2_TOR>(n_slots, st, g, a);
        case K2_DN: return k2_t<double, K2_DN>(n_slots, st, g, a);
        case K2_FROMR: return k2_t<double, K2_FROMR>(n_slots, st, g, a);
    }
    return cudaErrorInvalidValue;
}
const FftOps ops = {NN, N1, N2, WEST_CU, LPW, K2Cfg<N1, N2, WEST_GW_H, WEST_NB_H>::LPW, k1_entry, k2_entry, k3_entry};
}  // namespace

#define WEST_CAT2(a, b) a##b
#define WEST_CAT(a, b) WEST_CAT2(a, b)
const FftOps* WEST_CAT(west_fft_ops_, WEST_NN)() { return &ops; }
