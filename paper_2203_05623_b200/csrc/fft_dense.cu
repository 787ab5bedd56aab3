// Dense complex-to-complex 3D FFT on an n^3 cubic grid, n = 64, 128, 256, FP64 or FP32: the operation of Fig. 3.
//
// Three axis passes (z, y, x), each a batch of length-n 1D FFTs done as two register radix stages (n = N1 N2, codelets of
// dft_small.cuh) with ONE shared-memory exchange in between.  A CTA owns a tile of TC lines.  Global loads go straight into
// registers and global stores come straight from registers; along the strided axes (x, y) the TC lines of a tile are TC
// consecutive z, so every warp access is a set of full 128-byte runs, and along z the lanes of a line read/write runs of
// NL (or N1) consecutive elements.  Every pass reads its whole tile before it writes, and tiles are disjoint, so each pass may
// run in place.  Natural order in, natural order out: input j = N2 j1 + j2, output k = k1 + N1 k2.
#include <cuda_runtime.h>
#include "dft_small.cuh"
#include "fft_dense.h"

namespace {

template <int N> struct Split;
template <> struct Split<64>  { static constexpr int N1 = 8,  N2 = 8,  NL = 8;  };
template <> struct Split<128> { static constexpr int N1 = 8,  N2 = 16, NL = 8;  };
template <> struct Split<256> { static constexpr int N1 = 16, N2 = 16, NL = 16; };

template <typename T> __device__ __forceinline__ cx<T> tw_ld(const cx<double>* tw, int m, int sign) {
    const double2 w = __ldg(reinterpret_cast<const double2*>(tw) + m);
    return mk<T>((T)w.x, (T)(sign > 0 ? w.y : -w.y));
}

// One axis pass over the tiles tile0 + blockIdx.x of a batch of grids (the batch is folded into the tile index).
// AXIS 0 (z): the transformed axis is the contiguous one; a tile is TC consecutive lines (line = (b n + x) n + y).
// AXIS 1 (y) / 2 (x): the axis has stride n / n^2; a tile is TC consecutive z of one (b, x) / (b, y) column set.
template <typename T, int N, int TC, int AXIS, int SIGN, int MINB>
__global__ void __launch_bounds__(TC * Split<N>::NL, MINB)
dense_axis_pass(const cx<T>* __restrict__ in, cx<T>* __restrict__ out, const cx<double>* __restrict__ tw, long long tile0) {
    constexpr int N1 = Split<N>::N1, N2 = Split<N>::N2, NL = Split<N>::NL;
    constexpr int R1 = N2 / NL, R2 = N1 / NL;              // codelets per thread in stage 1 / stage 2
    constexpr bool ZAXIS = AXIS == 0;
    constexpr int P2 = ZAXIS ? N2 + 1 : N2;                // row pitch of the exchange tile (padded when lanes stride over k1)
    constexpr int LP = N1 * P2;                            // one line in the exchange tile (ZAXIS layout)
    constexpr long long ST = AXIS == 0 ? 1 : AXIS == 1 ? N : (long long)N * N;     // stride of the transformed axis
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* S = reinterpret_cast<cx<T>*>(smem_raw);

    const int tid = threadIdx.x;
    const int c = ZAXIS ? tid / NL : tid % TC;             // line of the tile
    const int lane = ZAXIS ? tid % NL : tid / TC;          // position inside the line's thread group
    const long long tile = tile0 + blockIdx.x;
    long long base;
    if (AXIS == 0) {
        base = (tile * TC + c) * N;
    } else if (AXIS == 1) {
        const long long gp = tile / (N / TC);              // b n + x
        base = gp * N * N + (tile % (N / TC)) * TC + c;
    } else {
        constexpr int TPG = N * (N / TC);                  // tiles per grid
        const long long b = tile / TPG;
        const int r = (int)(tile % TPG);
        base = b * N * N * N + (long long)(r / (N / TC)) * N + (r % (N / TC)) * TC + c;
    }
    in += base; out += base;
    // launched with programmatic stream serialisation: this CTA may become resident while the previous pass drains; wait here,
    // before the first global read, until that grid has completed and its stores are visible
    cudaGridDependencySynchronize();

    // stage 1: DFT-N1 over j1 for each j2 of this thread, twiddle w^(j2 k1), to the exchange tile
#pragma unroll
    for (int i = 0; i < R1; ++i) {
        const int j2 = lane + NL * i;
        cx<T> v[N1];
#pragma unroll
        for (int j1 = 0; j1 < N1; ++j1) v[j1] = in[(N2 * j1 + j2) * ST];
        Dft<T, N1, SIGN>::run(v);
#pragma unroll
        for (int k1 = 0; k1 < N1; ++k1) {
            const cx<T> r = k1 == 0 ? v[0] : cmul(v[k1], tw_ld<T>(tw, j2 * k1, SIGN));
            if (ZAXIS) S[c * LP + k1 * P2 + j2] = r;
            else       S[(k1 * N2 + j2) * TC + c] = r;
        }
    }
    __syncthreads();
    // stage 2: DFT-N2 over j2 for each k1 of this thread, output k = k1 + N1 k2
#pragma unroll
    for (int i = 0; i < R2; ++i) {
        const int k1 = lane + NL * i;
        cx<T> v[N2];
#pragma unroll
        for (int j2 = 0; j2 < N2; ++j2) v[j2] = ZAXIS ? S[c * LP + k1 * P2 + j2] : S[(k1 * N2 + j2) * TC + c];
        Dft<T, N2, SIGN>::run(v);
#pragma unroll
        for (int k2 = 0; k2 < N2; ++k2) out[(k1 + N1 * k2) * ST] = v[k2];
    }
}

template <typename T, int N, int TC, int AXIS, int SIGN, int MINB>
cudaError_t launch_pass(long long tile0, long long n_tiles, cudaStream_t stm, const cx<T>* in, cx<T>* out, const cx<double>* tw) {
    constexpr int N1 = Split<N>::N1, N2 = Split<N>::N2, NL = Split<N>::NL;
    constexpr size_t bytes = sizeof(cx<T>) * (size_t)TC * N1 * (AXIS == 0 ? N2 + 1 : N2);
    auto kern = dense_axis_pass<T, N, TC, AXIS, SIGN, MINB>;
    if (bytes > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
        if (e != cudaSuccess) return e;
    }
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)n_tiles); cfg.blockDim = dim3(TC * NL); cfg.dynamicSmemBytes = bytes; cfg.stream = stm;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, in, out, tw, tile0);
}

template <typename T, int N, int SIGN>
cudaError_t fft3_t(int n_batch, cudaStream_t stm, const void* in_, void* out_, const cx<double>* tw) {
    constexpr int TC = sizeof(T) == 8 ? 8 : 16;            // tile width: 128-byte runs along z for the strided passes
    constexpr int TCZ = 8;
    constexpr int MINB = N == 256 ? 3 : 6;
    const cx<T>* in = reinterpret_cast<const cx<T>*>(in_);
    cx<T>* out = reinterpret_cast<cx<T>*>(out_);
    const long long planes = (long long)n_batch * N;
    cudaError_t e;
    if ((e = launch_pass<T, N, TCZ, 0, SIGN, MINB>(0, planes * (N / TCZ), stm, in, out, tw)) != cudaSuccess) return e;
    if ((e = launch_pass<T, N, TC, 1, SIGN, MINB>(0, planes * (N / TC), stm, out, out, tw)) != cudaSuccess) return e;
    return launch_pass<T, N, TC, 2, SIGN, MINB>(0, planes * (N / TC), stm, out, out, tw);
}

template <typename T, int N>
cudaError_t fft3_s(int sign, int n_batch, cudaStream_t stm, const void* in, void* out, const cx<double>* tw) {
    return sign > 0 ? fft3_t<T, N, 1>(n_batch, stm, in, out, tw) : fft3_t<T, N, -1>(n_batch, stm, in, out, tw);
}
template <int N>
cudaError_t fft3_p(int f32, int sign, int n_batch, cudaStream_t stm, const void* in, void* out, const cx<double>* tw) {
    return f32 ? fft3_s<float, N>(sign, n_batch, stm, in, out, tw) : fft3_s<double, N>(sign, n_batch, stm, in, out, tw);
}

}  // namespace

bool west_dense_fft_supported(int n) { return n == 64 || n == 128 || n == 256; }

cudaError_t west_dense_fft3d(int n, int f32, int sign, int n_batch, cudaStream_t stm, const void* in, void* out, const void* tw) {
    const cx<double>* t = reinterpret_cast<const cx<double>*>(tw);
    switch (n) {
        case 64:  return fft3_p<64>(f32, sign, n_batch, stm, in, out, t);
        case 128: return fft3_p<128>(f32, sign, n_batch, stm, in, out, t);
        case 256: return fft3_p<256>(f32, sign, n_batch, stm, in, out, t);
    }
    return cudaErrorInvalidValue;
}
