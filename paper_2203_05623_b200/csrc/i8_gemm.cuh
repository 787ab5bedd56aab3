// FP64-accurate projector GEMMs on the INT8 tensor path of sm_100a (tcgen05.mma kind::i8, int32 accumulators in tensor memory).
//
// Why: the KB / P_v contractions (steps a6, a7) are 73 % of the cfg-5 step, and DMMA shares the FP64 pipe with
// DFMA (37 TFLOP/s) - there is nothing left on that pipe.  The int8 tensor rate of the chip is two orders of
// magnitude higher, and a product of two FP64 numbers can be formed from integer pieces WITHOUT rounding (Ozaki-type splitting):
//   every operand row a[0..K) (the contraction runs along the row) is scaled by a power of two 2^-e so that |a| 2^-e < 1 and cut into S
//   signed slices of 7 bits,  a = 2^e sum_i q_i 2^(-6-7i),  |q_i| <= 64  (error-free: scaling, rint and the remainders are exact in FP64;
//   what is dropped is below 2^(e-7S), i.e. 2^-56 of the row's largest element at S = 8 - finer than the FP64 mantissa of that element);
//   a slice pair contracts in int8 x int8 -> int32 EXACTLY (|q q'| <= 2^12: four pairs over a k range of <= 2^17 stay below 2^31);
//   pairs of equal weight 2^(-12-7(i+j)) share an accumulator; the pairs with i + j >= S (below 2^-7S relative) are dropped;
//   the S weight classes meet in one FP64 sum per output element, scaled by the two row scales.
// S (S + 1) / 2 int8 products replace one FP64 product: 36 at S = 8.
//
// Kernel: D[r][c] = sum_k A[r][k] B[c][k] for a 128 x 128 tile, operands as slice arrays [S][rows][Kp] int8 (K-major, 64-byte
// swizzle, staged by TMA through a 2-stage mbarrier ring).  Tensor memory holds four 128-column int32 accumulators (512 columns = all of
// it), i.e. S / 2 weight classes at a time, so an output tile is three consecutive PHASES with their own slice sets:
//   phase 0:  i, j <  S/2, i + j <= S/2 - 1          weight classes 0 .. S/2 - 1      A slices 0 .. S/2-1,  B slices 0 .. S/2-1
//   phase 1:  j <  S/2, S/2 - j <= i <= S - 1 - j    weight classes S/2 .. S - 1      A slices 1 .. S-1,    B slices 0 .. S/2-1
//   phase 2:  j >= S/2, i <= S - 1 - j               weight classes S/2 .. S - 1      A slices 0 .. S/2-1,  B slices S/2 .. S-1
// Measured alternatives of this staging (cfg-5 H*psi batch of 16 384 vectors, overlap / update product in ms; this version 153 / 189):
// 32-byte rows with a 5-stage ring 182 / 216; 64-byte rows, four sub-phases of <= 8 tiles, 3 stages 182 / 213; 128-byte rows, six sub-phases
// of <= 7 tiles, two drains per tile 161 / 196; 2-CTA clusters multicasting the A tiles, and CTA pairs with tcgen05.mma.cta_group::2 on
// 256 x 128 tiles: same time as this version.  The source-level ncu capture says why (profiles/r02_i8_gemm.md): the MMA issuer finds its
// stage ready at the first poll for every k-block, the producer waits on the `empty` barriers - the kernel is bound by MMA execution at the
// rate the tensor pipe sustains under the box's power cap, so staging changes nothing and only moving fewer bytes (tile order in
// launch_i8_gemm: K chunks of ~8 KB, vector tiles in groups; fewer slices) helps.
// Warp roles as in tc_gemm.cuh: EPI_WARPS epilogue warps (TMEM lane quarter = warp mod 4, column block = warp / 4), then the TMA producer
// warp and the MMA issuer warp (+ TMEM owner).  The epilogue warps keep the FP64 sums of a tile in registers across its three phases and write once:
//   ATOMIC  out[c * ldo + r] += value by atomicAdd (overlap block, split along K)       else  out[c * ldo + r] += value (update).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include "tc_gemm.cuh"

namespace wi8 {

using wtc::mbar_arrive;
using wtc::mbar_expect_tx;
using wtc::mbar_init;
using wtc::mbar_wait;
using wtc::smem_u32;
using wtc::tma_load_3d;
using wtc::tmem_ld32;
using wtc::umma_commit;

constexpr int BM = 128, BN = 128, BKB = 64;          // BKB int8 = 64 bytes = one swizzle row
#ifndef WEST_I8_EPI_WARPS
#define WEST_I8_EPI_WARPS 16       // 8 measured slower on the update product of small cells (1.90 against 1.75 ms at cfg-2 size), equal at cfg 5
#endif
constexpr int STAGES = 2, EPI_WARPS = WEST_I8_EPI_WARPS, NTHREADS = (EPI_WARPS + 2) * 32, EPI_COLS = BN / (EPI_WARPS / 4);
constexpr uint32_t TILE_BYTES = BM * BKB;            // 8 KB per slice tile
constexpr int MAX_K_PER_SPLIT = 1 << 16;             // int32 exactness: at most 4 pairs per accumulator and phase: 4 x 2^16 x 2^12 = 2^30 (a factor 2 to spare)

template <int S> struct Sched {
    static constexpr int H = S / 2;
    static_assert(S % 2 == 0 && S >= 2 && S <= 8, "slice count");
    // per phase: first A slice, A tile count, first B slice, B tile count
    __host__ __device__ static constexpr int a_lo(int ph) { return ph == 1 ? 1 : 0; }
    __host__ __device__ static constexpr int n_a(int ph) { return ph == 1 ? S - 1 : H; }
    __host__ __device__ static constexpr int b_lo(int ph) { return ph == 2 ? H : 0; }
    __host__ __device__ static constexpr int n_b(int ph) { return H; }
    static constexpr int MAX_TILES = S - 1 + H;
    static constexpr uint32_t STAGE_BYTES = MAX_TILES * TILE_BYTES;
    static constexpr size_t SMEM_BYTES = (size_t)STAGES * STAGE_BYTES + 1024 + 256;
};

// shared-memory matrix descriptor of a K-major tile with 64-byte swizzle: rows of 64 bytes, 8-row groups 512 bytes apart
__device__ __forceinline__ uint64_t umma_desc64(uint32_t saddr) {
    return (uint64_t)((saddr >> 4) & 0x3FFF) | (1ull << 16) | (32ull << 32) | (1ull << 46) | (4ull << 61);
}
// instruction descriptor: D = S32, A = B = signed int8, both K-major, M = 128, N = 128
constexpr uint32_t IDESC_I8 = (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(BN >> 3) << 17) | ((uint32_t)(BM >> 4) << 24);
__device__ __forceinline__ void umma_i8(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t accumulate) {
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(IDESC_I8), "r"(accumulate) : "memory");
}

struct Maps { CUtensorMap a, b; };                   // (k byte, slice, row) tensors, box {64, 1, 128}
// tile order: B tiles in groups of gb; inside a group the gb B tiles run fastest, then the A tiles; then the next group; K splits slowest.
// Concurrently running CTAs then cover ~148 / gb A tiles x gb B tiles, so both operands are shared in L2 (gb = 1: A tiles fastest).
struct TileGrid { int tiles_a, tiles_b, splits, gb; };

template <int S, bool ATOMIC>
__global__ void __launch_bounds__(NTHREADS, 1) i8_slice_gemm(const __grid_constant__ Maps maps, TileGrid tg, int rows_a, int rows_b, int n_kb, int kb_per_split,
                                                             const double* __restrict__ scale_a, const double* __restrict__ scale_b,
                                                             double* __restrict__ out, long long ldo) {
    using SC = Sched<S>;
    constexpr int H = SC::H;
    extern __shared__ unsigned char smem_raw[];
    unsigned char* tiles = reinterpret_cast<unsigned char*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint64_t* bars = reinterpret_cast<uint64_t*>(tiles + (size_t)STAGES * SC::STAGE_BYTES);
    uint64_t* full = bars;                    // [STAGES]  TMA -> MMA
    uint64_t* empty = bars + STAGES;          // [STAGES]  MMA -> TMA
    uint64_t* acc_full = bars + 2 * STAGES;   // MMA -> epilogue (one phase's accumulators complete)
    uint64_t* acc_empty = acc_full + 1;       // epilogue -> MMA (drained)
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(acc_empty + 1);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_tiles = tg.tiles_a * tg.tiles_b * tg.splits;

    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, 1); }
        mbar_init(acc_full, 1); mbar_init(acc_empty, EPI_WARPS);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == EPI_WARPS + 1) {              // TMEM owner: all 512 columns (four 128-column int32 accumulators)
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "n"(512) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = *tmem_slot;
    auto tile_of = [&](int t, int& r0, int& c0, int& kb0, int& nkb) {
        const int per_split = tg.tiles_a * tg.tiles_b;
        const int sp = t / per_split, u = t - sp * per_split;
        const int tbg = u / (tg.gb * tg.tiles_a), r = u - tbg * tg.gb * tg.tiles_a;
        const int gsize = min(tg.gb, tg.tiles_b - tbg * tg.gb);
        const int ta = r / gsize, tb = tbg * tg.gb + (r - ta * gsize);
        r0 = ta * BM; c0 = tb * BN; kb0 = sp * kb_per_split;
        nkb = min(kb_per_split, n_kb - kb0);
    };

    if (warp == EPI_WARPS) {
        // ===== TMA producer =====
        if (lane == 0) {
            int it = 0;
            for (int t = blockIdx.x; t < n_tiles; t += gridDim.x) {
                int r0, c0, kb0, nkb;
                tile_of(t, r0, c0, kb0, nkb);
                for (int ph = 0; ph < 3; ++ph) {
                    const int na = SC::n_a(ph), nb = SC::n_b(ph), alo = SC::a_lo(ph), blo = SC::b_lo(ph);
                    for (int i = 0; i < nkb; ++i, ++it) {
                        const int s = it % STAGES;
                        if (it >= STAGES) mbar_wait(empty + s, ((it / STAGES) - 1) & 1);
                        unsigned char* st = tiles + (size_t)s * SC::STAGE_BYTES;
                        mbar_expect_tx(full + s, (uint32_t)(na + nb) * TILE_BYTES);
                        const int k = (kb0 + i) * BKB;
                        for (int a = 0; a < na; ++a) tma_load_3d(st + (size_t)a * TILE_BYTES, &maps.a, full + s, k, alo + a, r0);
                        for (int b = 0; b < nb; ++b) tma_load_3d(st + (size_t)(na + b) * TILE_BYTES, &maps.b, full + s, k, blo + b, c0);
                    }
                }
            }
        }
    } else if (warp == EPI_WARPS + 1) {
        // ===== MMA issuer =====
        if (lane == 0) {
            int it = 0, g = 0;                                             // k-blocks consumed, phases started (all tiles)
            for (int t = blockIdx.x; t < n_tiles; t += gridDim.x) {
                int r0, c0, kb0, nkb;
                tile_of(t, r0, c0, kb0, nkb);
                for (int ph = 0; ph < 3; ++ph, ++g) {
                    const int na = SC::n_a(ph), alo = SC::a_lo(ph), blo = SC::b_lo(ph);
                    if (g >= 1) mbar_wait(acc_empty, (g - 1) & 1);         // the previous phase's accumulators have been drained
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    for (int i = 0; i < nkb; ++i, ++it) {
                        const int s = it % STAGES;
                        mbar_wait(full + s, (it / STAGES) & 1);
                        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                        const uint32_t sa = smem_u32(tiles + (size_t)s * SC::STAGE_BYTES);
                        uint32_t used = i > 0 ? 0xFu : 0u;                 // accumulators already written in this phase
#pragma unroll
                        for (int jj = 0; jj < H; ++jj) {
                            const int j = blo + jj;                        // B slice
                            // A slices paired with j in this phase
                            const int i_lo = ph == 0 ? 0 : (ph == 1 ? H - j : 0);
                            const int i_hi = ph == 0 ? H - 1 - j : S - 1 - j;
                            const uint64_t bd = umma_desc64(sa + (uint32_t)(na + jj) * TILE_BYTES);
                            for (int ii = i_lo; ii <= i_hi; ++ii) {
                                const int acc = ph == 0 ? ii + j : ii + j - H;
                                const uint64_t ad = umma_desc64(sa + (uint32_t)(ii - alo) * TILE_BYTES);
                                const uint32_t d = tmem + (uint32_t)(acc * BN);
#pragma unroll
                                for (int kk = 0; kk < BKB / 32; ++kk) {
                                    umma_i8(d, ad + (uint64_t)(kk * 2), bd + (uint64_t)(kk * 2), (used >> acc) & 1u);
                                    used |= 1u << acc;
                                }
                            }
                        }
                        umma_commit(empty + s);
                    }
                    umma_commit(acc_full);
                }
            }
        }
    } else {
        // ===== epilogue warps: TMEM lane quarter lq (row r = r0 + 32 lq + lane), columns [ch0, ch0 + EPI_COLS) =====
        const int lq = warp & 3, ch0 = (warp >> 2) * EPI_COLS;
        int g = 0;
        for (int t = blockIdx.x; t < n_tiles; t += gridDim.x) {
            int r0, c0, kb0, nkb;
            tile_of(t, r0, c0, kb0, nkb);
            double acc[EPI_COLS];
#pragma unroll
            for (int j = 0; j < EPI_COLS; ++j) acc[j] = 0.0;
            for (int ph = 0; ph < 3; ++ph, ++g) {
                mbar_wait(acc_full, g & 1);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
                for (int d = 0; d < H; ++d) {
                    // weight of accumulator d of this phase relative to 2^-12: 2^(-7 (d + (ph ? H : 0)))
                    const double w = __longlong_as_double((long long)(1023 - 7 * (d + (ph ? H : 0))) << 52);
#pragma unroll
                    for (int q = 0; q < EPI_COLS / 32; ++q) {
                        uint32_t v[32];
                        tmem_ld32(tmem + ((uint32_t)(lq * 32) << 16) + (uint32_t)(d * BN + ch0 + q * 32), v);
                        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                        for (int j = 0; j < 32; ++j) acc[q * 32 + j] += w * (double)(int)v[j];
                    }
                }
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                __syncwarp();
                if (lane == 0) mbar_arrive(acc_empty);
            }
            const int r = r0 + lq * 32 + lane;
            if (r < rows_a) {
                const double sr = scale_a[r] * (1.0 / 4096.0);             // 2^(e_a) 2^-12
#pragma unroll
                for (int q = 0; q < EPI_COLS / 16; ++q) {
                    double old[16];
                    if (!ATOMIC) {
#pragma unroll
                        for (int j = 0; j < 16; ++j) {
                            const int cc = c0 + ch0 + q * 16 + j;
                            old[j] = cc < rows_b ? __ldcg(out + (long long)cc * ldo + r) : 0.0;
                        }
                    }
#pragma unroll
                    for (int j = 0; j < 16; ++j) {
                        const int cc = c0 + ch0 + q * 16 + j;
                        if (cc < rows_b) {
                            const double val = acc[q * 16 + j] * sr * scale_b[cc];
                            if (ATOMIC) atomicAdd(out + (long long)cc * ldo + r, val);
                            else __stcg(out + (long long)cc * ldo + r, old[j] + val);
                        }
                    }
                }
            }
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == EPI_WARPS + 1) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(512) : "memory");
    }
}

// --------------------------------------------------------------------------------------------------------- operand preparation
// One value -> S slices (exact): t = v * inv (|t| < 1); q_0 = rint(64 t); then the remainder times 128, S - 1 more times.
template <int S>
__device__ __forceinline__ void slice_value(double v, double inv, signed char (&q)[S]) {
    double t = v * inv * 64.0;
#pragma unroll
    for (int i = 0; i < S; ++i) {
        const double r = rint(t);
        q[i] = (signed char)(int)r;
        t = (t - r) * 128.0;
    }
}
// scale of a row whose largest magnitude is m: the power of two 2^e with m 2^-e in [0.5, 1)  (1 for a zero row)
__device__ __forceinline__ double pow2_above(double m) {
    if (!(m > 0.0)) return 1.0;
    int e;
    frexp(m, &e);
    return ldexp(1.0, e);
}
// in [rows][ld_in] f64 -> out [S][rows_alloc][Kp] int8 slices of every row relative to the row's own power-of-two scale (written to
// scale[row]); columns K .. Kp-1 are zero.  One CTA per row, 256 threads; the row is read twice (max, then slices).
template <int S>
__global__ void __launch_bounds__(256) slice_rows(long long K, const double* __restrict__ in, long long ld_in, signed char* __restrict__ out, long long rows_alloc,
                                                  long long Kp, double* __restrict__ scale) {
    __shared__ double red[8];
    __shared__ double s_inv;
    const long long row = blockIdx.x;
    const double* src = in + row * ld_in;
    double m = 0.0;
    for (long long k = threadIdx.x; k < K; k += 256) m = fmax(m, fabs(src[k]));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        double mm = 0.0;
        for (int w = 0; w < 8; ++w) mm = fmax(mm, red[w]);
        const double p2 = pow2_above(mm);
        scale[row] = p2;
        s_inv = 1.0 / p2;
    }
    __syncthreads();
    const double inv = s_inv;
    // 8 consecutive k per thread: one 8-byte store per slice
    for (long long k0 = (long long)threadIdx.x * 8; k0 < Kp; k0 += 256 * 8) {
        signed char q[8][S];
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            const long long k = k0 + e;
            slice_value<S>(k < K ? src[k] : 0.0, inv, q[e]);
        }
#pragma unroll
        for (int i = 0; i < S; ++i) {
            unsigned long long pk = 0;
#pragma unroll
            for (int e = 0; e < 8; ++e) pk |= (unsigned long long)(unsigned char)q[e][i] << (8 * e);
            *reinterpret_cast<unsigned long long*>(out + ((long long)i * rows_alloc + row) * Kp + k0) = pk;
        }
    }
}
// column maxima of in [rows][ld_in]: colmax[k] = max_m |in[m][k]|   (set-up of the transposed operator slices)
__global__ void col_absmax(int rows, long long K, const double* __restrict__ in, long long ld_in, double* __restrict__ colscale) {
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= K) return;
    double m = 0.0;
    for (int r = 0; r < rows; ++r) m = fmax(m, fabs(in[(long long)r * ld_in + k]));
    colscale[k] = pow2_above(m);
}
// in [rows][ld_in] f64 -> transposed slices out [S][K][Mp] int8 (row of the output = k, contraction index m contiguous; columns
// rows .. Mp-1 zero), every output row k relative to colscale[k].  32 x 32 tiles through shared memory.
template <int S>
__global__ void slice_rows_transposed(int rows, long long K, const double* __restrict__ in, long long ld_in, const double* __restrict__ colscale,
                                      signed char* __restrict__ out, long long Mp) {
    __shared__ double t[32][33];
    const long long k0 = (long long)blockIdx.x * 32;
    const int m0 = blockIdx.y * 32;
    for (int y = threadIdx.y; y < 32; y += blockDim.y) {
        const int m = m0 + y; const long long k = k0 + threadIdx.x;
        t[y][threadIdx.x] = (m < rows && k < K) ? in[(long long)m * ld_in + k] : 0.0;
    }
    __syncthreads();
    for (int y = threadIdx.y; y < 32; y += blockDim.y) {
        const long long k = k0 + y; const int m = m0 + threadIdx.x;
        if (k < K && m < Mp) {
            signed char q[S];
            slice_value<S>(t[threadIdx.x][y], 1.0 / colscale[k], q);
#pragma unroll
            for (int i = 0; i < S; ++i) out[((long long)i * K + k) * Mp + m] = q[i];
        }
    }
}

}  // namespace wi8
