// Blackwell tensor path of the WEST_MIXED contractions ("matrix multiplication or FFTs, which are carried out using FP32";
// north_star (3)): tcgen05.mma kind::tf32 with the accumulator in tensor memory, operands staged by TMA (cp.async.bulk.tensor, 128-byte
// swizzle) through an mbarrier ring.  FP64 has no tcgen05 kind, so the FP64 path stays on DMMA (gemm_f64.cuh); this file serves the
// KB / P_v products of H*psi when precision = WEST_MIXED.
//
// Precision: every FP64 operand x is pre-split into two TF32 numbers, x ~ hi + lo (hi = rna_tf32(float(x)), lo = rna_tf32(float(x) - hi)),
// and a product is hi*hi + hi*lo + lo*hi: relative error ~2^-21 per product, the class of the FP32 FFT next to it.  The tensor core adds
// into its FP32 accumulator without round-to-nearest, a bias that grows with the number of accumulations, so the contraction is cut into
// chunks of CHUNK_KB k-blocks (48 accumulations): each chunk lands in one of two TMEM accumulators, and the epilogue warps drain it with
// tcgen05.ld and add it to FP32 registers with round-to-nearest while the next chunk is being multiplied.
//
// One kernel, D[r][c] = sum_k A[r][k] B[c][k] for a 128 x 128 tile:
//   A, B : FP32 hi / lo arrays, k contiguous ("K-major"), addressed as (k, batch, row) tensors with strides that are multiples of 4 floats
//          (16-byte TMA strides); a plain [rows][ld] matrix is the case of one batch entry;
//          rows / k beyond the arrays read as zero (TMA out-of-bounds fill)
//   out  : FP64, out[c * ldo + r] (r contiguous: lanes of a warp = consecutive r, so stores and atomics coalesce)
//          ATOMIC: out += D by atomicAdd (split-K partial sums)      else: out += D (each element owned by one CTA)
// Warp roles: warps 0-7 epilogue (TMEM lane quarter = warp id mod 4, column half = warp id / 4: eight warps keep twice the global loads of
// the read-modify-write epilogue in flight and halve the drain time of a chunk), warp 8 TMA producer (one lane), warp 9 MMA issuer (one lane) +
// TMEM owner.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace wtc {

constexpr int BM = 128, BN = 128, BK = 32;          // BK fp32 = 128 bytes = one swizzle row
constexpr int STAGES = 3, CHUNK_KB = 4;             // k-blocks per TMEM chunk: 4 x (32 / 8) x 3 = 48 accumulations
constexpr int NTHREADS = 320, EPI_WARPS = 8, EPI_COLS = BN / 2;      // columns per epilogue warp
constexpr uint32_t TILE_BYTES = BM * BK * 4;        // 16 KB per operand part (BM == BN)
constexpr uint32_t STAGE_BYTES = 4 * TILE_BYTES;    // A hi, A lo, B hi, B lo
constexpr size_t SMEM_BYTES = (size_t)STAGES * STAGE_BYTES + 1024 /* alignment slack */ + 256 /* barriers */;
constexpr uint32_t TMEM_COLS = 2 * BN;              // two chunk accumulators

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// bounded wait: a mis-programmed pipeline traps instead of hanging the GPU
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    const uint32_t a = smem_u32(bar);
    for (uint32_t spin = 0; spin < (1u << 28); ++spin) {
        uint32_t ok;
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(a), "r"(parity) : "memory");
        if (ok) return;
    }
    __trap();
}
// tile of a (k, batch, row) tensor: box {BK, 1, 128}: 128 rows of one batch entry, BK reals along k; lands as a dense [128][BK] tile
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* tm, uint64_t* bar, int c0, int c1, int c2) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
                 ::"r"(smem_u32(dst)), "l"(tm), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
// shared-memory matrix descriptor of a K-major tile with 128-byte swizzle: rows of 128 bytes, 8-row groups 1024 bytes apart
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr) {
    return (uint64_t)((saddr >> 4) & 0x3FFF) | (1ull << 16) | (64ull << 32) | (1ull << 46) | (2ull << 61);
}
// instruction descriptor: D = F32, A = B = TF32, both K-major, M = 128, N = BN
constexpr uint32_t IDESC = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(BN >> 3) << 17) | ((uint32_t)(BM >> 4) << 24);
__device__ __forceinline__ void umma_tf32(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t accumulate) {
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(IDESC), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, "
                 "%20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]), "=r"(v[10]),
                   "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]),
                   "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]),
                   "=r"(v[31])
                 : "r"(taddr));
}

struct Maps { CUtensorMap a_hi, a_lo, b_hi, b_lo; };

// Persistent kernel: min(n_tiles, #SMs) CTAs walk the tile list (row tiles of A fastest, then row tiles of B, then K splits) so that the
// TMA ring never drains between tiles and the epilogue of one tile overlaps the multiplications of the next (the two TMEM chunk
// accumulators double as the hand-over buffers).  k-block, chunk and tile counters run on across tiles; barrier parities follow them.
// kb_per_split: k-blocks (of BK) per split; n_kb: total k-blocks.
struct TileGrid { int tiles_a, tiles_b, splits, n_batch; long long out_batch_stride; };      // batch entries: independent products (own slice of both operands and of out)
template <bool ATOMIC>
__global__ void __launch_bounds__(NTHREADS, 1) tf32x3_gemm(const __grid_constant__ Maps maps, TileGrid tg, int rows_a, int rows_b, int n_kb, int kb_per_split,
                                                            double* __restrict__ out, long long ldo) {
    extern __shared__ unsigned char smem_raw[];
    unsigned char* tiles = reinterpret_cast<unsigned char*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);      // swizzle-128B atoms need 1024-byte alignment
    uint64_t* bars = reinterpret_cast<uint64_t*>(tiles + (size_t)STAGES * STAGE_BYTES);
    uint64_t* full = bars;                    // [STAGES]  TMA -> MMA
    uint64_t* empty = bars + STAGES;          // [STAGES]  MMA -> TMA
    uint64_t* acc_full = bars + 2 * STAGES;   // [2]       MMA -> epilogue
    uint64_t* acc_empty = acc_full + 2;       // [2]       epilogue -> MMA
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(acc_empty + 2);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_tiles = tg.tiles_a * tg.tiles_b * tg.splits * tg.n_batch;

    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, 1); }
        for (int b = 0; b < 2; ++b) { mbar_init(acc_full + b, 1); mbar_init(acc_empty + b, EPI_WARPS); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == EPI_WARPS + 1) {              // TMEM owner: allocate 2 x BN columns, publish the base address
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "n"(TMEM_COLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = *tmem_slot;
    // tile t -> (row tile of A, row tile of B, split), k-block range of the split
    auto tile_of = [&](int t, int& r0, int& c0, int& kb0, int& nkb, int& bt) {
        const int ta = t % tg.tiles_a, rest = t / tg.tiles_a;
        const int tb = rest % tg.tiles_b, rest2 = rest / tg.tiles_b;
        const int sp = rest2 % tg.splits;
        bt = rest2 / tg.splits;
        r0 = ta * BM; c0 = tb * BN; kb0 = sp * kb_per_split;
        nkb = min(kb_per_split, n_kb - kb0);
        if (nkb < 0) nkb = 0;
    };

    if (warp == EPI_WARPS) {
        // ===== TMA producer =====
        if (lane == 0) {
            int it = 0;                                                    // k-blocks issued so far (all tiles)
            for (int t = blockIdx.x; t < n_tiles; t += gridDim.x) {
                int r0, c0, kb0, nkb, bt;
                tile_of(t, r0, c0, kb0, nkb, bt);
                for (int i = 0; i < nkb; ++i, ++it) {
                    const int s = it % STAGES;
                    if (it >= STAGES) mbar_wait(empty + s, ((it / STAGES) - 1) & 1);
                    unsigned char* st = tiles + (size_t)s * STAGE_BYTES;
                    mbar_expect_tx(full + s, STAGE_BYTES);
                    const int k = (kb0 + i) * BK;
                    tma_load_3d(st, &maps.a_hi, full + s, k, bt, r0);
                    tma_load_3d(st + TILE_BYTES, &maps.a_lo, full + s, k, bt, r0);
                    tma_load_3d(st + 2 * TILE_BYTES, &maps.b_hi, full + s, k, bt, c0);
                    tma_load_3d(st + 3 * TILE_BYTES, &maps.b_lo, full + s, k, bt, c0);
                }
            }
        }
    } else if (warp == EPI_WARPS + 1) {
        // ===== MMA issuer =====
        if (lane == 0) {
            int it = 0, g = 0;                                             // k-blocks consumed, chunks started (all tiles)
            for (int t = blockIdx.x; t < n_tiles; t += gridDim.x) {
                int r0, c0, kb0, nkb, bt;
                tile_of(t, r0, c0, kb0, nkb, bt);
                const int n_chunks = (nkb + CHUNK_KB - 1) / CHUNK_KB;
                for (int ch = 0; ch < n_chunks; ++ch, ++g) {
                    const int buf = g & 1;
                    if (g >= 2) mbar_wait(acc_empty + buf, ((g >> 1) - 1) & 1);
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    const uint32_t d = tmem + (uint32_t)(buf * BN);
                    const int i_end = min(nkb, (ch + 1) * CHUNK_KB);
                    for (int i = ch * CHUNK_KB; i < i_end; ++i, ++it) {
                        const int s = it % STAGES;
                        mbar_wait(full + s, (it / STAGES) & 1);
                        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                        const uint32_t sa = smem_u32(tiles + (size_t)s * STAGE_BYTES);
                        const uint64_t ah = umma_desc(sa), al = umma_desc(sa + TILE_BYTES), bh = umma_desc(sa + 2 * TILE_BYTES), bl = umma_desc(sa + 3 * TILE_BYTES);
#pragma unroll
                        for (int kk = 0; kk < BK / 8; ++kk) {
                            const uint64_t o = (uint64_t)(kk * 2);          // 8 fp32 = 32 bytes = 2 sixteen-byte units along k
                            const uint32_t first = (i == ch * CHUNK_KB && kk == 0) ? 0u : 1u;
                            umma_tf32(d, al + o, bh + o, first);           // small terms first
                            umma_tf32(d, ah + o, bl + o, 1u);
                            umma_tf32(d, ah + o, bh + o, 1u);
                        }
                        umma_commit(empty + s);                            // frees the stage when these MMAs have read it
                    }
                    umma_commit(acc_full + buf);                           // chunk accumulator complete
                }
            }
        }
    } else {
        // ===== epilogue warps 0-7: TMEM lane quarter lq = warp & 3 (row r = r0 + 32 lq + lane), columns [ch0, ch0 + EPI_COLS) =====
        const int lq = warp & 3, ch0 = (warp >> 2) * EPI_COLS;
        int g = 0;
        for (int t = blockIdx.x; t < n_tiles; t += gridDim.x) {
            int r0, c0, kb0, nkb, bt;
            tile_of(t, r0, c0, kb0, nkb, bt);
            const int n_chunks = (nkb + CHUNK_KB - 1) / CHUNK_KB;
            float acc[EPI_COLS];
#pragma unroll
            for (int j = 0; j < EPI_COLS; ++j) acc[j] = 0.f;
            for (int ch = 0; ch < n_chunks; ++ch, ++g) {
                const int buf = g & 1;
                mbar_wait(acc_full + buf, (g >> 1) & 1);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
                for (int q = 0; q < EPI_COLS / 32; ++q) {
                    uint32_t v[32];
                    tmem_ld32(tmem + ((uint32_t)(lq * 32) << 16) + (uint32_t)(buf * BN + ch0 + q * 32), v);
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                    for (int j = 0; j < 32; ++j) acc[q * 32 + j] += __uint_as_float(v[j]);
                }
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                __syncwarp();
                if (lane == 0) mbar_arrive(acc_empty + buf);
            }
            const int r = r0 + lq * 32 + lane;
            double* outb = out + (long long)bt * tg.out_batch_stride;
            if (r < rows_a && n_chunks > 0) {
                if (ATOMIC) {
#pragma unroll
                    for (int j = 0; j < EPI_COLS; ++j)
                        if (c0 + ch0 + j < rows_b) atomicAdd(outb + (long long)(c0 + ch0 + j) * ldo + r, (double)acc[j]);
                } else {
                    // read-modify-write in groups of 16 columns: all loads of a group are in flight before the first add (one memory
                    // latency per group instead of one per element)
#pragma unroll
                    for (int q = 0; q < EPI_COLS / 16; ++q) {
                        double old[16];
#pragma unroll
                        for (int j = 0; j < 16; ++j) {
                            const int cc = c0 + ch0 + q * 16 + j;
                            old[j] = cc < rows_b ? __ldcg(outb + (long long)cc * ldo + r) : 0.0;
                        }
#pragma unroll
                        for (int j = 0; j < 16; ++j) {
                            const int cc = c0 + ch0 + q * 16 + j;
                            if (cc < rows_b) __stcg(outb + (long long)cc * ldo + r, old[j] + (double)acc[q * 16 + j]);
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
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(TMEM_COLS) : "memory");
    }
}

// --------------------------------------------------------------------------------------------------------- operand preparation
__device__ __forceinline__ void split_tf32(double x, float& hi, float& lo) {
    const float f = (float)x;
    uint32_t h, l;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(h) : "f"(f));
    const float r = f - __uint_as_float(h);
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(l) : "f"(r));
    hi = __uint_as_float(h); lo = __uint_as_float(l);
}
// in [rows][ld_in] f64 -> hi, lo [rows][ld_out] f32 (columns k < K; the padding columns K .. ld_out-1 are written as zero)
__global__ void split_rows(long long rows, long long K, const double* __restrict__ in, long long ld_in, float* __restrict__ hi, float* __restrict__ lo,
                           long long ld_out) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= rows * ld_out) return;
    const long long r = i / ld_out, k = i - r * ld_out;
    float h = 0.f, l = 0.f;
    if (k < K) split_tf32(in[r * ld_in + k], h, l);
    hi[i] = h; lo[i] = l;
}
// in [rows][ld_in] f64 -> transposed hi, lo [K][ld_out] f32 (ld_out >= rows; padding zero).  32 x 32 tiles through shared memory.
__global__ void split_rows_transposed(int rows, long long K, const double* __restrict__ in, long long ld_in, float* __restrict__ hi,
                                      float* __restrict__ lo, long long ld_out) {
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
        if (k < K && m < ld_out) {
            float h, l;
            split_tf32(t[threadIdx.x][y], h, l);
            hi[k * ld_out + m] = h; lo[k * ld_out + m] = l;
        }
    }
}

}  // namespace wtc
