// FP64 tensor-core (DMMA, mma.sync m8n8k4) GEMMs for the dense contractions of the hot path: Kleinman-Bylander
// projector overlaps, P_v / P_c projections ("cuBLAS", 291 "FP64 tensor cores").
// There is no tcgen05 FP64 kind on sm_100a; DMMA.8x8x4 is the FP64 tensor instruction this chip has.
//
//   gemm_tn     C[m][n] (+)= sum_k A[m][k] B[n][k]      both operands K-contiguous; K is the long axis (2 n_g reals),
//                                                        split over blockIdx.z, partial sums reduced with FP64 atomics
//   gemm_update Y[n][k] += sum_m C[m][n] A[m][k]        rank-m update of the vector block
// Warp tile 64 x 32 (64 accumulators / thread), k step 16 through a cp.async ring.  Shared-memory rows are padded by 4
// doubles so every fragment load is bank-conflict free.  Yardstick on the same box: cuBLAS DGEMM 35-36 TFLOP/s on these shapes.
// Both kernels are templates on TF32: false = the FP64 DMMA path above, true = the 3xTF32 path of WEST_MIXED (see split_tf32 below).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace wgemm {

// CTA tile BM x BN with BM = 128 and BN = 32 * WN (WN = warps along n).  The shipped configuration is WN = 2: 128 x 64
// tiles, 4 warps (2 x 2, warp tile 64 x 32), 2 stages, THREE CTAs per SM so that one CTA's barrier / prologue / epilogue
// bubbles are covered by the others' DMMA streams (measured: 1 CTA x 8 warps 28.3 / 23.9, 2 x 4 warps 30.7 / 26.9, 3 x 4 warps 33.1 / 31.9 TFLOP/s for tn / update).
constexpr int BM = 128, BK = 16;
constexpr int WN = 2, BN = 32 * WN, STAGES = 2, NTHREADS = 2 * WN * 32, MINB = 3;
constexpr int PITCH_TN = BK + 4;                  // doubles
constexpr int PITCH_UPC = BM + 4;                 // doubles, C^T panel (n contiguous)
constexpr int PITCH_UPA = BN + 4;                 // doubles, A panel (k contiguous)
constexpr size_t SMEM_TN = (size_t)STAGES * (BM + BN) * PITCH_TN * sizeof(double);
constexpr size_t SMEM_UP = (size_t)STAGES * BK * (PITCH_UPC + PITCH_UPA) * sizeof(double);

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem, bool pred) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    int bytes = pred ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem), "r"(bytes));
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N> __device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// WEST_MIXED variants (template parameter TF32 = true; "matrix multiplication or FFTs ... carried out using FP32"): the same
// FP64 operands and the same cp.async staging, but the products run on the TF32 tensor path as 3xTF32 - every operand is rounded to
// FP32 and split into hi + lo TF32 parts, lo*hi + hi*lo + hi*hi accumulate in FP32 (error ~2^-22 per product, FP32 class) - with
// mma.sync.m16n8k8; warp tile 64 x 32 = 4 x 4 MMA tiles.  Partial sums leave the kernel in FP64 (atomics / the FP64 vector block).
__device__ __forceinline__ void split_tf32(double x, uint32_t& hi, uint32_t& lo) {
    const float f = (float)x;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(hi) : "f"(f));
    const float r = f - __uint_as_float(hi);
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(lo) : "f"(r));
}
__device__ __forceinline__ void mma_tf32(float (&c)[4], const uint32_t (&a)[4], const uint32_t (&b)[2]) {
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};\n"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]));
}
// one k = 8 step of a 64 x 32 warp tile: A-operand element (row, k) at pa[row * sa_row + k * sa_k], B-operand element (k, col) at
// pb[col * sb_col + k * sb_k]; lane = 4 g + t holds rows g, g + 8 and k = t, t + 4 (A), k = t, t + 4 and col g (B)
__device__ __forceinline__ void tf32x3_step(float (&acc)[4][4][4], const double* pa, int sa_row, int sa_k, const double* pb, int sb_col,
                                            int sb_k, int g, int t) {
    uint32_t ah[4][4], al[4][4], bh[4][2], bl[4][2];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const double* q = pa + (i * 16 + g) * sa_row + t * sa_k;
        split_tf32(q[0], ah[i][0], al[i][0]);
        split_tf32(q[8 * sa_row], ah[i][1], al[i][1]);
        split_tf32(q[4 * sa_k], ah[i][2], al[i][2]);
        split_tf32(q[8 * sa_row + 4 * sa_k], ah[i][3], al[i][3]);
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const double* q = pb + (j * 8 + g) * sb_col + t * sb_k;
        split_tf32(q[0], bh[j][0], bl[j][0]);
        split_tf32(q[4 * sb_k], bh[j][1], bl[j][1]);
    }
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            // the tensor core adds into its accumulator with truncation, a bias that grows with the number of accumulations (measured:
            // 2e-5 relative after ~750); so the three products of a k = 8 step meet in a zeroed temporary and join the running sum
            // through one round-to-nearest FADD per element (random-walk error, ~3e-6 at K = 18 278)
            float tmp[4] = {0.f, 0.f, 0.f, 0.f};
            mma_tf32(tmp, al[i], bh[j]);
            mma_tf32(tmp, ah[i], bl[j]);
            mma_tf32(tmp, ah[i], bh[j]);
#pragma unroll
            for (int q = 0; q < 4; ++q) acc[i][j][q] += tmp[q];
        }
}

// ---------------------------------------------------------------------------------------------------------------------
// C[m][n] += sum_{k in this split} A[m][k] B[n][k].   lda, ldb even (16-byte aligned rows), A and B 16-byte aligned.
template <bool TF32>
__global__ void __launch_bounds__(NTHREADS, MINB) gemm_tn_kernel(int M, int Nn, long long K, const double* __restrict__ A, long long lda,
                                                           const double* __restrict__ B, long long ldb, double* __restrict__ C,
                                                           long long ldc, long long k_per_split, int use_atomic, int splits,
                                                           long long sA, long long sB, long long sC) {
    extern __shared__ __align__(16) double smem[];
    double* As = smem;                                   // [STAGES][BM][PITCH_TN]
    double* Bs = smem + (size_t)STAGES * BM * PITCH_TN;  // [STAGES][BN][PITCH_TN]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = warp / WN, wn = warp % WN;            // 2 x WN warps
    // row tiles of A (m) are the FASTEST grid axis: the CTAs that share one (vector tile, K split) panel of B run together, so B streams
    // from HBM once and the other row tiles hit L2 (with the vector tiles fastest every row tile re-streamed B: 24x at the cfg-5 shape)
    const int m0 = blockIdx.x * BM, n0 = blockIdx.y * BN;
    // blockIdx.z = batch * splits + split; the batch strides shift all three matrices
    const int batch = blockIdx.z / splits;
    A += (long long)batch * sA; B += (long long)batch * sB; C += (long long)batch * sC;
    const long long kb = (long long)(blockIdx.z - batch * splits) * k_per_split;
    long long ke = kb + k_per_split; if (ke > K) ke = K;
    const int nk = (int)((ke - kb + BK - 1) / BK);

    constexpr int NA = TF32 ? 1 : 8;
    double acc[NA][4][2];
    float accf[TF32 ? 4 : 1][4][4];
#pragma unroll
    for (int i = 0; i < NA; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
#pragma unroll
    for (int i = 0; i < (TF32 ? 4 : 1); ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int q = 0; q < 4; ++q) accf[i][j][q] = 0.f;

    auto load_stage = [&](int stage, int kt) {
        const long long k0 = kb + (long long)kt * BK;
        // rows x 8 chunks of 16 B.  k and ke are even whenever k_per_split and K are even, so a chunk never straddles ke
#pragma unroll
        for (int i = 0; i < BM * 8 / NTHREADS; ++i) {
            const int c = tid + i * NTHREADS, row = c >> 3, ch = c & 7;
            const long long k = k0 + ch * 2;
            const bool pa = (m0 + row < M) && (k < ke);
            cp_async16(As + ((size_t)stage * BM + row) * PITCH_TN + ch * 2, pa ? A + (long long)(m0 + row) * lda + k : A, pa);
        }
#pragma unroll
        for (int i = 0; i < BN * 8 / NTHREADS; ++i) {
            const int c = tid + i * NTHREADS, row = c >> 3, ch = c & 7;
            const long long k = k0 + ch * 2;
            const bool pb = (n0 + row < Nn) && (k < ke);
            cp_async16(Bs + ((size_t)stage * BN + row) * PITCH_TN + ch * 2, pb ? B + (long long)(n0 + row) * ldb + k : B, pb);
        }
    };
#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) {
        if (s < nk) load_stage(s, s);
        cp_commit();
    }
    for (int kt = 0; kt < nk; ++kt) {
        cp_wait<STAGES - 2>();
        __syncthreads();
        if (kt + STAGES - 1 < nk) load_stage((kt + STAGES - 1) % STAGES, kt + STAGES - 1);
        cp_commit();
        const double* as = As + (size_t)(kt % STAGES) * BM * PITCH_TN + (wm * 64 + (lane >> 2)) * PITCH_TN + (lane & 3);
        const double* bs = Bs + (size_t)(kt % STAGES) * BN * PITCH_TN + (wn * 32 + (lane >> 2)) * PITCH_TN + (lane & 3);
        if constexpr (TF32) {
            const double* ta = As + (size_t)(kt % STAGES) * BM * PITCH_TN + wm * 64 * PITCH_TN;
            const double* tb = Bs + (size_t)(kt % STAGES) * BN * PITCH_TN + wn * 32 * PITCH_TN;
#pragma unroll
            for (int kk = 0; kk < BK; kk += 8)
                tf32x3_step(accf, ta + kk, PITCH_TN, 1, tb + kk, PITCH_TN, 1, lane >> 2, lane & 3);
            continue;
        }
#pragma unroll
        for (int kk = 0; kk < BK; kk += 4) {
            double a[8], b[4];
#pragma unroll
            for (int i = 0; i < 8; ++i) a[i] = as[i * 8 * PITCH_TN + kk];
#pragma unroll
            for (int j = 0; j < 4; ++j) b[j] = bs[j * 8 * PITCH_TN + kk];
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) dmma(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        }
    }
    cp_wait<0>();
    if constexpr (TF32) {
        // C fragment of m16n8: rows g, g + 8; cols 2 t, 2 t + 1
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int m = m0 + wm * 64 + i * 16 + h * 8 + (lane >> 2);
                if (m >= M) continue;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int n = n0 + wn * 32 + j * 8 + 2 * (lane & 3);
                    double* c = C + (long long)m * ldc + n;
                    const double v0 = (double)accf[i][j][2 * h], v1 = (double)accf[i][j][2 * h + 1];
                    if (use_atomic) {
                        if (n < Nn) atomicAdd(c, v0);
                        if (n + 1 < Nn) atomicAdd(c + 1, v1);
                    } else {
                        if (n < Nn) c[0] = v0;
                        if (n + 1 < Nn) c[1] = v1;
                    }
                }
            }
        return;
    }
    // C fragment: row = lane/4, cols 2*(lane%4), +1
#pragma unroll
    for (int i = 0; i < NA; ++i) {
        const int m = m0 + wm * 64 + i * 8 + (lane >> 2);
        if (m >= M) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int n = n0 + wn * 32 + j * 8 + 2 * (lane & 3);
            double* c = C + (long long)m * ldc + n;
            if (use_atomic) {
                if (n < Nn) atomicAdd(c, acc[i][j][0]);
                if (n + 1 < Nn) atomicAdd(c + 1, acc[i][j][1]);
            } else {
                if (n < Nn) c[0] = acc[i][j][0];
                if (n + 1 < Nn) c[1] = acc[i][j][1];
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// Y[n][k] += sum_m C[m][n] A[m][k].  Output tile: 128 vectors (n) x 128 reals (k).  MMA roles: rows = n, cols = k,
// contraction = m.  A-operand element (n, m) = C[m][n] (n contiguous), B-operand element (m, k) = A[m][k] (k contiguous).
template <bool TF32>
__global__ void __launch_bounds__(NTHREADS, MINB) gemm_update_kernel(int M, int Nn, long long K, const double* __restrict__ C, long long ldc,
                                                               const double* __restrict__ A, long long lda, double* __restrict__ Y,
                                                               long long ldy) {
    extern __shared__ __align__(16) double smem[];
    double* Cs = smem;                                        // [STAGES][BK][PITCH_UPC]  (m, n)
    double* As = smem + (size_t)STAGES * BK * PITCH_UPC;      // [STAGES][BK][PITCH_UPA]  (m, k)
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = warp / WN, wn = warp % WN;
    // Grouped tile order: consecutive CTAs sweep GN vector tiles of the SAME k tile before moving to the next k tile, so one wave works
    // on GN coefficient panels (C, rows x 128 vectors) and ~30 operator panels (A, rows x 64 reals) that fit the L2 together.  In plain
    // (k fastest) order every vector tile re-streamed the whole operator matrix from HBM (ncu at the cfg-5 shape: 481 GB read for 42 GB
    // of algorithmic traffic).
    constexpr int GN = 16;
    const long long id = blockIdx.x + (long long)gridDim.x * blockIdx.y;
    const long long per_group = (long long)GN * gridDim.x;
    const int grp = (int)(id / per_group);
    const int gsz = min(GN, (int)gridDim.y - grp * GN);
    const long long in_g = id - grp * per_group;
    const int n0 = (grp * GN + (int)(in_g % gsz)) * BM;
    const long long k0 = (in_g / gsz) * BN;
    const int nm = (M + BK - 1) / BK;

    constexpr int NA = TF32 ? 1 : 8;
    double acc[NA][4][2];
    float accf[TF32 ? 4 : 1][4][4];
#pragma unroll
    for (int i = 0; i < NA; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
#pragma unroll
    for (int i = 0; i < (TF32 ? 4 : 1); ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int q = 0; q < 4; ++q) accf[i][j][q] = 0.f;

    auto load_stage = [&](int stage, int mt) {
        const int mb = mt * BK;
        // 16 rows x (BM/2 | BN/2) chunks of 16 B
#pragma unroll
        for (int i = 0; i < BK * (BM / 2) / NTHREADS; ++i) {
            const int c = tid + i * NTHREADS, row = c / (BM / 2), ch = c % (BM / 2);
            const bool pc = (mb + row < M) && (n0 + ch * 2 < Nn);          // Nn, ldc even -> chunk never straddles
            cp_async16(Cs + ((size_t)stage * BK + row) * PITCH_UPC + ch * 2, pc ? C + (long long)(mb + row) * ldc + n0 + ch * 2 : C, pc);
        }
#pragma unroll
        for (int i = 0; i < BK * (BN / 2) / NTHREADS; ++i) {
            const int c = tid + i * NTHREADS, row = c / (BN / 2), ch = c % (BN / 2);
            const bool pa = (mb + row < M) && (k0 + ch * 2 < K);           // K, lda even
            cp_async16(As + ((size_t)stage * BK + row) * PITCH_UPA + ch * 2, pa ? A + (long long)(mb + row) * lda + k0 + ch * 2 : A, pa);
        }
    };
#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) {
        if (s < nm) load_stage(s, s);
        cp_commit();
    }
    for (int mt = 0; mt < nm; ++mt) {
        cp_wait<STAGES - 2>();
        __syncthreads();
        if (mt + STAGES - 1 < nm) load_stage((mt + STAGES - 1) % STAGES, mt + STAGES - 1);
        cp_commit();
        // A-operand (row n = lane/4, contraction m = lane%4): Cs[m][n];  B-operand (m = lane%4, col k = lane/4): As[m][k]
        const double* cs = Cs + (size_t)(mt % STAGES) * BK * PITCH_UPC + (lane & 3) * PITCH_UPC + wm * 64 + (lane >> 2);
        const double* as = As + (size_t)(mt % STAGES) * BK * PITCH_UPA + (lane & 3) * PITCH_UPA + wn * 32 + (lane >> 2);
        if constexpr (TF32) {
            // MMA rows = n (A-operand element (n, m) = Cs[m][n]), cols = k (B-operand element (m, k) = As[m][k]), contraction = m
            const double* ta = Cs + (size_t)(mt % STAGES) * BK * PITCH_UPC + wm * 64;
            const double* tb = As + (size_t)(mt % STAGES) * BK * PITCH_UPA + wn * 32;
#pragma unroll
            for (int mm = 0; mm < BK; mm += 8)
                tf32x3_step(accf, ta + mm * PITCH_UPC, 1, PITCH_UPC, tb + mm * PITCH_UPA, 1, PITCH_UPA,
                            lane >> 2, lane & 3);
            continue;
        }
#pragma unroll
        for (int mm = 0; mm < BK; mm += 4) {
            double a[8], b[4];
#pragma unroll
            for (int i = 0; i < 8; ++i) a[i] = cs[mm * PITCH_UPC + i * 8];
#pragma unroll
            for (int j = 0; j < 4; ++j) b[j] = as[mm * PITCH_UPA + j * 8];
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) dmma(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        }
    }
    cp_wait<0>();
    if constexpr (TF32) {
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int n = n0 + wm * 64 + i * 16 + h * 8 + (lane >> 2);
                if (n >= Nn) continue;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const long long k = k0 + wn * 32 + j * 8 + 2 * (lane & 3);
                    if (k < K) {
                        double2* y = reinterpret_cast<double2*>(Y + (long long)n * ldy + k);
                        double2 v = *y;
                        v.x += (double)accf[i][j][2 * h]; v.y += (double)accf[i][j][2 * h + 1];
                        *y = v;
                    }
                }
            }
        return;
    }
#pragma unroll
    for (int i = 0; i < NA; ++i) {
        const int n = n0 + wm * 64 + i * 8 + (lane >> 2);
        if (n >= Nn) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const long long k = k0 + wn * 32 + j * 8 + 2 * (lane & 3);
            if (k < K) {                                        // K even: k and k+1 are both valid
                double2* y = reinterpret_cast<double2*>(Y + (long long)n * ldy + k);
                double2 v = *y;
                v.x += acc[i][j][0]; v.y += acc[i][j][1];
                *y = v;
            }
        }
    }
}

}  // namespace wgemm
