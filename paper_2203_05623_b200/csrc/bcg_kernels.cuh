// True block CG over the perturbations of one orbital (second half; reading R8b of DESIGN.md): the s right-hand sides
// b_iv, i = 1..s, of Eq. 10 that share the operator A_v = H - eps_v + alpha_v P_v are solved in ONE Krylov space,
//   Q = A P ;  G = P^T Q ;  alpha = G^+ (P^T R) ;  X += P alpha ;  R -= Q alpha ;  Z = M R ;  beta = G^+ (Q^T Z) ;  P = Z - P beta
// (O'Leary's block CG written with Gram matrices of the search block only, so that a rank-deficient search block - columns that
// converged, or became linearly dependent - is handled by a rank-revealing solve: G^+ is the inverse of G on the span of the pivot
// columns a diagonally pivoted Cholesky factorisation of the unit-diagonal scaled G accepts, i.e. dependent directions are dropped).
// The answer is the same dpsi ("solved independently for each perturbation" is a statement about the equations, not about
// the Krylov space); only the iteration count changes.  omega = 0 only (real symmetric positive definite operator).
//
// Layout: columns are [perturbation j][orbital v'] in compacted orbital order (n_orb active orbitals), every column K = 2 n_g reals;
// the block of orbital v' is the s columns j * n_orb + v', i.e. row stride n_orb * K.  Inner product: WEST_GAMMA <f,g> = 2 sum_reals f g
// - f(0) g(0) (real functions on the half sphere), WEST_FULL Re <f,g> = sum_reals f g (the Hermitian operator is real symmetric on R^2n).
#pragma once
#include <cuda_runtime.h>

namespace wbcg {

constexpr int SMAX = 128;          // largest block (perturbations per orbital) the coefficient kernel holds in shared memory

// ------------------------------------------------------------------------------------------------------------------- Gram blocks
// C_v[i][j] (+)= w * sum_{k in split} A_v[i][k] B_v[j][k]  (- A_v[i][0] B_v[j][0] in the split holding k = 0 when gamma), w = 2 | 1.
// CTA = one orbital x one TS x TS tile of the s x s block x one K split.  (TS/4)^2 threads own 4 x 4 outputs each (rows ti + (TS/4) a,
// columns tj + (TS/4) b: conflict-free shared-memory reads with an odd pitch), KS = 256 / (TS/4)^2 thread groups split the k of a tile.
template <int TS>
__global__ void __launch_bounds__(256) gram_kernel(int s, long long K, int n_orb, const int* __restrict__ orbmap, const double* __restrict__ A,
                                                   const double* __restrict__ B, double* __restrict__ C, int gamma, int splits, long long k_per_split) {
    constexpr int Q4 = TS / 4, NT2 = Q4 * Q4, KS = 256 / NT2, KT = 32, PITCH = KT + 1;
    __shared__ double As[TS * PITCH], Bs[TS * PITCH];
    __shared__ double red[KS > 1 ? 256 * 4 : 1];
    const int v = blockIdx.x;
    if (orbmap && orbmap[v] < 0) return;
    const int tiles = (s + TS - 1) / TS;
    const int tile = blockIdx.y % (tiles * tiles), split = blockIdx.y / (tiles * tiles);
    const int i0 = (tile / tiles) * TS, j0 = (tile % tiles) * TS;
    const long long row = (long long)n_orb * K;                  // stride between the block's columns
    const double* Av = A + (long long)v * K;
    const double* Bv = B + (long long)v * K;
    const long long kb = (long long)split * k_per_split;
    long long ke = kb + k_per_split; if (ke > K) ke = K;
    const int t = threadIdx.x, ks = t / NT2, tt = t % NT2, ti = tt / Q4, tj = tt % Q4;
    double acc[4][4];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) acc[a][b] = 0.0;
    for (long long k0 = kb; k0 < ke; k0 += KT) {
        // stage TS rows x KT reals of both operands (rows beyond s and k beyond ke read as zero)
        for (int e = t; e < TS * KT; e += 256) {
            const int r = e / KT, kk = e % KT;
            const long long k = k0 + kk;
            const bool okk = k < ke;
            As[r * PITCH + kk] = (okk && i0 + r < s) ? Av[(long long)(i0 + r) * row + k] : 0.0;
            Bs[r * PITCH + kk] = (okk && j0 + r < s) ? Bv[(long long)(j0 + r) * row + k] : 0.0;
        }
        __syncthreads();
#pragma unroll 4
        for (int kk = ks; kk < KT; kk += KS) {
            double a[4], b[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) { a[q] = As[(ti + Q4 * q) * PITCH + kk]; b[q] = Bs[(tj + Q4 * q) * PITCH + kk]; }
#pragma unroll
            for (int x = 0; x < 4; ++x)
#pragma unroll
                for (int y = 0; y < 4; ++y) acc[x][y] = fma(a[x], b[y], acc[x][y]);
        }
        __syncthreads();
    }
    // fold the KS k-groups (shared memory, four outputs per round), then the Gamma weighting and the store / atomic add
    const double w = gamma ? 2.0 : 1.0;
    double* Cv = C + (long long)v * s * s;
#pragma unroll
    for (int x = 0; x < 4; ++x) {
        if (KS > 1) {
#pragma unroll
            for (int y = 0; y < 4; ++y) red[(y * KS + ks) * NT2 + tt] = acc[x][y];
            __syncthreads();
            if (ks == 0) {
#pragma unroll
                for (int y = 0; y < 4; ++y) {
                    double sum = 0.0;
                    for (int q = 0; q < KS; ++q) sum += red[(y * KS + q) * NT2 + tt];
                    acc[x][y] = sum;
                }
            }
            __syncthreads();
        }
        if (ks == 0) {
            const int i = i0 + ti + Q4 * x;
#pragma unroll
            for (int y = 0; y < 4; ++y) {
                const int j = j0 + tj + Q4 * y;
                if (i < s && j < s) {
                    double val = w * acc[x][y];
                    if (gamma && kb == 0) val -= Av[(long long)i * row] * Bv[(long long)j * row];
                    if (splits > 1) atomicAdd(Cv + (long long)i * s + j, val);
                    else Cv[(long long)i * s + j] = val;
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------------------------ block updates
// Y_v[j][k] += sign * sum_m C_v[m][j] P_v[m][k],  j in this CTA's block of JB outputs.  One thread per pair of reals k (16-byte accesses),
// the coefficient block in shared memory (read as broadcasts), JB accumulator pairs in registers.
// Output addressing: Y column of (j, v) = j * out_stride + (out_orb ? out_orb[v] : v) columns of K reals (X lives in the caller's
// original [perturbation][orbital] order, R / Z in compacted order).
template <int JB>
__global__ void __launch_bounds__(256) update_kernel(int s, long long K, int n_orb, const int* __restrict__ orbmap, const double* __restrict__ C,
                                                     const double* __restrict__ P, double* __restrict__ Y, long long out_stride,
                                                     const int* __restrict__ out_orb, double sign) {
    extern __shared__ __align__(16) double Cs[];        // [s][JB]
    const int v = blockIdx.y;
    if (orbmap && orbmap[v] < 0) return;
    const int jb = blockIdx.z * JB;
    const double* Cv = C + (long long)v * s * s;
    for (int e = threadIdx.x; e < s * JB; e += 256) {
        const int m = e / JB, j = e % JB;
        Cs[e] = (jb + j < s) ? Cv[(long long)m * s + jb + j] : 0.0;
    }
    __syncthreads();
    const long long k = ((long long)blockIdx.x * 256 + threadIdx.x) * 2;
    if (k >= K) return;
    const long long row = (long long)n_orb * K;
    const double* Pv = P + (long long)v * K + k;
    double2 acc[JB];
#pragma unroll
    for (int j = 0; j < JB; ++j) acc[j] = make_double2(0.0, 0.0);
#pragma unroll 2
    for (int m = 0; m < s; ++m) {
        const double2 p = *reinterpret_cast<const double2*>(Pv + (long long)m * row);
        const double2* c2 = reinterpret_cast<const double2*>(Cs + m * JB);
#pragma unroll
        for (int j = 0; j < JB; j += 2) {
            const double2 c = c2[j / 2];
            acc[j].x = fma(c.x, p.x, acc[j].x); acc[j].y = fma(c.x, p.y, acc[j].y);
            acc[j + 1].x = fma(c.y, p.x, acc[j + 1].x); acc[j + 1].y = fma(c.y, p.y, acc[j + 1].y);
        }
    }
    const long long ocol = out_orb ? out_orb[v] : v;
#pragma unroll
    for (int j = 0; j < JB; ++j) {
        if (jb + j >= s) break;
        double2* y = reinterpret_cast<double2*>(Y + ((long long)(jb + j) * out_stride + ocol) * K + k);
        double2 o = *y;
        o.x = fma(sign, acc[j].x, o.x); o.y = fma(sign, acc[j].y, o.y);
        *y = o;
    }
}

// ----------------------------------------------------------------------------------------------------- coefficients: C = G^+ T
struct Fac {            // per-orbital factorisation kept between the alpha and the beta solve of one iteration
    double* L;          // [n_orb][s][s]  L[k][i]: column k of the Cholesky factor (pivot order), indexed by the original row i
    double* D;          // [n_orb][s]     diagonal scaling 1 / sqrt(G_ii) (0: direction dropped)
    int* order;         // [n_orb][s]     pivot order
    int* rank;          // [n_orb]
};

// mode 0: factor the block's G (symmetrised, scaled to unit diagonal, diagonally pivoted Cholesky stopped at pivot < tau) and solve;
// mode 1: solve with the stored factor.  C_v = sign * G^+ T_v, rows of dropped directions zero.  One CTA of 256 threads per orbital.
__global__ void __launch_bounds__(256) coef_kernel(int s, int mode, const int* __restrict__ orbmap, const double* __restrict__ G,
                                                   const double* __restrict__ T, double* __restrict__ C, Fac f, double tau, double sign) {
    extern __shared__ __align__(16) double sm[];
    const int PITCH = s | 1;
    double* A = sm;                               // [s][PITCH]: G during the factorisation, then the right-hand sides / solutions
    double* dg = A + s * PITCH;                   // [s] running diagonal
    double* lc = dg + s;                          // [s] current column
    double* Ds = lc + s;                          // [s]
    int* done = reinterpret_cast<int*>(Ds + s);   // [s]
    int* ord = done + s;                          // [s]
    __shared__ int s_p, s_rank;
    __shared__ double s_piv;
    const int v = blockIdx.x, t = threadIdx.x;
    if (orbmap && orbmap[v] < 0) return;
    double* Lv = f.L + (long long)v * s * s;
    if (mode == 0) {
        const double* Gv = G + (long long)v * s * s;
        for (int i = t; i < s; i += 256) {
            const double d = Gv[(long long)i * s + i];
            Ds[i] = (d > 0.0 && isfinite(d)) ? rsqrt(d) : 0.0;
            done[i] = 0;
        }
        __syncthreads();
        for (int e = t; e < s * s; e += 256) {
            const int i = e / s, j = e % s;
            A[i * PITCH + j] = 0.5 * (Gv[(long long)i * s + j] + Gv[(long long)j * s + i]) * Ds[i] * Ds[j];
        }
        __syncthreads();
        for (int i = t; i < s; i += 256) dg[i] = A[i * PITCH + i];
        if (t == 0) s_rank = 0;
        __syncthreads();
        for (int k = 0; k < s; ++k) {
            if (t < 32) {                          // pivot: largest remaining diagonal (ties -> lowest index)
                double best = -1.0; int bi = -1;
                for (int i = t; i < s; i += 32)
                    if (!done[i] && dg[i] > best) { best = dg[i]; bi = i; }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    const double ob = __shfl_xor_sync(0xffffffffu, best, o);
                    const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
                    if (ob > best || (ob == best && oi >= 0 && (bi < 0 || oi < bi))) { best = ob; bi = oi; }
                }
                if (t == 0) { s_p = bi; s_piv = best; }
            }
            __syncthreads();
            const int p = s_p;
            const double piv = s_piv;
            if (p < 0 || !(piv >= tau)) break;
            const double lkk = sqrt(piv);
            for (int i = t; i < s; i += 256) {
                const double l = i == p ? lkk : (done[i] ? 0.0 : A[i * PITCH + p] / lkk);
                lc[i] = l;
                Lv[(long long)k * s + i] = l;
            }
            __syncthreads();
            if (t == 0) { done[p] = 1; ord[k] = p; s_rank = k + 1; }
            for (int e = t; e < s * s; e += 256) {
                const int i = e / s, j = e % s;
                if (i != p && j != p && !done[i] && !done[j]) A[i * PITCH + j] -= lc[i] * lc[j];
            }
            for (int i = t; i < s; i += 256)
                if (i != p && !done[i]) dg[i] -= lc[i] * lc[i];
            __syncthreads();
        }
        __syncthreads();
        for (int i = t; i < s; i += 256) { f.D[(long long)v * s + i] = Ds[i]; f.order[(long long)v * s + i] = i < s_rank ? ord[i] : -1; }
        if (t == 0) f.rank[v] = s_rank;
    } else {
        for (int i = t; i < s; i += 256) { Ds[i] = f.D[(long long)v * s + i]; ord[i] = f.order[(long long)v * s + i]; }
        if (t == 0) s_rank = f.rank[v];
    }
    __syncthreads();
    const int r = s_rank;
    // right-hand sides in pivot order: A[a][j] = D[ord a] T[ord a][j]
    const double* Tv = T + (long long)v * s * s;
    for (int e = t; e < r * s; e += 256) {
        const int a = e / s, j = e % s;
        A[a * PITCH + j] = Ds[ord[a]] * Tv[(long long)ord[a] * s + j];
    }
    __syncthreads();
    double* Cv = C + (long long)v * s * s;
    for (int j = t; j < s; j += 256) {            // one right-hand side per thread (s <= 128 <= 256: one round)
        for (int a = 0; a < r; ++a) {             // L y = rhs
            const int pa = ord[a];
            double y = A[a * PITCH + j];
            for (int c = 0; c < a; ++c) y -= Lv[(long long)c * s + pa] * A[c * PITCH + j];
            A[a * PITCH + j] = y / Lv[(long long)a * s + pa];
        }
        for (int a = r - 1; a >= 0; --a) {        // L^T x = y
            double x = A[a * PITCH + j];
            for (int c = a + 1; c < r; ++c) x -= Lv[(long long)a * s + ord[c]] * A[c * PITCH + j];
            A[a * PITCH + j] = x / Lv[(long long)a * s + ord[a]];
        }
        for (int i = 0; i < s; ++i) Cv[(long long)i * s + j] = 0.0;
        for (int a = 0; a < r; ++a) Cv[(long long)ord[a] * s + j] = sign * Ds[ord[a]] * A[a * PITCH + j];
    }
}
inline size_t coef_smem(int s) { return sizeof(double) * ((size_t)s * (s | 1) + 3 * (size_t)s) + sizeof(int) * 2 * (size_t)s; }

// -------------------------------------------------------------------------------------- Z = M R, column norms, convergence flags
struct State {
    double* b2;         // [n_col] ||b||^2 per ORIGINAL column (j * n_occ + v)
    double* rr;         // [n_col] ||r||^2
    int* n_open;        // [n_occ] columns of the orbital still above tol (recounted every iteration)
    int* active;        // [n_occ] orbital still iterating
    int* iters;         // [n_occ] iterations the orbital's block took part in
    int* counters;      // [0] live orbitals
};

__device__ __forceinline__ double bcg_precond(double g2, double tk, int on) {
    if (on == 0) return 1.0;
    if (on == 2) {
        const double x = g2 / (1.5 * tk);
        const double num = 27.0 + x * (18.0 + x * (12.0 + 8.0 * x));
        return num / (num + 16.0 * x * x * x * x);
    }
    return 1.0 / fmax(1.0, g2 / (WEST_PC_C * tk));
}

// One CTA per compacted column c = j * n_orb + v'.  init != 0: also b2 = rr.
__global__ void __launch_bounds__(256) zr_kernel(long long n_g, int n_orb, int n_occ, int gamma, const int* __restrict__ orbmap,
                                                 const double* __restrict__ g2, const double* __restrict__ tk, int precond_on, double tol2, int init,
                                                 const double2* __restrict__ R, double2* __restrict__ Z, State st) {
    __shared__ double red[8];
    const int c = blockIdx.x, j = c / n_orb, vp = c % n_orb;
    const int v = orbmap ? orbmap[vp] : vp;
    if (v < 0) return;
    const double2* r = R + (long long)c * n_g;
    double2* z = Z + (long long)c * n_g;
    const double tkv = tk[v];
    double acc = 0.0;
    for (long long g = threadIdx.x; g < n_g; g += 256) {
        const double2 x = r[g];
        const double m = bcg_precond(g2[g], tkv, precond_on);
        z[g] = make_double2(m * x.x, m * x.y);
        acc += gamma ? (g == 0 ? x.x * x.x : 2.0 * (x.x * x.x + x.y * x.y)) : x.x * x.x + x.y * x.y;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < 8; ++w) s += red[w];
        const long long col = (long long)j * n_occ + v;
        st.rr[col] = s;
        if (init) st.b2[col] = s;
        const double b2 = init ? s : st.b2[col];
        if (s > tol2 * b2) atomicAdd(st.n_open + v, 1);
    }
}
// per orbital: close it when none of its columns is above tol; count the iteration.  start != 0: set up the flags instead.
__global__ void flags_kernel(int n_orb, const int* __restrict__ orbmap, int start, State st) {
    const int vp = blockIdx.x * blockDim.x + threadIdx.x;
    if (vp >= n_orb) return;
    const int v = orbmap ? orbmap[vp] : vp;
    if (v < 0) return;
    const int open = st.n_open[v];
    st.n_open[v] = 0;
    if (start) {
        st.active[v] = open > 0;
        st.iters[v] = 0;
        if (open > 0) atomicAdd(st.counters, 1);
    } else if (st.active[v]) {
        st.iters[v] += 1;
        if (open == 0) { st.active[v] = 0; atomicSub(st.counters, 1); }
    }
}
// compacted column -> original column (j * n_occ + orbital), -1 for inert padding
__global__ void colmap_kernel(int n_orb, int s, int n_occ, const int* __restrict__ orbmap, int* __restrict__ colmap) {
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n_orb * s) return;
    const int j = c / n_orb, vp = c % n_orb;
    const int v = orbmap ? orbmap[vp] : vp;
    colmap[c] = v < 0 ? -1 : j * n_occ + v;
}
// gather whole orbital blocks: out column (j, v'') <- in column (j, src[v''])
__global__ void __launch_bounds__(256) gather_blocks(long long n_g, int n_new, int n_old, const int* __restrict__ src, const double2* __restrict__ in,
                                                     double2* __restrict__ out) {
    const int c = blockIdx.x, j = c / n_new, vp = c % n_new;
    const double2* a = in + ((long long)j * n_old + src[vp]) * n_g;
    double2* b = out + (long long)c * n_g;
    for (long long g = threadIdx.x; g < n_g; g += 256) b[g] = a[g];
}
// final report, out[4]: max relative residual, number of columns above tol, min and max block iterations over the non-zero orbitals
__global__ void report_kernel(int n_col, int n_occ, double tol2, State st, double* out) {
    __shared__ double shm[256]; __shared__ int shc[256], shlo[256], shhi[256];
    double m = 0; int c = 0, lo = 0x7fffffff, hi = 0;
    for (int i = threadIdx.x; i < n_col; i += 256) {
        const double b2 = st.b2[i];
        if (b2 > 0) { const double q = st.rr[i] / b2; m = fmax(m, q); c += q > tol2; const int it = st.iters[i % n_occ]; lo = min(lo, it); hi = max(hi, it); }
    }
    shm[threadIdx.x] = m; shc[threadIdx.x] = c; shlo[threadIdx.x] = lo; shhi[threadIdx.x] = hi;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) {
            shm[threadIdx.x] = fmax(shm[threadIdx.x], shm[threadIdx.x + o]); shc[threadIdx.x] += shc[threadIdx.x + o];
            shlo[threadIdx.x] = min(shlo[threadIdx.x], shlo[threadIdx.x + o]); shhi[threadIdx.x] = max(shhi[threadIdx.x], shhi[threadIdx.x + o]);
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) { out[0] = sqrt(shm[0]); out[1] = (double)shc[0]; out[2] = (double)(shlo[0] == 0x7fffffff ? 0 : shlo[0]); out[3] = (double)shhi[0]; }
}

}  // namespace wbcg
