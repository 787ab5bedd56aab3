// Lanczos chains of the wfreq step (Eq. 15-18): one chain per column (perturbation m, orbital i),
// all columns advanced together with west's batched H*psi.  One CTA per column, three fused phases per step:
//   alpha = <q, Hq> ;  w = Hq - alpha q - beta_prev q_prev ;  beta = ||w|| ;  q_next = w / beta     (no re-orthogonalisation, as Eq. 15)
// GAMMA = real functions on the half sphere (<f,g> = 2 sum_reals - f(0) g(0)); otherwise complex vectors, Hermitian product.
#pragma once
#include "cg_kernels.cuh"

namespace wlz {
using wcg::NT;
using wcg::block_reduce;

template <bool GAMMA>
__device__ __forceinline__ double herm_re(const double2 x, const double2 y, int g) {
    const double d = x.x * y.x + x.y * y.y;
    return GAMMA ? (g == 0 ? x.x * y.x : 2.0 * d) : d;
}

// q <- q / ||q||, norm[col] = ||q||, optional copy of the normalised start vector
template <bool GAMMA>
__global__ void __launch_bounds__(NT) lz_normalize(long long n_g, double2* Q, double2* Q1_opt, double* norm, double* beta_prev) {
    __shared__ double sh[32];
    const int col = blockIdx.x;
    double2* q = Q + (long long)col * n_g;
    double acc[1] = {0};
    for (int g = threadIdx.x; g < n_g; g += NT) acc[0] += herm_re<GAMMA>(q[g], q[g], g);
    block_reduce<1>(acc, sh);
    const double nrm = sqrt(acc[0]), inv = nrm > 0 ? 1.0 / nrm : 0.0;
    for (int g = threadIdx.x; g < n_g; g += NT) {
        double2 v = q[g];
        v.x *= inv; v.y *= inv;
        if (GAMMA && g == 0) v.y = 0.0;
        q[g] = v;
        if (Q1_opt) Q1_opt[(long long)col * n_g + g] = v;
    }
    if (threadIdx.x == 0) { norm[col] = nrm; beta_prev[col] = 0.0; }
}

// one Lanczos step; QP holds q^{l-1} on entry and q^{l+1} on exit
template <bool GAMMA>
__global__ void __launch_bounds__(NT) lz_step(long long n_g, int n_steps, int l, const double2* Q, const double2* HQ, double2* QP,
                                              double* alpha, double* beta, double* beta_prev) {
    __shared__ double sh[32];
    const int col = blockIdx.x;
    const double2* q = Q + (long long)col * n_g; const double2* hq = HQ + (long long)col * n_g;
    double2* qp = QP + (long long)col * n_g;
    double acc[1] = {0};
    for (int g = threadIdx.x; g < n_g; g += NT) acc[0] += herm_re<GAMMA>(q[g], hq[g], g);
    block_reduce<1>(acc, sh);
    const double a = acc[0], bp = beta_prev[col];
    acc[0] = 0;
    for (int g = threadIdx.x; g < n_g; g += NT) {
        const double2 x = q[g], h = hq[g], p = qp[g];
        double2 w = make_double2(h.x - a * x.x - bp * p.x, h.y - a * x.y - bp * p.y);
        if (GAMMA && g == 0) w.y = 0.0;
        qp[g] = w;
        acc[0] += herm_re<GAMMA>(w, w, g);
    }
    block_reduce<1>(acc, sh);
    const double b = sqrt(acc[0]), inv = b > 0 ? 1.0 / b : 0.0;
    for (int g = threadIdx.x; g < n_g; g += NT) {
        double2 w = qp[g];
        w.x *= inv; w.y *= inv;
        qp[g] = w;
    }
    if (threadIdx.x == 0) {
        alpha[(long long)col * n_steps + l] = a;
        beta[(long long)col * n_steps + l] = b;
        beta_prev[col] = b;
    }
}

// GAMMA inner-product fix of a batch of Gram blocks: C[b][n][m] <- 2 C - A_n(0) B_m(0)   (real parts of the G = 0 coefficients)
__global__ void braket_fix(int n_batch, int n, long long sC, double* C, const double* A, const double* B, long long ld, long long sAB) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)n_batch * n * n) return;
    const int b = (int)(i / ((long long)n * n));
    const int r = (int)(i - (long long)b * n * n), row = r / n, colm = r - row * n;
    double* c = C + (long long)b * sC + (long long)row * n + colm;
    *c = 2.0 * (*c) - A[(long long)b * sAB + (long long)row * ld] * B[(long long)b * sAB + (long long)colm * ld];
}

// Eigenvalues d and eigenvectors U of the Lanczos tridiagonal matrices of Eq. 19, one WARP per chain:
//   T = tridiag(beta^2 .. beta^L ; alpha^1 .. alpha^L ; beta^2 .. beta^L),  T = U diag(d) U^T,  d ascending, U[0][l'] >= 0.
// Implicit-shift QL iteration (Wilkinson shift, Givens chase from the bottom of the unreduced block to its top), the
// textbook method for symmetric tridiagonal matrices.  The scalar recurrence on d, e is carried redundantly by every lane (warp-uniform
// control flow); each plane rotation is applied to the eigenvector matrix with one row per lane (n <= 64: two rows per lane).
// alpha, beta: [n_chain][n] as west_lanczos writes them (beta[l] = the off-diagonal between l and l+1; beta[n-1] is not part of T).
// d_out [n_chain][n]; U_out [n_chain][n][n] row-major, U[l][l'] = component l of eigenvector l'; status[chain] = sweeps used, or -1
// if some eigenvalue did not converge in 60 sweeps.
constexpr int TRI_MAX = 64, TRI_WARPS = 4;
__global__ void __launch_bounds__(32 * TRI_WARPS) tridiag_eig(int n_chain, int n, const double* __restrict__ alpha, const double* __restrict__ beta,
                                                              double* __restrict__ d_out, double* __restrict__ U_out, int* __restrict__ status, int* __restrict__ n_failed) {
    extern __shared__ double sm[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int chain = blockIdx.x * TRI_WARPS + warp;
    if (chain >= n_chain) return;                               // whole warps leave together; only __syncwarp below
    double* d = sm + (size_t)warp * (2 * TRI_MAX + (size_t)n * (n + 1));
    double* e = d + TRI_MAX;
    double* Z = e + TRI_MAX;                                    // [n][n + 1]: row k at pitch n + 1 (conflict-free column access)
    const int P = n + 1;
    for (int i = lane; i < n; i += 32) {
        d[i] = alpha[(long long)chain * n + i];
        e[i] = i + 1 < n ? beta[(long long)chain * n + i] : 0.0;
    }
    for (int i = lane; i < n * P; i += 32) Z[i] = 0.0;
    __syncwarp();
    for (int i = lane; i < n; i += 32) Z[i * P + i] = 1.0;
    __syncwarp();
    int sweeps = 0;
    bool ok = true;
    for (int l = 0; l < n && ok; ++l) {
        int iter = 0;
        while (true) {
            int m = l;
            for (; m < n - 1; ++m) {
                const double dd = fabs(d[m]) + fabs(d[m + 1]);
                if (fabs(e[m]) <= 2.220446049250313e-16 * dd) break;
            }
            if (m == l) break;
            if (++iter > 60) { ok = false; break; }
            ++sweeps;
            double g = (d[l + 1] - d[l]) / (2.0 * e[l]);
            double r = hypot(g, 1.0);
            g = d[m] - d[l] + e[l] / (g + copysign(r, g));
            double sn = 1.0, cs = 1.0, pp = 0.0;
            int i = m - 1;
            bool deflated = false;
            __syncwarp();
            for (; i >= l; --i) {
                double f = sn * e[i];
                const double b = cs * e[i];
                r = hypot(f, g);
                double e_next = r;
                if (r == 0.0) {                                 // the chase recovered a zero off-diagonal: split here
                    __syncwarp();
                    if (lane == 0) { e[i + 1] = 0.0; d[i + 1] -= pp; e[m] = 0.0; }
                    deflated = true;
                    break;
                }
                sn = f / r; cs = g / r;
                g = d[i + 1] - pp;
                r = (d[i] - g) * sn + 2.0 * cs * b;
                pp = sn * r;
                const double d_next = g + pp;
                g = cs * r - b;
                __syncwarp();                                   // every lane has read e[i], d[i], d[i + 1]
                if (lane == 0) { e[i + 1] = e_next; d[i + 1] = d_next; }
                for (int k = lane; k < n; k += 32) {            // rotate columns i, i + 1 of Z
                    f = Z[k * P + i + 1];
                    const double zi = Z[k * P + i];
                    Z[k * P + i + 1] = sn * zi + cs * f;
                    Z[k * P + i] = cs * zi - sn * f;
                }
                __syncwarp();
            }
            __syncwarp();
            if (!deflated) {
                if (lane == 0) { d[l] -= pp; e[l] = g; e[m] = 0.0; }
            }
            __syncwarp();
        }
    }
    __syncwarp();
    // ascending order by rank (ties by index), sign U[0][l'] >= 0, written straight to the output
    for (int j = lane; j < n; j += 32) {
        const double dj = d[j];
        int rank = 0;
        for (int i = 0; i < n; ++i) rank += (d[i] < dj) || (d[i] == dj && i < j);
        e[j] = (double)rank;                                    // e is free now
        d_out[(long long)chain * n + rank] = dj;
    }
    __syncwarp();
    double* U = U_out + (long long)chain * n * n;
    for (int idx = lane; idx < n * n; idx += 32) {
        const int k = idx / n, j = idx - k * n;
        const double sgn = Z[j] < 0.0 ? -1.0 : 1.0;             // Z[0][j]
        U[(long long)k * n + (int)e[j]] = sgn * Z[k * P + j];
    }
    if (lane == 0) {
        if (status) status[chain] = ok ? sweeps : -1;
        if (!ok) atomicAdd(n_failed, 1);
    }
}

}  // namespace wlz
