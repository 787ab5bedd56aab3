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

}  // namespace wlz
