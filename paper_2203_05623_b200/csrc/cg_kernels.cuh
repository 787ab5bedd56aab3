// Batched preconditioned CG / COCG for Eq. 10: one recurrence per column (perturbation i, state v),
// all columns advanced together, per-column scalars kept on the device.  Readings R3-R5, R7 of DESIGN.md.
//   MODE 0  WEST_GAMMA, omega = 0 : real functions, <f,g> = 2 sum_reals f g - f(0) g(0)
//   MODE 1  WEST_GAMMA, omega > 0 : column = (Re, Im) pair of real functions, COCG with the unconjugated bilinear form
//                                   (x,y) = <xR,yR> - <xI,yI> + i(<xR,yI> + <xI,yR>)  = int x(r) y(r) dr
//   MODE 2  WEST_FULL,  omega = 0 : complex vectors, Hermitian inner product
// One CTA per column; vectors are [col][nvpc][n_g] complex128, nvpc = 2 in MODE 1 else 1.
#pragma once
#include <cuda_runtime.h>
#include <cooperative_groups.h>

namespace wcg {

constexpr int NT = 256;
#ifndef WEST_PC_C
#define WEST_PC_C 1.35      // crossover of the default diagonal preconditioner in units of <psi_v|T|psi_v> (reading R4)
#endif

struct Scalars {
    double2* rz;      // (r, z)
    double*  rr;      // Hermitian ||r||^2
    double*  b2;      // ||b||^2
    int*     active;  // 1 while ||r|| > tol ||b||
    int*     iters;   // iterations this column took part in
    int*     counters;   // [0] number of active columns after the last p-update
};

__device__ __forceinline__ double2 cdiv(double2 a, double2 b) {
    const double d = b.x * b.x + b.y * b.y;
    return make_double2((a.x * b.x + a.y * b.y) / d, (a.y * b.x - a.x * b.y) / d);
}

__device__ __forceinline__ double2 cmul2(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }

// block reduction of up to 4 doubles
template <int NV>
__device__ __forceinline__ void block_reduce(double (&v)[NV], double* sh /* [NV*8] */) {
#pragma unroll
    for (int i = 0; i < NV; ++i)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[i] += __shfl_xor_sync(0xffffffffu, v[i], o);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0)
#pragma unroll
        for (int i = 0; i < NV; ++i) sh[i * 8 + warp] = v[i];
    __syncthreads();
#pragma unroll
    for (int i = 0; i < NV; ++i) {
        double s = 0;
#pragma unroll
        for (int w = 0; w < NT / 32; ++w) s += sh[i * 8 + w];
        v[i] = s;
    }
    __syncthreads();
}

// Diagonal preconditioners M_v(G) (reading R4; they change iteration counts only, never the converged result):
//   1: 1 / max(1, |G|^2 / (1.35 <psi_v|T|psi_v>))                      (the reading's default)
//   2: Teter-Payne-Allan: (27 + 18x + 12x^2 + 8x^3) / (27 + 18x + 12x^2 + 8x^3 + 16x^4), x = |G|^2 / (1.5 <psi_v|T|psi_v>)
__device__ __forceinline__ double precond(double g2, double tk, int on) {
    if (on == 0) return 1.0;
    if (on == 2) {
        const double x = g2 / (1.5 * tk);
        const double num = 27.0 + x * (18.0 + x * (12.0 + 8.0 * x));
        return num / (num + 16.0 * x * x * x * x);
    }
    const double q = g2 / (WEST_PC_C * tk);
    return 1.0 / fmax(1.0, q);
}

// accumulate the mode's inner products of (a, b) over this thread's elements.  out: [0]=re, [1]=im
template <int MODE>
__device__ __forceinline__ void dot_accum(const double2* a, const double2* b, long long n_g, int g, double w, double (&acc)[2]) {
    // w: extra real weight on b (preconditioner), applied as a -> (a, w b)
    if (MODE == 0) {
        const double2 x = a[g], y = b[g];
        acc[0] += (g == 0 ? x.x * y.x : 2.0 * (x.x * y.x + x.y * y.y)) * w;
    } else if (MODE == 1) {
        const double2 xr = a[g], xi = a[n_g + g], yr = b[g], yi = b[n_g + g];
        const double f = g == 0 ? 1.0 : 2.0;
        const double rr = g == 0 ? xr.x * yr.x : xr.x * yr.x + xr.y * yr.y;
        const double ii = g == 0 ? xi.x * yi.x : xi.x * yi.x + xi.y * yi.y;
        const double ri = g == 0 ? xr.x * yi.x : xr.x * yi.x + xr.y * yi.y;
        const double ir = g == 0 ? xi.x * yr.x : xi.x * yr.x + xi.y * yr.y;
        acc[0] += f * (rr - ii) * w;
        acc[1] += f * (ri + ir) * w;
    } else {
        const double2 x = a[g], y = b[g];
        acc[0] += (x.x * y.x + x.y * y.y) * w;
        acc[1] += (x.x * y.y - x.y * y.x) * w;
    }
}
template <int MODE>
__device__ __forceinline__ double norm_accum(const double2* a, long long n_g, int g) {
    if (MODE == 0) { const double2 x = a[g]; return g == 0 ? x.x * x.x : 2.0 * (x.x * x.x + x.y * x.y); }
    if (MODE == 1) {
        const double2 xr = a[g], xi = a[n_g + g];
        return g == 0 ? xr.x * xr.x + xi.x * xi.x : 2.0 * (xr.x * xr.x + xr.y * xr.y + xi.x * xi.x + xi.y * xi.y);
    }
    const double2 x = a[g];
    return x.x * x.x + x.y * x.y;
}

// r holds b on entry.  p = M r, rz = (r, M r), b2 = rr = ||r||^2, active = b2 > 0
template <int MODE>
__global__ void __launch_bounds__(NT) cg_init(long long n_g, int n_occ, const double* g2, const double* tk, int precond_on,
                                              const double2* R, double2* P, Scalars s, int* colmap) {
    __shared__ double sh[32];
    const int col = blockIdx.x, nvpc = MODE == 1 ? 2 : 1;
    if (threadIdx.x == 0) colmap[col] = col;
    const double2* r = R + (long long)col * nvpc * n_g;
    double2* p = P + (long long)col * nvpc * n_g;
    const double tkv = tk[col % n_occ];
    double acc[3] = {0, 0, 0};
    for (int g = threadIdx.x; g < n_g; g += NT) {
        const double m = precond(g2[g], tkv, precond_on);
        double d[2] = {0, 0};
        dot_accum<MODE>(r, r, n_g, g, m, d);
        acc[0] += d[0]; acc[1] += d[1];
        acc[2] += norm_accum<MODE>(r, n_g, g);
#pragma unroll
        for (int q = 0; q < nvpc; ++q) {
            const double2 x = r[q * n_g + g];
            p[q * n_g + g] = make_double2(m * x.x, m * x.y);
        }
    }
    block_reduce<3>(acc, sh);
    if (threadIdx.x == 0) {
        s.rz[col] = make_double2(acc[0], MODE == 1 ? acc[1] : 0.0);
        s.b2[col] = acc[2];
        s.rr[col] = acc[2];
        const int act = acc[2] > 0.0;
        s.active[col] = act;
        s.iters[col] = 0;
        if (act) atomicAdd(s.counters, 1);
    }
}

// One CG iteration's vector work for one column, fused (steps a8 + a9):
//   (p, Ap) -> a = rz / (p, Ap) ; x += a p ; r -= a Ap ; rznew = (r, M r), rr = ||r||^2 ; b = rznew / rz ; p = M r + b p
// One CTA per live column; the two reductions are CTA-wide, so no grid-wide dependency separates the three phases.  r, p,
// Ap are in compacted order (index k), x and the scalars in original column order (colmap[k]).  p and Ap are read twice and
// r is re-read after its update; the second touches hit L1/L2 (a column is 146 KB), so HBM sees 4 reads + 3 writes.
template <int MODE>
__global__ void __launch_bounds__(NT) cg_step(long long n_g, int n_occ, const double* g2, const double* tk, int precond_on, double tol2,
                                              double2* P, const double2* AP, double2* X, double2* R, Scalars s, const int* colmap) {
    __shared__ double sh[32];
    const int k = blockIdx.x, col = colmap[k], nvpc = MODE == 1 ? 2 : 1;
    if (col < 0 || !s.active[col]) return;       // col < 0: inert padding of a lagged compaction (cg_compact_map)
    const long long o = (long long)k * nvpc * n_g;
    double2* p = P + o; const double2* ap = AP + o;
    double2* x = X + (long long)col * nvpc * n_g; double2* r = R + o;
    const double tkv = tk[col % n_occ];
    // ---- (p, Ap)
    double d2[2] = {0, 0};
    for (int g = threadIdx.x; g < n_g; g += NT) dot_accum<MODE>(p, ap, n_g, g, 1.0, d2);
    block_reduce<2>(d2, sh);
    const double2 rz = s.rz[col];
    const double2 a = cdiv(rz, make_double2(d2[0], MODE == 1 ? d2[1] : 0.0));
    // ---- x, r, and the new inner products
    double acc[3] = {0, 0, 0};
    for (int g = threadIdx.x; g < n_g; g += NT) {
        const double m = precond(g2[g], tkv, precond_on);
        if (MODE == 1) {
            const double2 pr = p[g], pi = p[n_g + g], qr = ap[g], qi = ap[n_g + g];
            double2 xr = x[g], xi = x[n_g + g], rr = r[g], ri = r[n_g + g];
            xr.x += a.x * pr.x - a.y * pi.x; xr.y += a.x * pr.y - a.y * pi.y;
            xi.x += a.x * pi.x + a.y * pr.x; xi.y += a.x * pi.y + a.y * pr.y;
            rr.x -= a.x * qr.x - a.y * qi.x; rr.y -= a.x * qr.y - a.y * qi.y;
            ri.x -= a.x * qi.x + a.y * qr.x; ri.y -= a.x * qi.y + a.y * qr.y;
            x[g] = xr; x[n_g + g] = xi; r[g] = rr; r[n_g + g] = ri;
            const double f = g == 0 ? 1.0 : 2.0;
            const double srr = g == 0 ? rr.x * rr.x : rr.x * rr.x + rr.y * rr.y;
            const double sii = g == 0 ? ri.x * ri.x : ri.x * ri.x + ri.y * ri.y;
            const double sri = g == 0 ? rr.x * ri.x : rr.x * ri.x + rr.y * ri.y;
            acc[0] += f * (srr - sii) * m; acc[1] += f * (2.0 * sri) * m; acc[2] += f * (srr + sii);
        } else {
            const double2 pp = p[g], q = ap[g];
            double2 xx = x[g], rr = r[g];
            xx.x += a.x * pp.x; xx.y += a.x * pp.y;
            rr.x -= a.x * q.x;  rr.y -= a.x * q.y;
            x[g] = xx; r[g] = rr;
            const double n2 = (MODE == 0) ? (g == 0 ? rr.x * rr.x : 2.0 * (rr.x * rr.x + rr.y * rr.y)) : rr.x * rr.x + rr.y * rr.y;
            acc[0] += n2 * m; acc[2] += n2;
        }
    }
    block_reduce<3>(acc, sh);
    const double2 rznew = make_double2(acc[0], MODE == 1 ? acc[1] : 0.0);
    const bool still = acc[2] > tol2 * s.b2[col];
    // ---- p = M r + beta p (each thread re-reads the r elements it wrote itself)
    if (still) {
        const double2 beta = cdiv(rznew, rz);
        for (int g = threadIdx.x; g < n_g; g += NT) {
            const double m = precond(g2[g], tkv, precond_on);
            if (MODE == 1) {
                const double2 zr = r[g], zi = r[n_g + g], pr = p[g], pi = p[n_g + g];
                p[g] = make_double2(m * zr.x + beta.x * pr.x - beta.y * pi.x, m * zr.y + beta.x * pr.y - beta.y * pi.y);
                p[n_g + g] = make_double2(m * zi.x + beta.x * pi.x + beta.y * pr.x, m * zi.y + beta.x * pi.y + beta.y * pr.y);
            } else {
                const double2 z = r[g], pp = p[g];
                p[g] = make_double2(m * z.x + beta.x * pp.x, m * z.y + beta.x * pp.y);
            }
        }
    }
    if (threadIdx.x == 0) {
        s.rz[col] = rznew;
        s.rr[col] = acc[2];
        s.iters[col] += 1;
        if (!still) { s.active[col] = 0; atomicSub(s.counters, 1); }
    }
}

// The same iteration with the column RESIDENT on the SM (MODE 0 and 2, n_g <= EPT * NTR): cg_step's second touches of p, Ap and r
// were meant to hit L2, but 8 CTAs x 148 SMs x 4 vectors x 146 KB (cfg 2) is 690 MB of columns in flight against a 126 MB L2, so
// they came from HBM again (11 vector passes per iteration instead of 7).  Here one CTA of NTR threads owns a column, thread t
// owns elements g = e NTR + t: Ap, then the new r, stay in its registers and p in its own shared-memory slots (each thread reads
// back only what it wrote, so no barrier guards them), and HBM sees exactly 4 reads (p, Ap, x, r) and 3 writes (x, r, p).
// Measured at cfg 2: 44.3 -> 40.4 ms per step (1024 threads; 768 the same, 512 slower; an L2 prefetch of x and r during the first loop
// made it slower, 43.3 ms).  One column per SM is all that fits on chip, so the three phases of a CTA do not overlap with another CTA's.
template <int NV, int NWARP>
__device__ __forceinline__ void block_reduce_w(double (&v)[NV], double* sh /* [NV * NWARP] */) {
#pragma unroll
    for (int i = 0; i < NV; ++i)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[i] += __shfl_xor_sync(0xffffffffu, v[i], o);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0)
#pragma unroll
        for (int i = 0; i < NV; ++i) sh[i * NWARP + warp] = v[i];
    __syncthreads();
#pragma unroll
    for (int i = 0; i < NV; ++i) {
        double s = lane < NWARP ? sh[i * NWARP + lane] : 0.0;      // NWARP <= 32: every warp folds the partials itself
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        v[i] = s;
    }
    __syncthreads();
}

template <int MODE, int NTR, int EPT>
__global__ void __launch_bounds__(NTR, 1) cg_step_resident(long long n_g, int n_occ, const double* g2, const double* tk, int precond_on, double tol2,
                                                           double2* P, const double2* AP, double2* X, double2* R, Scalars s, const int* colmap) {
    static_assert(MODE == 0 || MODE == 2, "one vector per column");
    extern __shared__ __align__(16) double2 psh[];            // [EPT][NTR]: thread t owns psh[e * NTR + t]
    __shared__ double sh[3 * (NTR / 32)];
    const int k = blockIdx.x, col = colmap[k], t = threadIdx.x;
    if (col < 0 || !s.active[col]) return;
    const long long o = (long long)k * n_g;
    double2* p = P + o; const double2* ap = AP + o;
    double2* x = X + (long long)col * n_g; double2* r = R + o;
    const double tkv = tk[col % n_occ];
    // ---- (p, Ap): p to shared memory, Ap to registers
    double2 q[EPT];
    double d1[1] = {0};
#pragma unroll
    for (int e = 0; e < EPT; ++e) {
        const int g = e * NTR + t;
        if (g < n_g) {
            const double2 pp = p[g];
            q[e] = ap[g];
            psh[e * NTR + t] = pp;
            const double w = pp.x * q[e].x + pp.y * q[e].y;
            d1[0] += MODE == 0 ? (g == 0 ? pp.x * q[e].x : 2.0 * w) : w;
        }
    }
    block_reduce_w<1, NTR / 32>(d1, sh);
    const double2 rz = s.rz[col];
    const double a = rz.x / d1[0];
    // ---- x += a p ; r -= a Ap (kept in q) ; (r, M r), ||r||^2
    double acc[2] = {0, 0};
#pragma unroll
    for (int e = 0; e < EPT; ++e) {
        const int g = e * NTR + t;
        if (g < n_g) {
            const double2 pp = psh[e * NTR + t];
            double2 xx = x[g], rr = r[g];
            xx.x += a * pp.x; xx.y += a * pp.y;
            rr.x -= a * q[e].x; rr.y -= a * q[e].y;
            x[g] = xx; r[g] = rr; q[e] = rr;
            const double n2 = (MODE == 0) ? (g == 0 ? rr.x * rr.x : 2.0 * (rr.x * rr.x + rr.y * rr.y)) : rr.x * rr.x + rr.y * rr.y;
            acc[0] += n2 * precond(g2[g], tkv, precond_on); acc[1] += n2;
        }
    }
    block_reduce_w<2, NTR / 32>(acc, sh);
    const bool still = acc[1] > tol2 * s.b2[col];
    // ---- p = M r + beta p
    if (still) {
        const double beta = acc[0] / rz.x;
#pragma unroll
        for (int e = 0; e < EPT; ++e) {
            const int g = e * NTR + t;
            if (g < n_g) {
                const double m = precond(g2[g], tkv, precond_on);
                const double2 pp = psh[e * NTR + t];
                p[g] = make_double2(m * q[e].x + beta * pp.x, m * q[e].y + beta * pp.y);
            }
        }
    }
    if (t == 0) {
        s.rz[col] = make_double2(acc[0], 0.0);
        s.rr[col] = acc[1];
        s.iters[col] += 1;
        if (!still) { s.active[col] = 0; atomicSub(s.counters, 1); }
    }
}

// The resident iteration with the column split over a thread-block CLUSTER of CL CTAs (distributed shared memory carries the partial
// sums): a CTA holds 1 / CL of the column (p in shared memory, Ap / r in registers), so two CTAs of different columns share an SM and
// one's reduction latency and store drain overlap the other's loads.  Element g = (e CL + rank) NTR + t.
template <int MODE, int NTR, int EPT, int CL>
__global__ void __cluster_dims__(CL, 1, 1) __launch_bounds__(NTR, 2)
cg_step_cluster(long long n_g, int n_occ, const double* g2, const double* tk, int precond_on, double tol2, double2* P, const double2* AP,
                double2* X, double2* R, Scalars s, const int* colmap) {
    static_assert(MODE == 0 || MODE == 2, "one vector per column");
    namespace cgr = cooperative_groups;
    cgr::cluster_group cluster = cgr::this_cluster();
    extern __shared__ __align__(16) double2 psh[];            // [EPT][NTR]
    __shared__ double sh[3 * (NTR / 32)];
    __shared__ double part[3];                                // this CTA's partial sums: (p, Ap) | (r, M r), ||r||^2
    const int rank = (int)cluster.block_rank();
    const int k = blockIdx.x / CL, col = colmap[k], t = threadIdx.x;
    if (col < 0 || !s.active[col]) return;                    // the whole cluster reads the same flag; it changes only at the very end
    const long long o = (long long)k * n_g;
    double2* p = P + o; const double2* ap = AP + o;
    double2* x = X + (long long)col * n_g; double2* r = R + o;
    const double tkv = tk[col % n_occ];
    double2 q[EPT];
    double d1[1] = {0};
#pragma unroll
    for (int e = 0; e < EPT; ++e) {
        const int g = (e * CL + rank) * NTR + t;
        if (g < n_g) {
            const double2 pp = p[g];
            q[e] = ap[g];
            psh[e * NTR + t] = pp;
            const double w = pp.x * q[e].x + pp.y * q[e].y;
            d1[0] += MODE == 0 ? (g == 0 ? pp.x * q[e].x : 2.0 * w) : w;
        }
    }
    block_reduce_w<1, NTR / 32>(d1, sh);
    if (t == 0) part[0] = d1[0];
    cluster.sync();
    double pap = 0;
#pragma unroll
    for (int c = 0; c < CL; ++c) pap += *cluster.map_shared_rank(&part[0], c);
    const double2 rz = s.rz[col];
    const double a = rz.x / pap;
    double acc[2] = {0, 0};
#pragma unroll
    for (int e = 0; e < EPT; ++e) {
        const int g = (e * CL + rank) * NTR + t;
        if (g < n_g) {
            const double2 pp = psh[e * NTR + t];
            double2 xx = x[g], rr = r[g];
            xx.x += a * pp.x; xx.y += a * pp.y;
            rr.x -= a * q[e].x; rr.y -= a * q[e].y;
            x[g] = xx; r[g] = rr; q[e] = rr;
            const double n2 = (MODE == 0) ? (g == 0 ? rr.x * rr.x : 2.0 * (rr.x * rr.x + rr.y * rr.y)) : rr.x * rr.x + rr.y * rr.y;
            acc[0] += n2 * precond(g2[g], tkv, precond_on); acc[1] += n2;
        }
    }
    block_reduce_w<2, NTR / 32>(acc, sh);
    if (t == 0) { part[1] = acc[0]; part[2] = acc[1]; }
    cluster.sync();
    double rzn = 0, rrn = 0;
#pragma unroll
    for (int c = 0; c < CL; ++c) {
        const double* pc = cluster.map_shared_rank(&part[0], c);
        rzn += pc[1]; rrn += pc[2];
    }
    const bool still = rrn > tol2 * s.b2[col];
    if (still) {
        const double beta = rzn / rz.x;
#pragma unroll
        for (int e = 0; e < EPT; ++e) {
            const int g = (e * CL + rank) * NTR + t;
            if (g < n_g) {
                const double m = precond(g2[g], tkv, precond_on);
                const double2 pp = psh[e * NTR + t];
                p[g] = make_double2(m * q[e].x + beta * pp.x, m * q[e].y + beta * pp.y);
            }
        }
    }
    cluster.sync();                                           // no CTA leaves while a partner may still read its partial sums
    if (rank == 0 && t == 0) {
        s.rz[col] = make_double2(rzn, 0.0);
        s.rr[col] = rrn;
        s.iters[col] += 1;
        if (!still) { s.active[col] = 0; atomicSub(s.counters, 1); }
    }
}

// ------------------------------------------------------------------------------------------------- multi-shift CG
// All imaginary frequencies from ONE Krylov sequence (Frommer's shifted CG): the seed system is the
// real symmetric A = H - eps_v + alpha P_v (WEST_GAMMA, unpreconditioned), the shifted systems are (A + sigma_s) x_s = b with
// sigma_s = -i omega_s.  Shifted residuals stay collinear with the seed residual, r_s = zeta_s r, so one H*psi per iteration
// serves every frequency:
//   zeta_{k+1} = zeta_k zeta_{k-1} a_{k-1} / [ a_k b_{k-1} (zeta_{k-1} - zeta_k) + zeta_{k-1} a_{k-1} (1 + sigma a_k) ]
//   a_s = a_k zeta_{k+1} / zeta_k ;  b_s = b_k (zeta_{k+1} / zeta_k)^2 ;  x_s += a_s p_s ;  p_s = zeta_{k+1} r_{k+1} + b_s p_s
// Vectors: r, p, Ap real functions in compacted order; XS, PS [shift][col][2][n_g] (Re and Im part as two real functions)
// in original column order.
constexpr int MS_MAX_SHIFTS = 16;

struct MsState {
    double*  a_prev;     // [n_col]
    double*  b_prev;     // [n_col]
    double*  rr;         // [n_col] <r_k, r_k>
    double*  b2;         // [n_col] <b, b>
    double2* zeta;       // [n_shift][n_col]
    double2* zeta_prev;  // [n_shift][n_col]
    double*  res2;       // [n_shift][n_col] |zeta|^2 rr / b2 at the moment the shift was frozen (or now)
    int*     active;     // [n_col]
    int*     iters;      // [n_col] iterations this column took part in
    int*     sactive;    // [n_shift][n_col]
    int*     counters;   // [0] live columns; [2..3] one 64-bit count of (column, shift) vector updates
};
struct MsShifts { int n; double omega[MS_MAX_SHIFTS]; };

__device__ __forceinline__ double rdot_gamma(const double2 x, const double2 y, int g) {
    return g == 0 ? x.x * y.x : 2.0 * (x.x * y.x + x.y * y.y);
}

// r holds b.  p = r, x_s = 0 (memset by the host), p_s = (b, 0)
__global__ void __launch_bounds__(NT) ms_init(long long n_g, int n_col, MsShifts sh, const double2* R, double2* P, double2* PS, MsState st,
                                              int* colmap) {
    __shared__ double red[32];
    const int col = blockIdx.x;
    const double2* r = R + (long long)col * n_g;
    double2* p = P + (long long)col * n_g;
    double acc[1] = {0};
    for (int g = threadIdx.x; g < n_g; g += NT) {
        const double2 v = r[g];
        acc[0] += rdot_gamma(v, v, g);
        p[g] = v;
        if (PS)                                   // PS == nullptr: Krylov-history variant (ms_hist_step), no per-shift search directions
            for (int s = 0; s < sh.n; ++s) {
                double2* ps = PS + ((long long)s * n_col + col) * 2 * n_g;
                ps[g] = v;
                ps[n_g + g] = make_double2(0.0, 0.0);
            }
    }
    block_reduce<1>(acc, red);
    if (threadIdx.x == 0) {
        colmap[col] = col;
        st.rr[col] = acc[0]; st.b2[col] = acc[0]; st.a_prev[col] = 1.0; st.b_prev[col] = 0.0;
        const int act = acc[0] > 0.0;
        st.active[col] = act;
        st.iters[col] = 0;
        if (act) atomicAdd(st.counters, 1);
        for (int s = 0; s < sh.n; ++s) {
            const long long i = (long long)s * n_col + col;
            st.zeta[i] = make_double2(1.0, 0.0); st.zeta_prev[i] = make_double2(1.0, 0.0);
            st.sactive[i] = act; st.res2[i] = act ? 1.0 : 0.0;
        }
    }
}

__global__ void __launch_bounds__(NT) ms_step(long long n_g, int n_col, MsShifts sh, double tol2, int want_imag, double2* P, const double2* AP,
                                              double2* R, double2* XS, double2* PS, MsState st, const int* colmap) {
    __shared__ double red[32];
    __shared__ double2 s_zn[MS_MAX_SHIFTS], s_as[MS_MAX_SHIFTS], s_bs[MS_MAX_SHIFTS];
    __shared__ int s_on[MS_MAX_SHIFTS];
    const int k = blockIdx.x, col = colmap[k];
    if (col < 0 || !st.active[col]) return;
    double2* p = P + (long long)k * n_g; const double2* ap = AP + (long long)k * n_g; double2* r = R + (long long)k * n_g;
    // ---- a_k
    double acc[1] = {0};
    for (int g = threadIdx.x; g < n_g; g += NT) acc[0] += rdot_gamma(p[g], ap[g], g);
    block_reduce<1>(acc, red);
    const double rr = st.rr[col], a = rr / acc[0];
    // ---- r_{k+1}, b_k
    acc[0] = 0;
    for (int g = threadIdx.x; g < n_g; g += NT) {
        double2 v = r[g]; const double2 q = ap[g];
        v.x -= a * q.x; v.y -= a * q.y;
        r[g] = v;
        acc[0] += rdot_gamma(v, v, g);
    }
    block_reduce<1>(acc, red);
    const double rrn = acc[0], b = rrn / rr;
    // ---- shifted scalars
    if (threadIdx.x < sh.n) {
        const int s = threadIdx.x;
        const long long i = (long long)s * n_col + col;
        int on = st.sactive[i];
        if (on) {
            const double2 z = st.zeta[i], zp = st.zeta_prev[i];
            const double ap_ = st.a_prev[col], bp_ = st.b_prev[col];
            const double2 sigma = make_double2(0.0, -sh.omega[s]);
            // den = a b_{k-1} (zp - z) + zp a_{k-1} (1 + sigma a)
            const double2 t1 = make_double2(a * bp_ * (zp.x - z.x), a * bp_ * (zp.y - z.y));
            const double2 one_sa = make_double2(1.0 + sigma.x * a, sigma.y * a);
            const double2 t2 = cmul2(make_double2(zp.x * ap_, zp.y * ap_), one_sa);
            const double2 num = cmul2(z, make_double2(zp.x * ap_, zp.y * ap_));
            const double2 zn = cdiv(num, make_double2(t1.x + t2.x, t1.y + t2.y));
            const double2 ratio = cdiv(zn, z);
            s_zn[s] = zn;
            s_as[s] = make_double2(a * ratio.x, a * ratio.y);
            const double2 r2 = cmul2(ratio, ratio);
            s_bs[s] = make_double2(b * r2.x, b * r2.y);
            st.zeta_prev[i] = z; st.zeta[i] = zn;
            const double res2 = (zn.x * zn.x + zn.y * zn.y) * rrn / st.b2[col];
            st.res2[i] = res2;
            if (!(res2 > tol2)) st.sactive[i] = 0;       // x_s still takes this iteration's update below, then freezes
        }
        s_on[s] = on;
    }
    __syncthreads();
    // ---- vector updates
    for (int g = threadIdx.x; g < n_g; g += NT) {
        const double2 rn = r[g];
        for (int s = 0; s < sh.n; ++s) {
            if (!s_on[s]) continue;
            double2* xs = XS + ((long long)s * n_col + col) * 2 * n_g;
            double2* ps = PS + ((long long)s * n_col + col) * 2 * n_g;
            const double2 as = s_as[s], bs = s_bs[s], zn = s_zn[s];
            const double2 pr = ps[g], pi = ps[n_g + g];
            double2 xr = xs[g];
            xr.x += as.x * pr.x - as.y * pi.x; xr.y += as.x * pr.y - as.y * pi.y;
            xs[g] = xr;
            if (want_imag) {        // Im x_s is only needed when the caller asked for dpsi: dn uses Re x_s alone (real orbitals)
                double2 xi = xs[n_g + g];
                xi.x += as.x * pi.x + as.y * pr.x; xi.y += as.x * pi.y + as.y * pr.y;
                xs[n_g + g] = xi;
            }
            ps[g] = make_double2(zn.x * rn.x + bs.x * pr.x - bs.y * pi.x, zn.x * rn.y + bs.x * pr.y - bs.y * pi.y);
            ps[n_g + g] = make_double2(zn.y * rn.x + bs.x * pi.x + bs.y * pr.x, zn.y * rn.y + bs.x * pi.y + bs.y * pr.y);
        }
        const double2 pp = p[g];
        p[g] = make_double2(rn.x + b * pp.x, rn.y + b * pp.y);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        st.a_prev[col] = a; st.b_prev[col] = b; st.rr[col] = rrn;
        st.iters[col] += 1;
        int n_on = 0;
        for (int s = 0; s < sh.n; ++s) n_on += s_on[s];
        atomicAdd(reinterpret_cast<unsigned long long*>(st.counters + 2), (unsigned long long)n_on);     // (column, shift) updates done: the byte model of the bench
        int any = 0;
        for (int s = 0; s < sh.n; ++s) any |= st.sactive[(long long)s * n_col + col];
        if (!any) { st.active[col] = 0; atomicSub(st.counters, 1); }
    }
}

// ---------------------------------------------------------------------------------------------- multi-shift CG with a Krylov history
// The per-shift vector recurrences of ms_step move 6 vector passes per live shift and iteration.  They are linear in the seed
// residuals: with  p_s,k = zeta_k r_k + Q_k,  Q_{k+1} = b_s,k p_s,k,  x_s += a_s,k p_s,k  (a_s,k, b_s,k, zeta_k as in ms_step) the
// iterations k = j0 .. n-1 of a segment add
//     x_s += sum_j zeta_j w_j r_j + w_j0 Q_j0,        w_j = a_s,j + b_s,j w_{j+1},  w_n = 0
//     Q_n  = sum_j zeta_j B_j r_j + B_j0 Q_j0,         B_j = b_s,j B_{j+1},          B_n = 1
// so it is enough to KEEP the residuals r_j (they are written anyway: the seed recurrence writes r_{k+1} into the next slot of a ring
// instead of over r_k), store three complex scalars per (iteration, shift, column), and contract once per segment (ms_hist_combine):
// every history vector is read once for ALL shifts.  This is the Lanczos form of the shifted solves (PAPER.md:138-157 uses the same
// idea for its frequency dependence); results equal ms_step's up to summation order.
// Ring: r_j lives in slot j mod H of HIST [H][n_col][n_g] (original column order), the scalars of iteration k in slot k mod H of
// HS [H][3][n_shift][n_col] (a_s, b_s, zeta_k; zero once the shift is frozen).  A segment ends (flush) before slot j0 would be overwritten.
struct MsHist {
    double2* vec;      // [H][n_col][n_g]
    double2* scal;     // [H][3][n_shift][n_col]
    int H;
};

__global__ void __launch_bounds__(NT) ms_hist_step(long long n_g, int n_col, MsShifts sh, double tol2, int k_iter, MsHist hs, double2* P,
                                                   const double2* AP, MsState st, const int* colmap) {
    __shared__ double red[32];
    const int k = blockIdx.x, col = colmap[k];
    if (col < 0 || !st.active[col]) return;
    double2* p = P + (long long)k * n_g; const double2* ap = AP + (long long)k * n_g;
    const double2* r = hs.vec + ((long long)(k_iter % hs.H) * n_col + col) * n_g;
    double2* rnew = hs.vec + ((long long)((k_iter + 1) % hs.H) * n_col + col) * n_g;
    // ---- a_k
    double acc[1] = {0};
    for (int g = threadIdx.x; g < n_g; g += NT) acc[0] += rdot_gamma(p[g], ap[g], g);
    block_reduce<1>(acc, red);
    const double rr = st.rr[col], a = rr / acc[0];
    // ---- r_{k+1} (next ring slot), b_k
    acc[0] = 0;
    for (int g = threadIdx.x; g < n_g; g += NT) {
        double2 v = r[g]; const double2 q = ap[g];
        v.x -= a * q.x; v.y -= a * q.y;
        rnew[g] = v;
        acc[0] += rdot_gamma(v, v, g);
    }
    block_reduce<1>(acc, red);
    const double rrn = acc[0], b = rrn / rr;
    // ---- shifted scalars (same recurrences as ms_step), kept for the segment's contraction
    if (threadIdx.x < sh.n) {
        const int s = threadIdx.x;
        const long long i = (long long)s * n_col + col;
        double2* slot = hs.scal + (long long)(k_iter % hs.H) * 3 * sh.n * n_col;
        double2 as = make_double2(0.0, 0.0), bs = as, zc = as;
        if (st.sactive[i]) {
            const double2 z = st.zeta[i], zp = st.zeta_prev[i];
            const double ap_ = st.a_prev[col], bp_ = st.b_prev[col];
            const double2 sigma = make_double2(0.0, -sh.omega[s]);
            const double2 t1 = make_double2(a * bp_ * (zp.x - z.x), a * bp_ * (zp.y - z.y));
            const double2 one_sa = make_double2(1.0 + sigma.x * a, sigma.y * a);
            const double2 t2 = cmul2(make_double2(zp.x * ap_, zp.y * ap_), one_sa);
            const double2 num = cmul2(z, make_double2(zp.x * ap_, zp.y * ap_));
            const double2 zn = cdiv(num, make_double2(t1.x + t2.x, t1.y + t2.y));
            const double2 ratio = cdiv(zn, z);
            as = make_double2(a * ratio.x, a * ratio.y);
            const double2 r2 = cmul2(ratio, ratio);
            bs = make_double2(b * r2.x, b * r2.y);
            zc = z;
            st.zeta_prev[i] = z; st.zeta[i] = zn;
            const double res2 = (zn.x * zn.x + zn.y * zn.y) * rrn / st.b2[col];
            st.res2[i] = res2;
            if (!(res2 > tol2)) st.sactive[i] = 0;       // x_s still takes this iteration's update (as is stored), then freezes
        }
        slot[i] = as; slot[(long long)sh.n * n_col + i] = bs; slot[2ll * sh.n * n_col + i] = zc;
    }
    // ---- p = r_{k+1} + b p
    for (int g = threadIdx.x; g < n_g; g += NT) {
        const double2 rn = rnew[g], pp = p[g];
        p[g] = make_double2(rn.x + b * pp.x, rn.y + b * pp.y);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        st.a_prev[col] = a; st.b_prev[col] = b; st.rr[col] = rrn;
        st.iters[col] += 1;
        int any = 0;
        for (int s = 0; s < sh.n; ++s) any |= st.sactive[(long long)s * n_col + col];
        if (!any) { st.active[col] = 0; atomicSub(st.counters, 1); }
    }
}

// The same iteration with the column resident on one SM (n_g <= NTR * EPT; cfgs 1-4): p parked in shared memory, Ap and then r_{k+1} in
// registers, so HBM sees 3 reads (p, Ap, r_k) and 2 writes (r_{k+1}, p) of the column instead of the 8 passes of the streaming kernel.
__device__ __forceinline__ void ms_shift_scalars(const MsShifts& sh, int n_col, int col, int k_iter, const MsHist& hs, MsState& st, double a, double b,
                                                 double rrn, double tol2) {
    if (threadIdx.x < sh.n) {
        const int s = threadIdx.x;
        const long long i = (long long)s * n_col + col;
        double2* slot = hs.scal + (long long)(k_iter % hs.H) * 3 * sh.n * n_col;
        double2 as = make_double2(0.0, 0.0), bs = as, zc = as;
        if (st.sactive[i]) {
            const double2 z = st.zeta[i], zp = st.zeta_prev[i];
            const double ap_ = st.a_prev[col], bp_ = st.b_prev[col];
            const double2 sigma = make_double2(0.0, -sh.omega[s]);
            const double2 t1 = make_double2(a * bp_ * (zp.x - z.x), a * bp_ * (zp.y - z.y));
            const double2 one_sa = make_double2(1.0 + sigma.x * a, sigma.y * a);
            const double2 t2 = cmul2(make_double2(zp.x * ap_, zp.y * ap_), one_sa);
            const double2 num = cmul2(z, make_double2(zp.x * ap_, zp.y * ap_));
            const double2 zn = cdiv(num, make_double2(t1.x + t2.x, t1.y + t2.y));
            const double2 ratio = cdiv(zn, z);
            as = make_double2(a * ratio.x, a * ratio.y);
            const double2 r2 = cmul2(ratio, ratio);
            bs = make_double2(b * r2.x, b * r2.y);
            zc = z;
            st.zeta_prev[i] = z; st.zeta[i] = zn;
            const double res2 = (zn.x * zn.x + zn.y * zn.y) * rrn / st.b2[col];
            st.res2[i] = res2;
            if (!(res2 > tol2)) st.sactive[i] = 0;       // x_s still takes this iteration's update (as is stored), then freezes
        }
        slot[i] = as; slot[(long long)sh.n * n_col + i] = bs; slot[2ll * sh.n * n_col + i] = zc;
    }
}
template <int NTR, int EPT>
__global__ void __launch_bounds__(NTR, 1) ms_hist_step_resident(long long n_g, int n_col, MsShifts sh, double tol2, int k_iter, MsHist hs, double2* P,
                                                                const double2* AP, MsState st, const int* colmap) {
    extern __shared__ __align__(16) double2 psh[];            // [EPT][NTR]: thread t owns psh[e * NTR + t]
    __shared__ double shr[NTR / 32];
    const int k = blockIdx.x, col = colmap[k], t = threadIdx.x;
    if (col < 0 || !st.active[col]) return;
    double2* p = P + (long long)k * n_g; const double2* ap = AP + (long long)k * n_g;
    const double2* r = hs.vec + ((long long)(k_iter % hs.H) * n_col + col) * n_g;
    double2* rnew = hs.vec + ((long long)((k_iter + 1) % hs.H) * n_col + col) * n_g;
    double2 q[EPT];
    double d1[1] = {0};
#pragma unroll
    for (int e = 0; e < EPT; ++e) {
        const int g = e * NTR + t;
        if (g < n_g) {
            const double2 pp = p[g];
            q[e] = ap[g];
            psh[e * NTR + t] = pp;
            d1[0] += rdot_gamma(pp, q[e], g);
        }
    }
    block_reduce_w<1, NTR / 32>(d1, shr);
    const double rr = st.rr[col], a = rr / d1[0];
    double acc[1] = {0};
#pragma unroll
    for (int e = 0; e < EPT; ++e) {
        const int g = e * NTR + t;
        if (g < n_g) {
            double2 v = r[g];
            v.x -= a * q[e].x; v.y -= a * q[e].y;
            rnew[g] = v; q[e] = v;
            acc[0] += rdot_gamma(v, v, g);
        }
    }
    block_reduce_w<1, NTR / 32>(acc, shr);
    const double rrn = acc[0], b = rrn / rr;
#pragma unroll
    for (int e = 0; e < EPT; ++e) {
        const int g = e * NTR + t;
        if (g < n_g) {
            const double2 pp = psh[e * NTR + t];
            p[g] = make_double2(q[e].x + b * pp.x, q[e].y + b * pp.y);
        }
    }
    ms_shift_scalars(sh, n_col, col, k_iter, hs, st, a, b, rrn, tol2);      // after the vector work: the column's registers are dead by now
    __syncthreads();
    if (t == 0) {
        st.a_prev[col] = a; st.b_prev[col] = b; st.rr[col] = rrn;
        st.iters[col] += 1;
        int any = 0;
        for (int s = 0; s < sh.n; ++s) any |= st.sactive[(long long)s * n_col + col];
        if (!any) { st.active[col] = 0; atomicSub(st.counters, 1); }
    }
}

// Contraction of one segment [j0, n) of the history for column blockIdx.x, elements [blockIdx.y * MSH_CHUNK, +MSH_CHUNK):
//   XS[s][col] (Re part, and Im part if IMAG) += sum_j cx_j r_j + dx Q_s          QS[s][col] = sum_j cq_j r_j + dq Q_s   (CARRY_OUT)
// carry_in = 0: Q_s is taken as zero (first segment) and never read.  Columns use only the iterations they took part in
// (j < iters[col]); a column that left before j0 has nothing to add.  Carry vectors are formed only for the shifts that are still
// live at the end of the segment (B_j0 != 0: a shift that froze inside it never reads its Q again), so a flush needs the x accumulators of
// XG shifts and the carry accumulators of at most MSH_QG live shifts per pass over the history: one pass for up to 8 frequencies unless
// more than four of a column's shifts are still live (then further carry-only passes).  Q of a dead shift is never written NOR read.
// Dynamic shared memory: 2 * n_shift * (n - j0 + 1) double2.
constexpr int MSH_CHUNK = 2048;
constexpr int MSH_HMAX = 128;        // most ring slots (bounds the coefficient tables: 2 * 16 shifts * 129 double2 = 66 KB)
constexpr int MSH_QG = 4;            // carry accumulators (live shifts) per pass
// XG = shifts whose x accumulators a pass holds: 8 for Re x_s only, 4 when Im x_s is wanted too (dpsi requested)
template <bool IMAG, bool CARRY_OUT, int XG>
__global__ void __launch_bounds__(NT) ms_hist_combine(long long n_g, int n_col, int n_shift, int j0, int n_end, int carry_in, MsHist hs,
                                                      const int* iters, double2* XS, double2* QS, unsigned long long* pass_counter) {
    extern __shared__ double2 msh_sm[];
    __shared__ int s_qlist[MS_MAX_SHIFTS], s_nq, s_xin[MS_MAX_SHIFTS];
    const int col = blockIdx.x;
    const int jend = min(n_end, iters[col]);
    const int len = jend - j0;
    if (len <= 0) return;
    const int L = n_end - j0 + 1;                       // row length of the coefficient tables (last entry: the carry coefficients dx, dq)
    double2* cx = msh_sm;                               // [n_shift][L]
    double2* cq = msh_sm + (size_t)n_shift * L;         // [n_shift][L]
    // stage the segment's scalars: cx <- a_s, cq <- b_s, then the backward recurrences in place (zeta read from global, L2-resident)
    for (int t = threadIdx.x; t < n_shift * len; t += NT) {
        const int s = t / len, i = t - s * len;
        const double2* slot = hs.scal + (long long)((j0 + i) % hs.H) * 3 * n_shift * n_col + (long long)s * n_col + col;
        cx[s * L + i] = slot[0];
        cq[s * L + i] = slot[(long long)n_shift * n_col];
    }
    __syncthreads();
    if (threadIdx.x < n_shift) {
        const int s = threadIdx.x;
        double2 w = make_double2(0.0, 0.0), bt = make_double2(1.0, 0.0);
        for (int i = len - 1; i >= 0; --i) {
            const double2 as = cx[s * L + i], bs = cq[s * L + i];
            const double2 zc = hs.scal[(long long)((j0 + i) % hs.H) * 3 * n_shift * n_col + 2ll * n_shift * n_col + (long long)s * n_col + col];
            const double2 bw = cmul2(bs, w);
            w = make_double2(as.x + bw.x, as.y + bw.y);
            bt = cmul2(bs, bt);
            cx[s * L + i] = cmul2(zc, w);
            cq[s * L + i] = cmul2(zc, bt);
        }
        cx[s * L + L - 1] = w;                          // dx
        cq[s * L + L - 1] = bt;                         // dq
        s_xin[s] = carry_in && (w.x != 0.0 || w.y != 0.0);                                        // x_s takes a contribution of the old carry
        s_qlist[s] = (CARRY_OUT && jend == n_end && (bt.x != 0.0 || bt.y != 0.0)) ? 1 : 0;        // live at the end of the segment (flag, compacted below)
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int nq = 0, nxin = 0;
        for (int s = 0; s < n_shift; ++s) { const int live = s_qlist[s]; nxin += s_xin[s] || (live && carry_in); if (live) s_qlist[nq++] = s; }
        s_nq = nq;
        if (blockIdx.y == 0 && pass_counter) {
            // column-vector passes (16 n_g bytes each) of this column's contraction: one history read per pass, x_s traffic, carry reads / writes
            const int nxp = (n_shift + XG - 1) / XG, nqp = (nq + MSH_QG - 1) / MSH_QG;
            const int P = nxp - 1 + max(1, nqp);
            atomicAdd(pass_counter, (unsigned long long)len * P + (unsigned long long)n_shift * (IMAG ? 4 : 2) + 2ull * nxin + 2ull * nq);
        }
    }
    __syncthreads();
    const int nq = s_nq;
    const int nxp = (n_shift + XG - 1) / XG, nqp = (nq + MSH_QG - 1) / MSH_QG;
    const int n_pass = nxp - 1 + max(1, nqp);           // the last x pass also takes the first carry group
    const long long g_lo = (long long)blockIdx.y * MSH_CHUNK, g_hi = min(n_g, g_lo + MSH_CHUNK);
    for (int pass = 0; pass < n_pass; ++pass) {
        const int s0 = pass * XG, nx = pass < nxp ? min(XG, n_shift - s0) : 0;
        const int qg = pass - (nxp - 1), q0 = qg * MSH_QG, nqs = (CARRY_OUT && qg >= 0) ? max(0, min(MSH_QG, nq - q0)) : 0;
        int qoff[MSH_QG];                                // coefficient rows of this pass's live shifts
#pragma unroll
        for (int q = 0; q < MSH_QG; ++q) qoff[q] = (CARRY_OUT && q < nqs) ? s_qlist[q0 + q] : 0;
        for (long long g = g_lo + threadIdx.x; g < g_hi; g += NT) {
            double2 xr[XG], xi[IMAG ? XG : 1], qr[CARRY_OUT ? MSH_QG : 1], qi[CARRY_OUT ? MSH_QG : 1];
#pragma unroll
            for (int q = 0; q < XG; ++q) { xr[q] = make_double2(0.0, 0.0); if (IMAG) xi[q] = make_double2(0.0, 0.0); }
            if (CARRY_OUT) {
#pragma unroll
                for (int q = 0; q < MSH_QG; ++q) qr[q] = qi[q] = make_double2(0.0, 0.0);
            }
            const double2* hv = hs.vec + (long long)col * n_g + g;
#pragma unroll 4
            for (int i = 0; i < len; ++i) {
                const double2 v = hv[(long long)((j0 + i) % hs.H) * n_col * n_g];
#pragma unroll
                for (int q = 0; q < XG; ++q) {
                    if (q < nx) {
                        const double2 c1 = cx[(s0 + q) * L + i];
                        xr[q].x += c1.x * v.x; xr[q].y += c1.x * v.y;
                        if (IMAG) { xi[q].x += c1.y * v.x; xi[q].y += c1.y * v.y; }
                    }
                }
                if (CARRY_OUT) {
#pragma unroll
                    for (int q = 0; q < MSH_QG; ++q) {
                        if (q < nqs) {
                            const double2 c2 = cq[qoff[q] * L + i];
                            qr[q].x += c2.x * v.x; qr[q].y += c2.x * v.y;
                            qi[q].x += c2.y * v.x; qi[q].y += c2.y * v.y;
                        }
                    }
                }
            }
#pragma unroll
            for (int q = 0; q < XG; ++q) {
                if (q < nx) {
                    const int s = s0 + q;
                    const long long base = ((long long)s * n_col + col) * 2 * n_g + g;
                    if (s_xin[s]) {
                        const double2 Qr = QS[base], Qi = QS[base + n_g];
                        const double2 dx = cx[s * L + L - 1];
                        xr[q].x += dx.x * Qr.x - dx.y * Qi.x; xr[q].y += dx.x * Qr.y - dx.y * Qi.y;
                        if (IMAG) { xi[q].x += dx.x * Qi.x + dx.y * Qr.x; xi[q].y += dx.x * Qi.y + dx.y * Qr.y; }
                    }
                    double2 x0 = XS[base];
                    x0.x += xr[q].x; x0.y += xr[q].y;
                    XS[base] = x0;
                    if (IMAG) {
                        double2 x1 = XS[base + n_g];
                        x1.x += xi[q].x; x1.y += xi[q].y;
                        XS[base + n_g] = x1;
                    }
                }
            }
            if (CARRY_OUT) {
                // (the x update of a live shift read its old carry above, in this pass or an earlier one: carry groups never run before the
                // x pass of their shifts)
#pragma unroll
                for (int q = 0; q < MSH_QG; ++q) {
                    if (q < nqs) {
                        const int s = qoff[q];
                        const long long base = ((long long)s * n_col + col) * 2 * n_g + g;
                        if (carry_in) {
                            const double2 Qr = QS[base], Qi = QS[base + n_g];
                            const double2 dq = cq[s * L + L - 1];
                            qr[q].x += dq.x * Qr.x - dq.y * Qi.x; qr[q].y += dq.x * Qr.y - dq.y * Qi.y;
                            qi[q].x += dq.x * Qi.x + dq.y * Qr.x; qi[q].y += dq.x * Qi.y + dq.y * Qr.y;
                        }
                        QS[base] = qr[q]; QS[base + n_g] = qi[q];
                    }
                }
            }
        }
    }
}

// block-wide min / max / sum helpers of the final reports (one CTA of NT threads)
__device__ __forceinline__ void report_reduce(double m, int c, int lo, int hi, double* out) {
    __shared__ double shm[NT]; __shared__ int shc[NT], shlo[NT], shhi[NT];
    shm[threadIdx.x] = m; shc[threadIdx.x] = c; shlo[threadIdx.x] = lo; shhi[threadIdx.x] = hi;
    __syncthreads();
    for (int o = NT / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) {
            shm[threadIdx.x] = fmax(shm[threadIdx.x], shm[threadIdx.x + o]); shc[threadIdx.x] += shc[threadIdx.x + o];
            shlo[threadIdx.x] = min(shlo[threadIdx.x], shlo[threadIdx.x + o]); shhi[threadIdx.x] = max(shhi[threadIdx.x], shhi[threadIdx.x + o]);
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) { out[0] = sqrt(shm[0]); out[1] = (double)shc[0]; out[2] = (double)(shlo[0] == 0x7fffffff ? 0 : shlo[0]); out[3] = (double)shhi[0]; }
}
// final report, out[4]: max relative residual, number of unconverged (column[, shift]) pairs, min and max over the non-zero columns of
// the iterations a column took part in
__global__ void ms_report(int n_col, int n_shift, double tol2, MsState st, double* out) {
    double m = 0; int c = 0, lo = 0x7fffffff, hi = 0;
    for (long long i = threadIdx.x; i < (long long)n_col * n_shift; i += NT) {
        const double q = st.res2[i];
        m = fmax(m, q); c += q > tol2;
    }
    for (int i = threadIdx.x; i < n_col; i += NT)
        if (st.b2[i] > 0) { lo = min(lo, st.iters[i]); hi = max(hi, st.iters[i]); }
    report_reduce(m, c, lo, hi, out);
}
__global__ void cg_report(int n_col, double tol2, Scalars s, double* out) {
    double m = 0; int c = 0, lo = 0x7fffffff, hi = 0;
    for (int i = threadIdx.x; i < n_col; i += NT) {
        const double b2 = s.b2[i];
        if (b2 > 0) { const double q = s.rr[i] / b2; m = fmax(m, q); c += q > tol2; lo = min(lo, s.iters[i]); hi = max(hi, s.iters[i]); }
    }
    report_reduce(m, c, lo, hi, out);
}

// Compaction of the active columns (order preserving).  One CTA: new_map[j] = original column of the j-th still-active
// entry of old_map[0..n_old), src[j] = its old compacted position.  The host asks for n_new columns, the count it read one
// iteration ago (lagged poll); columns that converged since leave fewer, and the rest is padded with inert entries
// (new_map = -1: skipped by the vector kernels; src = 0: a copy of finite data for the FFT / GEMM batches).
__global__ void __launch_bounds__(1024) cg_compact_map(int n_old, const int* old_map, const int* active, int* new_map, int* src, int n_new) {
    __shared__ int warp_sums[32];
    __shared__ int base;
    if (threadIdx.x == 0) base = 0;
    __syncthreads();
    for (int start = 0; start < n_old; start += 1024) {
        const int i = start + threadIdx.x;
        const int col = i < n_old ? old_map[i] : -1;
        const int flag = (col >= 0 && active[col]) ? 1 : 0;
        int v = flag;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { int t = __shfl_up_sync(0xffffffffu, v, o); if ((threadIdx.x & 31) >= o) v += t; }
        if ((threadIdx.x & 31) == 31) warp_sums[threadIdx.x >> 5] = v;
        __syncthreads();
        if (threadIdx.x < 32) {
            int w = warp_sums[threadIdx.x];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { int t = __shfl_up_sync(0xffffffffu, w, o); if (threadIdx.x >= o) w += t; }
            warp_sums[threadIdx.x] = w;
        }
        __syncthreads();
        const int before = base + v - flag + ((threadIdx.x >> 5) ? warp_sums[(threadIdx.x >> 5) - 1] : 0);
        if (flag && before < n_new) { new_map[before] = col; src[before] = i; }
        __syncthreads();
        if (threadIdx.x == 0) base += warp_sums[31];
        __syncthreads();
    }
    for (int j = base + threadIdx.x; j < n_new; j += 1024) { new_map[j] = -1; src[j] = 0; }
}
// dst[j] = src_vec[src[j]] for whole columns (nvpc * n_g complex each)
__global__ void __launch_bounds__(NT) cg_gather_cols(long long len, const int* src, const double2* in, double2* out) {
    const double2* a = in + (long long)src[blockIdx.x] * len;
    double2* b = out + (long long)blockIdx.x * len;
    for (long long g = threadIdx.x; g < len; g += NT) b[g] = a[g];
}

// C[m][n] <- coef(m, n) * (gamma ? 2 C[m][n] - A[m][0] X[n][0] : C[m][n])      (A[m][0], X[n][0]: real part of G = 0)
// coef(m, n) = dcoef[m] for the first n_rows_d rows (KB: D_k); for the others alpha_vec[orbital of column n] if given (alpha_v P_v,
// reading R3; colmap: compacted -> original column, nvpc vectors per column, orbital = column mod n_occ), else alpha_const.
__global__ void lowrank_fix(int M, int Nn, long long ldc, double* C, const double* A, long long lda, const double* X, long long ldx,
                            const double* dcoef, int n_rows_d, double alpha_const, const double* alpha_vec, const int* colmap, int nvpc,
                            int n_occ, int gamma) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)M * Nn) return;
    const int m = (int)(i / Nn), n = (int)(i - (long long)m * Nn);
    double c = C[(long long)m * ldc + n];
    if (gamma) c = 2.0 * c - A[(long long)m * lda] * X[(long long)n * ldx];
    double coef;
    if (m < n_rows_d) coef = dcoef[m];
    else if (alpha_vec) {
        int col = n / nvpc;
        if (colmap) { col = colmap[col]; if (col < 0) col = 0; }
        coef = alpha_vec[col % n_occ];
    } else coef = alpha_const;
    C[(long long)m * ldc + n] = coef * c;
}

// The same step for the tensor path of WEST_MIXED (tc_gemm.cuh): the overlap block arrives TRANSPOSED, Ct[n][ldt] (m contiguous), and
// leaves as the TF32 hi / lo split of coef(m, n) * fix(Ct[n][m]), [n][ldt] f32 each (rows m >= M are written as zero padding).
__global__ void lowrank_fix_split(int M, int Nn, long long ldt, const double* Ct, const double* A, long long lda, const double* X, long long ldx,
                                  const double* dcoef, int n_rows_d, double alpha_const, const double* alpha_vec, const int* colmap, int nvpc,
                                  int n_occ, int gamma, float* hi, float* lo) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)Nn * ldt) return;
    const int n = (int)(i / ldt), m = (int)(i - (long long)n * ldt);
    float h = 0.f, l = 0.f;
    if (m < M) {
        double c = Ct[i];
        if (gamma) c = 2.0 * c - A[(long long)m * lda] * X[(long long)n * ldx];
        double coef;
        if (m < n_rows_d) coef = dcoef[m];
        else if (alpha_vec) {
            int col = n / nvpc;
            if (colmap) { col = colmap[col]; if (col < 0) col = 0; }
            coef = alpha_vec[col % n_occ];
        } else coef = alpha_const;
        const float f = (float)(coef * c);
        unsigned int hb, lb;
        asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(hb) : "f"(f));
        const float r = f - __uint_as_float(hb);
        asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(lb) : "f"(r));
        h = __uint_as_float(hb); l = __uint_as_float(lb);
    }
    hi[i] = h; lo[i] = l;
}

// The same fix for the int8-slice path (i8_gemm.cuh): the overlap block arrives TRANSPOSED, Ct[n][ldt] (m contiguous), and is overwritten in
// place by coef(m, n) * fix(Ct[n][m]) in FP64 (the slicing kernel reads it next); entries m >= M are set to zero.
__global__ void lowrank_fix_t(int M, int Nn, long long ldt, double* Ct, const double* A, long long lda, const double* X, long long ldx,
                              const double* dcoef, int n_rows_d, double alpha_const, const double* alpha_vec, const int* colmap, int nvpc,
                              int n_occ, int gamma) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)Nn * ldt) return;
    const int n = (int)(i / ldt), m = (int)(i - (long long)n * ldt);
    double v = 0.0;
    if (m < M) {
        double c = Ct[i];
        if (gamma) c = 2.0 * c - A[(long long)m * lda] * X[(long long)n * ldx];
        double coef;
        if (m < n_rows_d) coef = dcoef[m];
        else if (alpha_vec) {
            int col = n / nvpc;
            if (colmap) { col = colmap[col]; if (col < 0) col = 0; }
            coef = alpha_vec[col % n_occ];
        } else coef = alpha_const;
        v = coef * c;
    }
    Ct[i] = v;
}

}  // namespace wcg
