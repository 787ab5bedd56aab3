// Sphere-pruned batched 3D FFT for the dual-space H*psi, "sticks and planes" decomposition:
//   K1  g2r_z   : sphere -> z sticks  (one 1D transform per non-empty (n_x,n_y) column)            -> W[slot][pz][col]
//   K2  planes  : per (slot, z-plane): y inverse on the disc rows, x inverse line by line, real-space op
//                 (x V_loc | store | dn accumulate | load product), x forward, y forward                -> W in place
//   K3  r2g_z   : z sticks -> sphere, fused with 1/N^3, the kinetic diagonal and the (eps + i omega) shift
// A 1D transform of length N = N1*N2 is two in-place register passes (strided DFT-N1 + twiddle, contiguous DFT-N2);
// the inverse leaves real-space index j = k1 + N1 k2 at POSITION p = N2 k1 + k2 and the forward transform consumes
// exactly that order, so no transposition or bit reversal is ever done.  All real-space arrays inside the library
// ([pz][py][px], x fastest) live in this position order; west.cu converts at the API boundary.
//
// Every phase between two barriers is a function of (tid, nthreads) so that the same code can be stepped on the host.
#pragma once
#include "dft_small.cuh"

#ifndef WEST_PAD
#define WEST_PAD 1        // row padding (complex elements) of every shared-memory line buffer
#endif

struct WestGeom {
    int N, n_max, nr, n_cols, n_units, gamma;
    long long n_g;
    const int* row_off;     // [nr+1]  first column of each n_x row of the disc (columns are lexicographic (n_x, n_y))
    const int* unit_off;    // [n_units] offset in sphere storage of the stick's first stored coefficient
    const int* unit_zmax;   // [n_units]
    const cx<double>* tw;   // [N] exp(+2 pi i m / N)
    const double* g2;       // [n_g] |G|^2 in storage order
};

// vector <-> slot mapping of K1/K3: FFT f (0 or 1) of slot s is vector s*vstride + f*voffb; vectors >= n_vec are zero padding.
struct VecMap {
    int vstride, voffb, n_vec;
    int slot0;      // first slot of this launch (W is indexed by the launch-local slot, vectors by slot0 + slot)
};

template <typename T> WHD cx<T> cvt(cx<double> a) { return mk<T>((T)a.x, (T)a.y); }
template <typename T> WHD cx<double> cvd(cx<T> a) { return mk<double>((double)a.x, (double)a.y); }
WHD int wrap_signed(int n, int N) { return n < N / 2 ? n : n - N; }

// zp[m] = z^m for m = 1 .. R-1 by binary splitting (dependency depth log2 R)
template <typename T, int R> WHD void tw_powers(cx<T> z, cx<T> (&zp)[R]) {
    zp[0] = mk<T>(1, 0);
    if (R > 1) zp[1] = z;
#pragma unroll
    for (int m = 2; m < R; ++m) zp[m] = cmul(zp[m / 2], zp[m - m / 2]);
}
// Alias-free grids have N >= 4 n_max + 1, so every non-zero frequency satisfies |n| <= (N-1)/4.  For the strided pass
// (n = N2 n1 + n2) this tells at COMPILE time which n1 can hold a non-zero input / a needed output at all.
template <int N1, int N2> WHD constexpr bool keep_n1(int n1) {
    constexpr int N = N1 * N2, LIM = (N - 1) / 4;
    // the run n = N2 n1 .. N2 n1 + N2 - 1 meets [0, LIM] or [N - LIM, N - 1]
    return (N2 * n1 <= LIM) || (N2 * n1 + N2 - 1 >= N - LIM);
}

// ---------------------------------------------------------------------------------------------------------------- K1
template <typename T, int N1, int N2, bool GAMMA, int CU>
struct K1 {
    static constexpr int N = N1 * N2, PITCH = N + WEST_PAD, NF = GAMMA ? 2 : 1, NL = CU * NF;
    static constexpr size_t smem_bytes = sizeof(cx<T>) * (size_t)(NL * PITCH + 2 * N);

    // phase A: strided DFT-N1 straight from the sphere coefficients, twiddle, store to the line buffer
    static WHD void phaseA(int tid, int nthr, cx<T>* lines, const cx<T>* tw, const WestGeom& g, VecMap vm, int slot, int u0,
                           const cx<double>* X) {
        for (int it = tid; it < NL * N2; it += nthr) {
            const int line = it / N2, n2 = it - line * N2;
            const int u = u0 + line / NF, f = line % NF;
            cx<T> v[N1];
            const long long vec = (long long)(vm.slot0 + slot) * vm.vstride + (long long)f * vm.voffb;
            if (u < g.n_units && vec < vm.n_vec) {
                const int zmax = g.unit_zmax[u];
                const cx<double>* src = X + vec * g.n_g + g.unit_off[u];
                const bool half00 = GAMMA && u == 0;
#pragma unroll
                for (int n1 = 0; n1 < N1; ++n1) {
                    const int nz = wrap_signed(N2 * n1 + n2, N);
                    cx<T> val = mk<T>(0, 0);
                    if (keep_n1<N1, N2>(n1) && nz <= zmax && nz >= -zmax) {
                        if (half00) {
                            cx<double> c = src[nz >= 0 ? nz : -nz];
                            val = mk<T>((T)c.x, (T)(nz >= 0 ? c.y : -c.y));
                            if (nz == 0) val.y = 0;     // c(0) of a real function is real
                        } else {
                            val = cvt<T>(src[nz + zmax]);
                        }
                    }
                    v[n1] = val;
                }
                Dft<T, N1, +1>::run(v);
            } else {
#pragma unroll
                for (int n1 = 0; n1 < N1; ++n1) v[n1] = mk<T>(0, 0);
            }
            cx<T>* dst = lines + line * PITCH + n2;
{
                cx<T> zp[N1];
                tw_powers<T, N1>(tw[N2 + n2], zp);
#pragma unroll
                for (int k1 = 0; k1 < N1; ++k1) dst[N2 * k1] = k1 == 0 ? v[0] : cmul(v[k1], zp[k1]);
            }
        }
    }
    // ---- GAMMA: two phases, one barrier, the line buffer is written once and read once.
    // GAMMA: the two lines of a unit are formed WHILE LOADING as  line 2ul = a(n) + i b(n)  and  line 2ul+1 = conj(a(-n)) + i conj(b(-n)),
    // whose transforms are S+ = A + iB and S- = conj(A) + i conj(B) themselves, so phase BC stores its registers straight to the
    // column cp and its mirror.  FULL: phaseA as above, then phaseBC.
    static WHD cx<T> coef(const cx<double>* src, int m, int zmax, bool half00) {
        if (half00) {                                   // column (0,0): only n_z >= 0 is stored, c(-n) = conj(c(n)), c(0) real
            const cx<double> c = src[m >= 0 ? m : -m];
            return mk<T>((T)c.x, m == 0 ? (T)0 : (T)(m > 0 ? c.y : -c.y));
        }
        return cvt<T>(src[m + zmax]);
    }
    static WHD void phaseA2(int tid, int nthr, cx<T>* lines, const cx<T>* tw, const WestGeom& g, VecMap vm, int slot, int u0,
                            const cx<double>* X) {
        if (!GAMMA) { phaseA(tid, nthr, lines, tw, g, vm, slot, u0, X); return; }
        for (int it = tid; it < NL * N2; it += nthr) {
            const int line = it / N2, n2 = it - line * N2;
            const int u = u0 + line / 2, sgn = line & 1;
            cx<T> v[N1];
            const long long vec0 = (long long)(vm.slot0 + slot) * vm.vstride, vec1 = vec0 + vm.voffb;
            // column 0 is its own mirror: its minus line is never stored
            if (u < g.n_units && vec0 < vm.n_vec && !(u == 0 && sgn)) {
                const int zmax = g.unit_zmax[u];
                const bool half00 = u == 0, has_b = vec1 < vm.n_vec;
                const cx<double>* sa = X + vec0 * g.n_g + g.unit_off[u];
                const cx<double>* sb = X + vec1 * g.n_g + g.unit_off[u];
#pragma unroll
                for (int n1 = 0; n1 < N1; ++n1) {
                    const int nz = wrap_signed(N2 * n1 + n2, N);
                    cx<T> val = mk<T>(0, 0);
                    if (keep_n1<N1, N2>(n1) && nz <= zmax && nz >= -zmax) {
                        const int m = sgn ? -nz : nz;
                        const cx<T> a = coef(sa, m, zmax, half00);
                        const cx<T> b = has_b ? coef(sb, m, zmax, half00) : mk<T>(0, 0);
                        val = sgn ? mk<T>(a.x + b.y, b.x - a.y) : mk<T>(a.x - b.y, a.y + b.x);
                    }
                    v[n1] = val;
                }
                Dft<T, N1, +1>::run(v);
            } else {
#pragma unroll
                for (int n1 = 0; n1 < N1; ++n1) v[n1] = mk<T>(0, 0);
            }
            cx<T>* dst = lines + line * PITCH + n2;
            {
                cx<T> zp[N1];
                tw_powers<T, N1>(tw[N2 + n2], zp);
#pragma unroll
                for (int k1 = 0; k1 < N1; ++k1) dst[N2 * k1] = k1 == 0 ? v[0] : cmul(v[k1], zp[k1]);
            }
        }
    }
    // contiguous DFT-N2 of (line, k1), registers straight to W; lanes run over the lines, i.e. over consecutive columns
    static WHD void phaseBC(int tid, int nthr, const cx<T>* lines, const WestGeom& g, int slot, int u0, cx<T>* W) {
        for (int it = tid; it < NL * N1; it += nthr) {
            const int k1 = it / NL, line = it - k1 * NL;
            const int u = u0 + line / NF, sgn = GAMMA ? (line & 1) : 0;
            if (u >= g.n_units || (GAMMA && sgn && u == 0)) continue;
            const cx<T>* p = lines + line * PITCH + N2 * k1;
            cx<T> v[N2];
#pragma unroll
            for (int j = 0; j < N2; ++j) v[j] = p[j];
            Dft<T, N2, +1>::run(v);
            const int cp = GAMMA ? u + (g.n_cols - g.n_units) : u;
            const int col = sgn ? g.n_cols - 1 - cp : cp;
            cx<T>* dst = W + ((long long)slot * N + N2 * k1) * g.n_cols + col;
#pragma unroll
            for (int j = 0; j < N2; ++j) dst[(long long)j * g.n_cols] = v[j];
        }
    }
};

// ---------------------------------------------------------------------------------------------------------------- K3
struct K3Epi {
    double scale;           // 1/N^3
    int kinetic;            // 1: y += (g2 - shift[vec]) * x
    const double* shift;    // [n_vec] or NULL (0)
    double omega;           // i*omega shift: FULL y -= i omega x ; GAMMA (pairs f=0: Re, f=1: Im)  y_a += omega x_b, y_b -= omega x_a
    const cx<double>* X;    // input vectors (kinetic / shift terms), may be NULL when kinetic == 0
};

template <typename T, int N1, int N2, bool GAMMA, int CU>
struct K3 {
    static constexpr int N = N1 * N2, PITCH = N + WEST_PAD, NF = GAMMA ? 2 : 1, NL = CU * NF;
    static constexpr size_t smem_bytes = sizeof(cx<T>) * (size_t)(NL * PITCH + 2 * N);

    // W -> registers -> (GAMMA: separate the two real functions with the partner lane) -> DFT-N2, twiddle -> line buffer.  Item (k1, line), lanes over the lines: lane pair (2m, 2m+1)
    // holds column cp (S+) and its mirror (S-) of the same unit at the same N2 positions.  On the host (stepped test) the
    // partner's values are simply loaded again.
    static WHD void phaseAB(int tid, int nthr, cx<T>* lines, const cx<T>* tw, const WestGeom& g, int slot, int u0, const cx<T>* W) {
        constexpr int ITEMS = NL * N1, ROUND = (ITEMS + 31) / 32 * 32;       // whole warps take part in the exchange
        for (int it = tid; it < ROUND; it += nthr) {
            const int k1 = it / NL, line = it - k1 * NL;
            const int u = u0 + line / NF, sgn = GAMMA ? (line & 1) : 0;
            const bool valid = it < ITEMS && u < g.n_units;
            cx<T> v[N2];
            const int cp = GAMMA ? u + (g.n_cols - g.n_units) : u;
            const int mirror = (GAMMA && u != 0) ? g.n_cols - 1 - cp : cp;     // column 0 is its own mirror
            const cx<T>* src = W + ((long long)slot * N + N2 * k1) * g.n_cols;
#pragma unroll
            for (int j = 0; j < N2; ++j) v[j] = valid ? src[(long long)j * g.n_cols + (sgn ? mirror : cp)] : mk<T>(0, 0);
            if (GAMMA) {
#pragma unroll
                for (int j = 0; j < N2; ++j) {
                    cx<T> o;
#ifdef __CUDA_ARCH__
                    o.x = __shfl_xor_sync(0xffffffffu, v[j].x, 1);
                    o.y = __shfl_xor_sync(0xffffffffu, v[j].y, 1);
#else
                    o = valid ? src[(long long)j * g.n_cols + (sgn ? cp : mirror)] : mk<T>(0, 0);
#endif
                    // sgn 0 holds S+ and receives S-: a = (S+ + conj S-)/2 ; sgn 1 holds S- and receives S+: b = (S+ - conj S-)/(2i)
                    v[j] = sgn ? mk<T>((T)0.5 * (o.y + v[j].y), (T)0.5 * (v[j].x - o.x)) : mk<T>((T)0.5 * (v[j].x + o.x), (T)0.5 * (v[j].y - o.y));
                }
            }
            if (it >= ITEMS) continue;
            Dft<T, N2, -1>::run(v);
            cx<T>* p = lines + line * PITCH + N2 * k1;
            {
                cx<T> zp[N2];
                tw_powers<T, N2>(tw[N + N1 + k1], zp);
#pragma unroll
                for (int j = 0; j < N2; ++j) p[j] = j == 0 ? v[j] : cmulc(v[j], zp[j]);
            }
        }
    }
    // phase A': strided DFT-N1 (sign -), epilogue to the sphere
    static WHD void phaseC(int tid, int nthr, const cx<T>* lines, const WestGeom& g, VecMap vm, int slot, int u0,
                           K3Epi e, cx<double>* Y) {
        for (int it = tid; it < NL * N2; it += nthr) {
            const int line = it / N2, n2 = it - line * N2;
            const int u = u0 + line / NF, f = line % NF;
            const long long vec = (long long)(vm.slot0 + slot) * vm.vstride + (long long)f * vm.voffb;
            if (u >= g.n_units || vec >= vm.n_vec) continue;
            const int zmax = g.unit_zmax[u];
            const bool half00 = GAMMA && u == 0;
            const long long base = vec * g.n_g + g.unit_off[u];
            const long long pbase = GAMMA ? ((long long)(vm.slot0 + slot) * vm.vstride + (long long)(1 - f) * vm.voffb) * g.n_g + g.unit_off[u] : 0;
            const double sh = (e.kinetic && e.shift) ? e.shift[vec] : 0.0;
            const cx<T>* p = lines + line * PITCH + n2;
            cx<T> v[N1];
#pragma unroll
            for (int k1 = 0; k1 < N1; ++k1) v[k1] = p[N2 * k1];
            Dft<T, N1, -1>::run(v);
#pragma unroll
            for (int n1 = 0; n1 < N1; ++n1) {
                if (!keep_n1<N1, N2>(n1)) continue;
                const int nz = wrap_signed(N2 * n1 + n2, N);
                if (nz > zmax || nz < (half00 ? 0 : -zmax)) continue;
                const long long o = half00 ? nz : nz + zmax;
                cx<double> r = mk<double>(e.scale * (double)v[n1].x, e.scale * (double)v[n1].y);
                if (e.kinetic) {
                    const double d = g.g2[g.unit_off[u] + o] - sh;
                    const cx<double> x = e.X[base + o];
                    r.x += d * x.x; r.y += d * x.y;
                    if (e.omega != 0.0) {
                        if (GAMMA) {
                            const cx<double> xp = e.X[pbase + o];
                            const double w = f == 0 ? e.omega : -e.omega;
                            r.x += w * xp.x; r.y += w * xp.y;
                        } else {
                            r.x += e.omega * x.y; r.y -= e.omega * x.x;
                        }
                    }
                }
                if (half00 && nz == 0) r.y = 0.0;
                Y[base + o] = r;
            }
        }
    }
};

// ---------------------------------------------------------------------------------------------------------------- K2
enum { K2_H = 0, K2_TOR = 1, K2_DN = 2, K2_FROMR = 3 };

template <typename T>
struct K2Args {
    cx<T>* W;                   // [n_slots][N][n_cols] stick intermediate (in place)
    const T* V;                 // K2_H: V_loc in position order [pz][py][px]
    cx<double>* R;              // K2_TOR: out [n_slots][N^3] ; K2_FROMR with ucache == NULL: in
    const cx<double>* ucache;   // K2_DN / K2_FROMR: occupied orbitals in real space [n_uslots][N^3] position order
    const double* dV;           // K2_FROMR: [n_pert][N^3] position order (real)
    double* dn;                 // K2_DN: [n_pert][N^3] position order, accumulated with atomics
    int n_uslots;               // global slot = ipert * n_uslots + uslot
    int slot0;                  // first global slot of this launch (W and R are indexed by the launch-local slot)
    double fac;                 // K2_DN: 4/Omega
};

// LC = lines (x) or rows (y) a thread group owns per round; NB = independent items every thread runs in lockstep inside a pass (loads
// of all NB items are issued before the first butterfly, stores after the last: NB load -> butterfly -> store chains in flight per
// thread instead of one; the round then covers NB * LC lines).  NB = 1 is the plain one-item-per-thread pass.
template <typename T, int N1, int N2, int MODE, int LC>
struct K2 {
    // Shared-memory line layout.  Position p = N2 k1 + k2 of a line sits at element B2 k1 + k2: when N2 is even the N2-blocks are padded
    // by one element (B2 = N2 + 1), because the contiguous passes put the lanes of a warp B2 elements apart and an even stride maps
    // them onto half (N2 = 12: a quarter) of the eight 16-byte bank groups (measured at N = 144: 57 % of the shared-memory wavefronts
    // were conflict replays).  The row pitch is the smallest value >= the line length that is congruent to N2 modulo 8, so that the
    // strided passes (lanes = (line, n2), consecutive) stay conflict-free as well.
    static constexpr int N = N1 * N2, B2 = N2 + ((N2 % 2 == 0) ? 1 : 0), NP = N1 * B2;
    // even N2: the row pitch is made ODD as well - the x passes gather / scatter one element per row of S (lanes = consecutive n_x rows)
    // and an even pitch folds those onto fewer bank groups (pitch 156 at N = 144 still showed 24 % replays)
    static constexpr int PITCH = (N2 % 2 == 0) ? (NP | 1) : NP + ((N2 - NP) % 8 + 8) % 8 + ((NP + ((N2 - NP) % 8 + 8) % 8 == N) ? 8 : 0);
    static WHD int pos(int p) { return (N2 % 2 == 0) ? p + p / N2 : p; }          // padded element index of position p
    static WHD size_t smem_bytes(int nr) { return sizeof(cx<T>) * (size_t)((nr + LC) * PITCH + 2 * N); }

    // layout of V_loc for the K2_H variant: position (pz, py = py0 + l, px = N2 k1 + k2), py0 a multiple of LC
    static constexpr int NCH = (N + LC - 1) / LC;
    static WHD size_t vloc_elems() { return (size_t)N * NCH * N2 * LC * N1; }
    static WHD long long vloc_index(int pz, int py0, int l, int k1, int k2) {
        return ((((long long)pz * NCH + py0 / LC) * N2 + k2) * LC + l) * N1 + k1;
    }
    static WHD cx<T> load_disc(const cx<T>* Wp, const WestGeom& g, int row, int n) {
        const int c0 = g.row_off[row], ymax = (g.row_off[row + 1] - c0 - 1) >> 1;
        const int ny = wrap_signed(n, N);
        return (ny <= ymax && ny >= -ymax) ? Wp[c0 + ny + ymax] : mk<T>(0, 0);
    }
    // strided-pass epilogue: v[k1] * w^(n2 k1) -> dst[N2 k1]   (level twiddles as powers of ONE table entry per thread: the kernels are
    // bound by L1TEX wavefronts, so FP64 work is traded for table look-ups)
    static WHD void tw_store_strided(cx<T> (&v)[N1], cx<T> z, cx<T>* dst) {
        cx<T> zp[N1];
        tw_powers<T, N1>(z, zp);
#pragma unroll
        for (int k1 = 0; k1 < N1; ++k1) dst[B2 * k1] = k1 == 0 ? v[0] : cmul(v[k1], zp[k1]);
    }
    // contiguous-pass epilogue of the forward direction: v[j] * conj(w^(k1 j)) -> p[j]
    static WHD void tw_store_contig(cx<T> (&v)[N2], cx<T> z, cx<T>* p) {
        cx<T> zp[N2];
        tw_powers<T, N2>(z, zp);
#pragma unroll
        for (int j = 0; j < N2; ++j) p[j] = j == 0 ? v[j] : cmulc(v[j], zp[j]);
    }

    // y inverse, pass A: rows of the disc straight from W
    template <int NB = 1>
    static WHD void yA(int tid, int nthr, cx<T>* S, const cx<T>* tw, const WestGeom& g, const cx<T>* Wp, int row0, int nrow) {
        for (int it0 = tid; it0 < nrow * N2; it0 += NB * nthr) {
            cx<T> v[NB][N1];
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                const int it = it0 + b * nthr;
                const int rl = it / N2, n2 = it - rl * N2, row = row0 + rl;
#pragma unroll
                for (int n1 = 0; n1 < N1; ++n1)
                    v[b][n1] = ((NB == 1 || it < nrow * N2) && keep_n1<N1, N2>(n1)) ? load_disc(Wp, g, row, N2 * n1 + n2) : mk<T>(0, 0);
            }
#pragma unroll
            for (int b = 0; b < NB; ++b) Dft<T, N1, +1>::run(v[b]);
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                const int it = it0 + b * nthr;
                if (NB > 1 && it >= nrow * N2) continue;
                const int rl = it / N2, n2 = it - rl * N2, row = row0 + rl;
                tw_store_strided(v[b], tw[N2 + n2], S + row * PITCH + n2);
            }
        }
    }
    template <int NB = 1>
    static WHD void yB(int tid, int nthr, cx<T>* S, const WestGeom& g, int row0, int nrow) {
        for (int it0 = tid; it0 < nrow * N1; it0 += NB * nthr) {
            cx<T> v[NB][N2];
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                const int it = it0 + b * nthr;
                const bool ok = NB == 1 || it < nrow * N1;            // (the loop bound covers b = 0)
                const cx<T>* p = S + (row0 + it / N1) * PITCH + B2 * (it % N1);
#pragma unroll
                for (int j = 0; j < N2; ++j) v[b][j] = ok ? p[j] : mk<T>(0, 0);
            }
#pragma unroll
            for (int b = 0; b < NB; ++b) Dft<T, N2, +1>::run(v[b]);
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                const int it = it0 + b * nthr;
                if (NB > 1 && it >= nrow * N1) continue;
                cx<T>* p = S + (row0 + it / N1) * PITCH + B2 * (it % N1);
#pragma unroll
                for (int j = 0; j < N2; ++j) p[j] = v[b][j];
            }
        }
    }
    // x inverse, pass A: gather the 2 n_max + 1 non-zero inputs of LC lines from S
    template <int NB = 1>
    static WHD void xA(int tid, int nthr, const cx<T>* S, cx<T>* X, const cx<T>* tw, const WestGeom& g, int py0) {
        for (int it0 = tid; it0 < LC * N2; it0 += NB * nthr) {
            if (NB == 1 && py0 + it0 / N2 >= N) continue;                 // NB = 1: an item beyond the grid is skipped outright
            cx<T> v[NB][N1];
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                const int it = it0 + b * nthr;
                const int l = it / N2, n2 = it - l * N2, py = py0 + l;
                const bool ok = NB == 1 || (it < LC * N2 && py < N);
#pragma unroll
                for (int n1 = 0; n1 < N1; ++n1) {
                    const int nx = wrap_signed(N2 * n1 + n2, N);
                    v[b][n1] = (ok && keep_n1<N1, N2>(n1) && nx <= g.n_max && nx >= -g.n_max) ? S[(nx + g.n_max) * PITCH + pos(py)] : mk<T>(0, 0);
                }
            }
#pragma unroll
            for (int b = 0; b < NB; ++b) Dft<T, N1, +1>::run(v[b]);
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                const int it = it0 + b * nthr;
                const int l = it / N2, n2 = it - l * N2;
                if (NB > 1 && (it >= LC * N2 || py0 + l >= N)) continue;
                tw_store_strided(v[b], tw[N2 + n2], X + l * PITCH + n2);
            }
        }
    }
    // the real-space operation on the N2 contiguous values of item (l, k1) between x inverse pass B and x forward pass B'
    static WHD bool xB_mid(cx<T> (&v)[N2], const K2Args<T>& a, int slot, int pz, int py0, int l, int k1) {
        const int py = py0 + l;
        const long long r0 = ((long long)pz * N + py) * N + N2 * k1;      // position-order real-space index
        const long long n3 = (long long)N * N * N;
        if (MODE == K2_H) {
            // V_loc is stored per chunk of LC lines as [pz][py0 / LC][k2][l][k1] (vloc_index): for a fixed j = k2 the LC * N1
            // threads of a line group read LC * N1 consecutive words - whole 128-byte lines instead of one 8 N1-byte piece per line
            const T* V = a.V + vloc_index(pz, py0, l, k1, 0);
#pragma unroll
            for (int j = 0; j < N2; ++j) { const T w = V[j * (LC * N1)]; v[j].x *= w; v[j].y *= w; }
            return true;
        } else if (MODE == K2_TOR) {
            cx<double>* R = a.R + (long long)slot * n3 + r0;
#pragma unroll
            for (int j = 0; j < N2; ++j) R[j] = cvd<T>(v[j]);
            return false;
        } else if (MODE == K2_DN) {
            const int gs = a.slot0 + slot, ip = gs / a.n_uslots, us = gs - ip * a.n_uslots;
            const cx<double>* U = a.ucache + (long long)us * n3 + r0;
            double* D = a.dn + (long long)ip * n3 + r0;
#pragma unroll
            for (int j = 0; j < N2; ++j) {
                const cx<double> u = U[j];
                const double val = a.fac * ((double)v[j].x * u.x + (double)v[j].y * u.y);
#ifdef __CUDA_ARCH__
                atomicAdd(D + j, val);
#else
                D[j] += val;
#endif
            }
            return false;
        } else {   // K2_FROMR
            if (a.ucache) {
                const int gs = a.slot0 + slot, ip = gs / a.n_uslots, us = gs - ip * a.n_uslots;
                const cx<double>* U = a.ucache + (long long)us * n3 + r0;
                const double* D = a.dV + (long long)ip * n3 + r0;
#pragma unroll
                for (int j = 0; j < N2; ++j) { const double w = D[j]; const cx<double> u = U[j]; v[j] = mk<T>((T)(u.x * w), (T)(u.y * w)); }
            } else {
                const cx<double>* R = a.R + (long long)slot * n3 + r0;
#pragma unroll
                for (int j = 0; j < N2; ++j) v[j] = cvt<T>(R[j]);
            }
            return true;
        }
    }
    // x inverse pass B, the real-space operation, x forward pass B' - all on the same N2 contiguous values
    template <int NB = 1>
    static WHD void xB(int tid, int nthr, cx<T>* X, const cx<T>* tw, const K2Args<T>& a, int slot, int pz, int py0) {
        for (int it0 = tid; it0 < LC * N1; it0 += NB * nthr) {
            if (NB == 1 && py0 + it0 / N1 >= N) continue;
            cx<T> v[NB][N2];
            bool ok[NB], fwd[NB];
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                const int it = it0 + b * nthr;
                const int l = it / N1, k1 = it - l * N1;
                ok[b] = NB == 1 || (it < LC * N1 && py0 + l < N);
                if (MODE != K2_FROMR) {
                    const cx<T>* p = X + l * PITCH + B2 * k1;
#pragma unroll
                    for (int j = 0; j < N2; ++j) v[b][j] = ok[b] ? p[j] : mk<T>(0, 0);
                }
            }
            if (MODE != K2_FROMR) {
#pragma unroll
                for (int b = 0; b < NB; ++b) Dft<T, N2, +1>::run(v[b]);
            }
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                const int it = it0 + b * nthr;
                fwd[b] = ok[b] && xB_mid(v[b], a, slot, pz, py0, it / N1, it % N1);
            }
            if (MODE == K2_H || MODE == K2_FROMR) {
#pragma unroll
                for (int b = 0; b < NB; ++b) Dft<T, N2, -1>::run(v[b]);
#pragma unroll
                for (int b = 0; b < NB; ++b) {
                    const int it = it0 + b * nthr;
                    const int l = it / N1, k1 = it - l * N1;
                    if (fwd[b]) tw_store_contig(v[b], tw[N + N1 + k1], X + l * PITCH + B2 * k1);
                }
            }
        }
    }
    // x forward pass A': strided DFT-N1, keep |n_x| <= n_max, back into S
    template <int NB = 1>
    static WHD void xC(int tid, int nthr, cx<T>* S, const cx<T>* X, const WestGeom& g, int py0) {
        for (int it0 = tid; it0 < LC * N2; it0 += NB * nthr) {
            if (NB == 1 && py0 + it0 / N2 >= N) continue;
            cx<T> v[NB][N1];
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                const int it = it0 + b * nthr;
                const int l = it / N2, n2 = it - l * N2;
                const bool ok = NB == 1 || (it < LC * N2 && py0 + l < N);
                const cx<T>* p = X + l * PITCH + n2;
#pragma unroll
                for (int k1 = 0; k1 < N1; ++k1) v[b][k1] = ok ? p[B2 * k1] : mk<T>(0, 0);
            }
#pragma unroll
            for (int b = 0; b < NB; ++b) Dft<T, N1, -1>::run(v[b]);
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                const int it = it0 + b * nthr;
                const int l = it / N2, n2 = it - l * N2, py = py0 + l;
                if (NB > 1 && (it >= LC * N2 || py >= N)) continue;
#pragma unroll
                for (int n1 = 0; n1 < N1; ++n1) {
                    if (!keep_n1<N1, N2>(n1)) continue;
                    const int nx = wrap_signed(N2 * n1 + n2, N);
                    if (nx <= g.n_max && nx >= -g.n_max) S[(nx + g.n_max) * PITCH + pos(py)] = v[b][n1];
                }
            }
        }
    }
    template <int NB = 1>
    static WHD void yC(int tid, int nthr, cx<T>* S, const cx<T>* tw, const WestGeom& g, int row0, int nrow) {
        for (int it0 = tid; it0 < nrow * N1; it0 += NB * nthr) {
            cx<T> v[NB][N2];
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                const int it = it0 + b * nthr;
                const bool ok = NB == 1 || it < nrow * N1;            // (the loop bound covers b = 0)
                const cx<T>* p = S + (row0 + it / N1) * PITCH + B2 * (it % N1);
#pragma unroll
                for (int j = 0; j < N2; ++j) v[b][j] = ok ? p[j] : mk<T>(0, 0);
            }
#pragma unroll
            for (int b = 0; b < NB; ++b) Dft<T, N2, -1>::run(v[b]);
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                const int it = it0 + b * nthr;
                if (NB > 1 && it >= nrow * N1) continue;
                const int k1 = it % N1;
                tw_store_contig(v[b], tw[N + N1 + k1], S + (row0 + it / N1) * PITCH + B2 * k1);
            }
        }
    }
    template <int NB = 1>
    static WHD void yD(int tid, int nthr, const cx<T>* S, const WestGeom& g, cx<T>* Wp, int row0, int nrow) {
        for (int it0 = tid; it0 < nrow * N2; it0 += NB * nthr) {
            cx<T> v[NB][N1];
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                const int it = it0 + b * nthr;
                const bool ok = NB == 1 || it < nrow * N2;
                const cx<T>* p = S + (row0 + it / N2) * PITCH + it % N2;
#pragma unroll
                for (int k1 = 0; k1 < N1; ++k1) v[b][k1] = ok ? p[B2 * k1] : mk<T>(0, 0);
            }
#pragma unroll
            for (int b = 0; b < NB; ++b) Dft<T, N1, -1>::run(v[b]);
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                const int it = it0 + b * nthr;
                if (NB > 1 && it >= nrow * N2) continue;
                const int rl = it / N2, n2 = it - rl * N2, row = row0 + rl;
                const int c0 = g.row_off[row], ymax = (g.row_off[row + 1] - c0 - 1) >> 1;
#pragma unroll
                for (int n1 = 0; n1 < N1; ++n1) {
                    if (!keep_n1<N1, N2>(n1)) continue;
                    const int ny = wrap_signed(N2 * n1 + n2, N);
                    if (ny <= ymax && ny >= -ymax) Wp[c0 + ny + ymax] = v[b][n1];
                }
            }
        }
    }
};

#ifdef __CUDACC__
#ifndef WEST_ZMINB
#define WEST_ZMINB 1      // resident CTAs per SM the z-stick kernels are compiled for (register cap)
#endif
#ifndef WEST_ZNT
#define WEST_ZNT 256       // threads per CTA of the z-stick kernels
#endif
template <typename T, int N1, int N2>
__device__ __forceinline__ void load_tw(cx<T>* tw_s, const cx<double>* tw_g) {
    // level twiddles in the two orders the passes read them, so that the lanes of a warp hit consecutive entries:
    // tw_s[k1 * N2 + n2] = w^(n2 k1) (strided pass, lanes run over n2); tw_s[N + j * N1 + k1] = w^(k1 j) (contiguous pass, lanes over k1)
    constexpr int N = N1 * N2;
    for (int i = threadIdx.x; i < N; i += blockDim.x) {
        const int k1 = i / N2, n2 = i - k1 * N2;
        tw_s[i] = cvt<T>(tw_g[n2 * k1]);
        const int j = i / N1, k1b = i - j * N1;
        tw_s[N + i] = cvt<T>(tw_g[k1b * j]);
    }
}

template <typename T, int N1, int N2, bool GAMMA, int CU>
__global__ void __launch_bounds__(WEST_ZNT, WEST_ZMINB) k1_g2r_z(WestGeom g, VecMap vm, const cx<double>* X, cx<T>* W) {
    using K = K1<T, N1, N2, GAMMA, CU>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* lines = reinterpret_cast<cx<T>*>(smem_raw);
    cx<T>* tw = lines + K::NL * K::PITCH;
    load_tw<T, N1, N2>(tw, g.tw);
    __syncthreads();
    const int slot = blockIdx.y, u0 = blockIdx.x * CU;
    K::phaseA2(threadIdx.x, blockDim.x, lines, tw, g, vm, slot, u0, X);
    __syncthreads();
    K::phaseBC(threadIdx.x, blockDim.x, lines, g, slot, u0, W);
}

template <typename T, int N1, int N2, bool GAMMA, int CU>
__global__ void __launch_bounds__(WEST_ZNT, WEST_ZMINB) k3_r2g_z(WestGeom g, VecMap vm, const cx<T>* W, K3Epi e, cx<double>* Y) {
    using K = K3<T, N1, N2, GAMMA, CU>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* lines = reinterpret_cast<cx<T>*>(smem_raw);
    cx<T>* tw = lines + K::NL * K::PITCH;
    load_tw<T, N1, N2>(tw, g.tw);
    const int slot = blockIdx.y, u0 = blockIdx.x * CU;
    if (e.kinetic) {
        // the epilogue reads x(G) of this CTA's sticks at the very end: pull those lines towards L2 now (128 B per request)
        for (int it = threadIdx.x; it < K::NL * 5; it += blockDim.x) {
            const int line = it / 5, seg = it - line * 5;
            const int u = u0 + line / K::NF, f = line % K::NF;
            const long long vec = (long long)(vm.slot0 + slot) * vm.vstride + (long long)f * vm.voffb;
            if (u < g.n_units && vec < vm.n_vec && seg * 8 <= 2 * g.unit_zmax[u])
                asm volatile("prefetch.global.L2 [%0];" ::"l"(e.X + vec * g.n_g + g.unit_off[u] + seg * 8));
        }
    }
    __syncthreads();                                   // twiddles
    K::phaseAB(threadIdx.x, blockDim.x, lines, tw, g, slot, u0, W);
    __syncthreads();
    K::phaseC(threadIdx.x, blockDim.x, lines, g, vm, slot, u0, e, Y);
}

// Plane kernel.  NW warps per CTA in groups of GW warps (GW = 1 or 2); each group owns LPG = 32 GW / max(N1, N2) lines per item slot and
// NB item slots per thread (K2's NB), i.e. NB * LPG lines per round, and runs the three passes of "its" lines with group-level barriers
// only (__syncwarp, or a named barrier for a warp pair), so the CTA synchronises just twice (after y inverse, before y forward).
// Warp pairs raise the lane utilisation of the passes: at N = 72 a warp holds 3 lines (27 / 24 of 32 lanes busy), a pair holds 7
// (63 / 56 of 64).  NB = 2 gives every thread two independent load -> butterfly -> store chains per pass (the kernel is latency-bound:
// 0.8 eligible of 4.3 resident warps per scheduler at NB = 1, profiles/r01_k2_pipe_experiments.md).
template <int N1, int N2, int GW = 1, int NB = 1> struct K2Cfg { static constexpr int LPW = NB * (32 * GW / (N1 > N2 ? N1 : N2)); };

template <int GW>
__device__ __forceinline__ void group_sync(int group) {
    if (GW == 1) __syncwarp();
    else asm volatile("bar.sync %0, %1;" ::"r"(group + 1), "r"(GW * 32) : "memory");
}

template <typename T, int N1, int N2, int MODE, int NW, int MINB, int GW = 1, int NB = 1>
__global__ void __launch_bounds__(NW * 32, MINB) k2_planes(WestGeom g, K2Args<T> a) {
    constexpr int LPG = K2Cfg<N1, N2, GW, NB>::LPW, GT = GW * 32, NG = NW / GW;
    static_assert(NW % GW == 0 && (GW == 1 || NG <= 15), "warp-pair groups use named barriers 1..15");
    using K = K2<T, N1, N2, MODE, LPG>;
    constexpr int N = K::N;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* S = reinterpret_cast<cx<T>*>(smem_raw);
    cx<T>* X = S + g.nr * K::PITCH;
    cx<T>* tw = X + NG * LPG * K::PITCH;
    const int group = threadIdx.x / GT, gt = threadIdx.x - group * GT;
    cx<T>* Xw = X + group * LPG * K::PITCH;
    load_tw<T, N1, N2>(tw, g.tw);
    const int pz = blockIdx.x, slot = blockIdx.y;
    cx<T>* Wp = a.W + ((long long)slot * N + pz) * g.n_cols;
    __syncthreads();
    if (MODE != K2_FROMR) {
        for (int r0 = group * LPG; r0 < g.nr; r0 += NG * LPG) {
            const int nrow = g.nr - r0 < LPG ? g.nr - r0 : LPG;
            K::template yA<NB>(gt, GT, S, tw, g, Wp, r0, nrow);
            group_sync<GW>(group);
            K::template yB<NB>(gt, GT, S, g, r0, nrow);
        }
        __syncthreads();
    }
    for (int py0 = group * LPG; py0 < N; py0 += NG * LPG) {
        if (MODE != K2_FROMR) {
            K::template xA<NB>(gt, GT, S, Xw, tw, g, py0);
            group_sync<GW>(group);
        }
        K::template xB<NB>(gt, GT, Xw, tw, a, slot, pz, py0);
        if (MODE == K2_H || MODE == K2_FROMR) {
            group_sync<GW>(group);
            K::template xC<NB>(gt, GT, S, Xw, g, py0);
        }
        group_sync<GW>(group);
    }
    if (MODE == K2_H || MODE == K2_FROMR) {
        __syncthreads();
        for (int r0 = group * LPG; r0 < g.nr; r0 += NG * LPG) {
            const int nrow = g.nr - r0 < LPG ? g.nr - r0 : LPG;
            K::template yC<NB>(gt, GT, S, tw, g, r0, nrow);
            group_sync<GW>(group);
            K::template yD<NB>(gt, GT, S, g, Wp, r0, nrow);
        }
    }
}
#endif
