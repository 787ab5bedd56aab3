// C-ABI implementation (include/west.h): context, operator set-up, and the drivers that chain the hand-written kernels
// of the chi0*dV hot path (Eq. 10-11).  Every step of the path runs in kernels of this library;
// there is no CPU fallback.
#include <cuda_runtime.h>
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <string>
#include <map>
#include <mutex>
#include <vector>

#include "../../include/west.h"
#include "cg_kernels.cuh"
#include "fft_ops.h"
#include "fft_dense.h"
#include "gemm_f64.cuh"
#include "gsphere.hpp"
#include "lanczos_kernels.cuh"
#include "bcg_kernels.cuh"
#include "tc_gemm.cuh"
#include "i8_gemm.cuh"
#include <cudaTypedefs.h>

namespace {

std::string g_create_error;

struct DevBuf {
    void* p = nullptr;
    size_t bytes = 0;
    uint64_t epoch = 0;        // hot buffers only: the arena epoch (= hot call) this carve-out belongs to
};

// Workspace arena of the hot calls ("the caller allocates every device buffer including the workspace; the library never
// allocates or frees in a hot call").  Either the caller's block (west_set_workspace) or, while none is set, a block the context owns and
// grows on demand (the documented lazy mode: growth synchronises the stream, frees and reallocates).  Every hot call starts a new epoch
// and carves its buffers from offset 0 (bump allocation, 256-byte alignment).
struct Arena {
    char* base = nullptr;
    size_t cap = 0, off = 0;
    bool user = false;
    uint64_t epoch = 0;
};

}  // namespace

struct west_ctx {
    west_cell cell{};
    cudaStream_t st = nullptr;
    HostSphere hs;
    const FftOps* ops = nullptr;
    WestGeom geom{};
    std::string err;
    int64_t launches = 0;
    int64_t dev_bytes = 0;
    int fft_chunk = 0;
    int cg_kernel = 0;                 // west_set_cg_kernel: 0 automatic, 1 always streaming
    int ms_hist = 0;                   // west_set_ms_history: 0 automatic, -1 per-shift recurrences (ms_step), 2 .. 128 fixed ring size
    std::vector<void*> owned;          // every cudaMalloc of this context

    // geometry tables
    int *d_row_off = nullptr, *d_unit_off = nullptr, *d_unit_zmax = nullptr;
    cx<double>* d_tw = nullptr;
    double* d_g2 = nullptr;

    // operator data
    double* d_vpos = nullptr;          // V_loc, position order, f64
    float* d_vpos_f = nullptr;         // same, f32 (WEST_MIXED)
    bool have_vloc = false;
    int n_proj = 0, n_occ = 0;         // n_occ: orbitals the solvers run over (WEST_GAMMA pads an odd count with one zero orbital)
    int n_occ_user = 0;                // orbitals the caller handed to west_set_states (layout of dpsi / Lanczos outputs)
    int rows_kb = 0, rows_psi = 0;     // rows of the stacked real operator matrix (x2 in WEST_FULL)
    int n_defl = 0, rows_defl = 0;     // optional deflation states (lowest conduction orbitals), stacked after the psi rows
    DevBuf A_defl, eps_defl;           // operator data (west_set_deflation)
    DevBuf dcoef_dev, eps_dev;         // operator data: device copies of D_k and eps_v
    DevBuf craw, dcoef_defl;           // hot
    long long craw_ld = 0;
    std::vector<double> h_eps_defl;
    DevBuf A_kb, A_psi;                // [rows][2 n_g] f64 each (kept apart; concatenated lazily into A_all)
    DevBuf A_all;                      // [rows_kb + rows_psi + rows_defl][2 n_g]
    // WEST_MIXED tensor path (tc_gemm.cuh): the operator matrix pre-split into TF32 hi / lo parts, row-major [rows][Kp] and transposed
    // [K][rows_p] (both k- resp. row-contiguous "K-major" operands of tcgen05.mma), built on first mixed use after a west_set_* change
    DevBuf A_hi, A_lo, AT_hi, AT_lo;
    bool tc_dirty = true;
    // WEST_FP64_I8 path (i8_gemm.cuh): the operator matrix as int8 slices, row-major [S][rows][Kp] with one power-of-two scale per row and
    // transposed [S][K][Mp] with one scale per plane-wave component k; built on first use after a west_set_* change
    DevBuf A_i8, AT_i8, A_i8_scale, AT_i8_scale;
    bool i8_dirty = true;
    bool gemm_i8 = false;              // set by every hot call from its precision argument
    int i8_slices = 8;                 // slices per operand the int8 GEMMs of the current hot call use: 8 (2^-56 of the row maxima), or 6 (2^-42) when
                                       // the CG tolerance of the call is 1e-9 or looser (west.h, WEST_FP64_I8)
    bool arena_release_ok = false;     // true only while a hot call builds operator data BEFORE carving its workspace (ensure() may then free the lazy arena)
    void* tm_encode = nullptr;         // cuTensorMapEncodeTiled (driver entry point; NULL: the mma.sync 3xTF32 kernels are used instead)
    bool A_dirty = true;
    std::vector<double> h_dcoef;       // per stacked KB row
    std::vector<double> h_eps;
    DevBuf tk;                         // [n_occ] <psi_v|T|psi_v>
    DevBuf ucache;                     // [n_uslots][N^3] c128 position order
    int n_uslots = 0;
    std::map<int, void*> dense_tw;     // twiddle tables of west_fft3d_dense, one per grid size used

    double* d_dcoef = nullptr;         // [rows_kb] D_k per stacked KB row (device copy made in west_set_kb)
    double* d_eps = nullptr;           // [n_occ] eigenvalues (device copy made in west_set_states)
    double eps_min = 0, eps_max = 0;   // extent of the occupied band (alpha_pv validation / the per-orbital default)

    // hot-call workspaces: carved from the arena at the start of every hot call (hot_begin / hot)
    Arena arena;
    DevBuf W, Cbuf, Rbuf, Xsplit, Csplit, Xi8, Ci8, Xi8_scale, Ci8_scale, vecs[4], vec5, shift, dVpos, dnpos, scal, misc, maps, xs, ps, msst, alpha_v, blk, hist, hist_scal;
    int* h_pinned = nullptr;           // pinned host scratch (64 ints): lagged convergence polls [0], [1]; reports [8..]
    cudaEvent_t ev_poll[2] = {nullptr, nullptr};

    // optional per-kernel-class timing (west_set_profile): CUDA events on the context's stream around every launch
    bool profile = false;
    std::vector<cudaEvent_t> ev_pool;
    size_t ev_used = 0;
    struct Span { size_t e0, e1; int cls; };
    std::vector<Span> spans;
};

namespace {

int fail(west_ctx* c, int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (c) c->err = buf; else g_create_error = buf;
    return code;
}
#define CK(call)                                                                                              \
    do {                                                                                                      \
        cudaError_t e_ = (call);                                                                              \
        if (e_ != cudaSuccess) return fail(c, WEST_ECUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
    } while (0)

int dev_alloc(west_ctx* c, void** p, size_t bytes) {
    *p = nullptr;
    if (bytes == 0) bytes = 16;
    cudaError_t e = cudaMalloc(p, bytes);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(c, WEST_ENOMEM, "cudaMalloc of %zu bytes failed: %s", bytes, cudaGetErrorString(e));
    }
    c->owned.push_back(*p);
    c->dev_bytes += (int64_t)bytes;
    return WEST_OK;
}
// grow-only buffer
int ensure(west_ctx* c, DevBuf& b, size_t bytes) {
    if (b.bytes >= bytes && b.p) return WEST_OK;
    if (b.p) {
        cudaStreamSynchronize(c->st);
        cudaFree(b.p);
        c->owned.erase(std::remove(c->owned.begin(), c->owned.end(), b.p), c->owned.end());
        c->dev_bytes -= (int64_t)b.bytes;
        b.p = nullptr; b.bytes = 0;
    }
    int rc = dev_alloc(c, &b.p, bytes);
    if (rc == WEST_ENOMEM && c->arena_release_ok && c->arena.base && !c->arena.user) {
        // operator data does not fit next to the context's own (lazy, grow-only) workspace of an earlier, larger call: give that block back
        // and try again - the next hot call regrows it to what it needs (never done with a caller-owned workspace)
        cudaStreamSynchronize(c->st);
        cudaFree(c->arena.base);
        c->dev_bytes -= (int64_t)c->arena.cap;
        c->arena.base = nullptr; c->arena.cap = 0; c->arena.off = 0;
        c->arena.epoch += 1;
        rc = dev_alloc(c, &b.p, bytes);
    }
    if (rc == WEST_OK) b.bytes = bytes;
    return rc;
}

inline size_t al256(size_t b) { return (std::max<size_t>(b, 16) + 255) & ~(size_t)255; }

// Start of a hot call that needs `need` bytes of workspace (the sum of al256 over its buffers).
int hot_begin(west_ctx* c, size_t need) {
    Arena& a = c->arena;
    a.epoch += 1;
    a.off = 0;
    if (need <= a.cap) return WEST_OK;
    if (a.user)
        return fail(c, WEST_EWORKSPACE, "the workspace set by west_set_workspace holds %zu bytes, this call needs %zu (west_workspace_bytes)", a.cap, need);
    // lazy mode: the context owns the arena and regrows it (synchronises the stream; documented in west.h)
    if (a.base) {
        cudaStreamSynchronize(c->st);
        cudaFree(a.base);
        c->dev_bytes -= (int64_t)a.cap;
        a.base = nullptr; a.cap = 0;
    }
    void* p = nullptr;
    cudaError_t e = cudaMalloc(&p, need);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(c, WEST_ENOMEM, "cudaMalloc of a %zu-byte workspace failed: %s", need, cudaGetErrorString(e));
    }
    a.base = (char*)p; a.cap = need;
    c->dev_bytes += (int64_t)need;
    return WEST_OK;
}
// Carve (or re-use within the same hot call) a workspace buffer.
int hot(west_ctx* c, DevBuf& b, size_t bytes) {
    Arena& a = c->arena;
    if (b.epoch == a.epoch && b.p && b.bytes >= bytes) return WEST_OK;
    const size_t n = al256(bytes);
    if (a.off + n > a.cap)
        return fail(c, WEST_EWORKSPACE, "workspace exhausted: %zu + %zu > %zu bytes (a sizing error of the library, or a workspace smaller than west_workspace_bytes)", a.off, n, a.cap);
    b.p = a.base + a.off; b.bytes = n; b.epoch = a.epoch;
    a.off += n;
    return WEST_OK;
}
// bytes the hot arena may take: the caller's block, or (lazy mode) what the device has free plus what the context's own arena holds
size_t arena_budget(const west_ctx* c) {
    if (c->arena.user) return c->arena.cap;
    size_t fr = 0, tot = 0;
    if (cudaMemGetInfo(&fr, &tot) != cudaSuccess) { cudaGetLastError(); return c->arena.cap; }
    const size_t margin = (size_t)1 << 30;      // leave 1 GB to the caller / allocator granularity
    const size_t avail = fr + c->arena.cap;
    return avail > margin ? avail - margin : 0;
}

// profiling classes
enum { PC_K1 = 0, PC_K2 = 1, PC_K3 = 2, PC_GEMM_TN = 3, PC_GEMM_UP = 4, PC_CGVEC = 5, PC_FFT_OTHER = 6, PC_MISC = 7, PC_N = 8 };
struct Prof {
    west_ctx* c; int cls; size_t e0 = 0; bool on;
    static size_t grab(west_ctx* c) {
        if (c->ev_used == c->ev_pool.size()) { cudaEvent_t e; cudaEventCreate(&e); c->ev_pool.push_back(e); }
        return c->ev_used++;
    }
    Prof(west_ctx* c_, int cls_) : c(c_), cls(cls_), on(c_->profile) {
        if (on) { e0 = grab(c); cudaEventRecord(c->ev_pool[e0], c->st); }
    }
    ~Prof() {
        if (on) { size_t e1 = grab(c); cudaEventRecord(c->ev_pool[e1], c->st); c->spans.push_back({e0, e1, cls}); }
    }
};

inline long long n3_of(const west_ctx* c) { return (long long)c->cell.N * c->cell.N * c->cell.N; }
inline bool is_gamma(const west_ctx* c) { return c->cell.mode == WEST_GAMMA; }

// ------------------------------------------------------------------------------------------ boundary conversion kernels
// position p of real-space index j along one axis: p = N2 (j mod N1) + j div N1 ;  j = p div N2 + N1 (p mod N2)
__device__ __forceinline__ int j_of_p(int p, int N1, int N2) { return p / N2 + N1 * (p % N2); }

// natural [b][ix][iy][iz] real f64 -> position order [b][pz][py][px] (T)
// xt != 0: the x position inside each line is stored transposed (index k2 N1 + k1 for position N2 k1 + k2): the V_loc layout
template <typename T>
__global__ void nat_to_pos_real(int N, int N1, int N2, long long total, const double* in, T* out, int xt = 0) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    const long long n3 = (long long)N * N * N, b = i / n3;
    long long r = i - b * n3;
    int px = (int)(r % N); r /= N;
    if (xt) px = N2 * (px % N1) + px / N1;
    const int py = (int)(r % N); const int pz = (int)(r / N);
    const int ix = j_of_p(px, N1, N2), iy = j_of_p(py, N1, N2), iz = j_of_p(pz, N1, N2);
    out[i] = (T)in[b * n3 + ((long long)ix * N + iy) * N + iz];
}
// V_loc, natural [ix][iy][iz] -> the plane kernel's layout [pz][py / LC][k2][py % LC][k1] (K2::vloc_index; px = N2 k1 + k2)
template <typename T>
__global__ void vloc_layout(int N, int N1, int N2, int LC, const double* in, T* out) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)N * N * N) return;
    long long r = i;
    const int iz = (int)(r % N); r /= N;
    const int iy = (int)(r % N); const int ix = (int)(r / N);
    const int k1 = ix % N1, k2 = ix / N1, py = N2 * (iy % N1) + iy / N1, pz = N2 * (iz % N1) + iz / N1;
    const int nch = (N + LC - 1) / LC;
    out[((((long long)pz * nch + py / LC) * N2 + k2) * LC + py % LC) * N1 + k1] = (T)in[i];
}
// position order real [b][pz][py][px] -> natural [b][ix][iy][iz]
__global__ void pos_to_nat_real(int N, int N1, int N2, long long total, const double* in, double* out, int acc = 0) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    const long long n3 = (long long)N * N * N, b = i / n3;
    long long r = i - b * n3;
    const int iz = (int)(r % N); r /= N;
    const int iy = (int)(r % N); const int ix = (int)(r / N);
    const int px = N2 * (ix % N1) + ix / N1, py = N2 * (iy % N1) + iy / N1, pz = N2 * (iz % N1) + iz / N1;
    const double v = in[b * n3 + ((long long)pz * N + py) * N + px];
    out[i] = acc ? out[i] + v : v;
}
// complex position-order slots [s][N^3] -> user grids.  gamma: real grids 2s (Re), 2s+1 (Im); full: complex grid s
__global__ void pos_to_user(int N, int N1, int N2, int gamma, int slot0, int n_slots, int n_batch, const cx<double>* R, double* out) {
    const long long n3 = (long long)N * N * N;
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n3 * n_slots) return;
    const long long s = i / n3;
    long long r = i - s * n3;
    const int iz = (int)(r % N); r /= N;
    const int iy = (int)(r % N); const int ix = (int)(r / N);
    const int px = N2 * (ix % N1) + ix / N1, py = N2 * (iy % N1) + iy / N1, pz = N2 * (iz % N1) + iz / N1;
    const cx<double> v = R[s * n3 + ((long long)pz * N + py) * N + px];
    const long long nat = ((long long)ix * N + iy) * N + iz;
    const long long gs = slot0 + s;
    if (gamma) {
        if (2 * gs < n_batch) out[(2 * gs) * n3 + nat] = v.x;
        if (2 * gs + 1 < n_batch) out[(2 * gs + 1) * n3 + nat] = v.y;
    } else {
        reinterpret_cast<cx<double>*>(out)[gs * n3 + nat] = v;
    }
}
__global__ void user_to_pos(int N, int N1, int N2, int gamma, int slot0, int n_slots, int n_batch, const double* in, cx<double>* R) {
    const long long n3 = (long long)N * N * N;
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n3 * n_slots) return;
    const long long s = i / n3;
    long long r = i - s * n3;
    const int px = (int)(r % N); r /= N;
    const int py = (int)(r % N); const int pz = (int)(r / N);
    const int ix = j_of_p(px, N1, N2), iy = j_of_p(py, N1, N2), iz = j_of_p(pz, N1, N2);
    const long long nat = ((long long)ix * N + iy) * N + iz;
    const long long gs = slot0 + s;
    cx<double> v = mk<double>(0, 0);
    if (gamma) {
        if (2 * gs < n_batch) v.x = in[(2 * gs) * n3 + nat];
        if (2 * gs + 1 < n_batch) v.y = in[(2 * gs + 1) * n3 + nat];
    } else {
        v = reinterpret_cast<const cx<double>*>(in)[gs * n3 + nat];
    }
    R[i] = v;
}

// stacked real operator rows from complex rows: FULL: row 2k = (re, im) as stored, row 2k+1 = i * row ; GAMMA: copy
__global__ void stack_rows(long long n_g, int n_rows_in, int full, const cx<double>* in, double* out) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_g * n_rows_in) return;
    const long long k = i / n_g, g = i - k * n_g;
    const cx<double> v = in[i];
    if (full) {
        double* r0 = out + (2 * k) * 2 * n_g + 2 * g;
        double* r1 = out + (2 * k + 1) * 2 * n_g + 2 * g;
        r0[0] = v.x; r0[1] = v.y;
        r1[0] = -v.y; r1[1] = v.x;
    } else {
        double* r0 = out + k * 2 * n_g + 2 * g;
        r0[0] = v.x; r0[1] = g == 0 ? 0.0 : v.y;     // c(0) of a real function is real
    }
}
// tk[v] = <psi_v|T|psi_v> over the FULL sphere
__global__ void kinetic_expect(long long n_g, int gamma, const double* g2, const cx<double>* psi, double* tk) {
    __shared__ double sh[256];
    const cx<double>* p = psi + (long long)blockIdx.x * n_g;
    double a = 0;
    for (long long g = threadIdx.x; g < n_g; g += blockDim.x) {
        const cx<double> v = p[g];
        a += g2[g] * (v.x * v.x + v.y * v.y) * ((gamma && g != 0) ? 2.0 : 1.0);
    }
    sh[threadIdx.x] = a;
    __syncthreads();
    for (int o = blockDim.x / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) tk[blockIdx.x] = sh[0];
}
__global__ void fill_shift(int n_vec, int nvpc, int n_occ, const double* eps, double* shift, const int* colmap) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n_vec) {
        int col = i / nvpc;
        if (colmap) { col = colmap[col]; if (col < 0) col = 0; }      // -1: inert padding column of a lagged compaction
        shift[i] = eps[col % n_occ];
    }
}

inline unsigned blocks_for(long long n, int t) { return (unsigned)((n + t - 1) / t); }

}  // namespace

// ===================================================================================================== internal drivers
namespace {

// slots per chunk.  Measured on B200 (profiles/r01_chunk_sweep.md): keeping a chunk's stick intermediate W inside the L2
// (48 MB chunks) is SLOWER than large chunks - the three kernels are bound by FP64 issue and shared memory, not by HBM,
// and small chunks pay wave-quantisation tails on every launch.  Default: up to 2 GB of W per chunk.
int chunk_slots(const west_ctx* c, int f32) {
    if (c->fft_chunk > 0) return c->fft_chunk;
    const size_t per_slot = (size_t)c->cell.N * c->hs.n_cols * (f32 ? 8 : 16);
    long long n = (long long)((2048ull << 20) / per_slot);
    if (n < 4) n = 4;
    if (n > 32768) n = 32768;
    return (int)n;
}
size_t bytes_W(const west_ctx* c, long long n_slots, int f32) {
    const long long n = std::max<long long>(1, std::min<long long>(chunk_slots(c, f32), n_slots));
    return (size_t)n * c->cell.N * c->hs.n_cols * (f32 ? 8 : 16);
}
int ensure_W(west_ctx* c, long long n_slots, int f32) { return hot(c, c->W, bytes_W(c, n_slots, f32)); }
size_t bytes_C(int rows, long long n_vec) { return (size_t)((rows + 3) / 4 * 4) * (size_t)((n_vec + 1) / 2 * 2) * sizeof(double); }

// opt-in to the GEMM kernels' dynamic shared memory (all four instantiations), once per process
cudaError_t gemm_attrs() {
    using namespace wgemm;
    static bool done = false;
    if (done) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(gemm_tn_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_TN);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(gemm_tn_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_TN);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(gemm_update_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_UP);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(gemm_update_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_UP);
    done = e == cudaSuccess;
    return e;
}

int launch_gemm_tn(west_ctx* c, int M, int Nn, long long K, const double* A, long long lda, const double* B, long long ldb,
                   double* C, long long ldc, int n_batch = 1, long long sA = 0, long long sB = 0, long long sC = 0, bool zero_c = true,
                   bool tf32 = false) {
    using namespace wgemm;
    if (M <= 0 || Nn <= 0) return WEST_OK;
    CK(gemm_attrs());
    const int tm = (M + BM - 1) / BM, tn = (Nn + BN - 1) / BN;
    // split K so that the CTA count fills whole waves of the 148 SMs (MINB CTAs per SM): pick the split count with
    // the best wave efficiency, each split keeping at least 32 k-steps
    const long long tiles = (long long)tm * tn * n_batch;
    const long long max_splits = std::max<long long>(1, std::min<long long>(16, K / (32 * BK)));
    long long splits = 1;
    double best = -1.0;
    for (long long sp = 1; sp <= max_splits; ++sp) {
        const double waves = (double)(tiles * sp) / (148.0 * MINB);
        const double eff = waves / std::ceil(waves) - 0.004 * (double)sp;     // mild preference for fewer splits (atomic traffic)
        if (eff > best) { best = eff; splits = sp; }
    }
    long long kps = (K + splits - 1) / splits;
    kps = (kps + BK - 1) / BK * BK;
    splits = (K + kps - 1) / kps;
    if (zero_c) CK(cudaMemsetAsync(C, 0, (size_t)M * ldc * sizeof(double), c->st));     // batched callers zero their own output
    dim3 grid(tm, tn, (unsigned)(splits * n_batch));        // row tiles fastest (gemm_f64.cuh)
    Prof prof_(c, PC_GEMM_TN);
    if (tf32) gemm_tn_kernel<true><<<grid, NTHREADS, SMEM_TN, c->st>>>(M, Nn, K, A, lda, B, ldb, C, ldc, kps, 1, (int)splits, sA, sB, sC);
    else gemm_tn_kernel<false><<<grid, NTHREADS, SMEM_TN, c->st>>>(M, Nn, K, A, lda, B, ldb, C, ldc, kps, 1, (int)splits, sA, sB, sC);
    CK(cudaGetLastError());
    c->launches += 1;
    return WEST_OK;
}
int launch_gemm_update(west_ctx* c, int M, int Nn, long long K, const double* C, long long ldc, const double* A, long long lda,
                       double* Y, long long ldy, bool tf32 = false) {
    using namespace wgemm;
    if (M <= 0 || Nn <= 0) return WEST_OK;
    CK(gemm_attrs());
    dim3 grid((unsigned)((K + BN - 1) / BN), (unsigned)((Nn + BM - 1) / BM));
    Prof prof_(c, PC_GEMM_UP);
    if (tf32) gemm_update_kernel<true><<<grid, NTHREADS, SMEM_UP, c->st>>>(M, Nn, K, C, ldc, A, lda, Y, ldy);
    else gemm_update_kernel<false><<<grid, NTHREADS, SMEM_UP, c->st>>>(M, Nn, K, C, ldc, A, lda, Y, ldy);
    CK(cudaGetLastError());
    c->launches += 1;
    return WEST_OK;
}

// (re)build the concatenated operator matrix [KB rows ; psi rows ; deflation rows] (operator data: grown outside the hot arena, only
// after a west_set_* call changed it)
int ensure_opmatrix(west_ctx* c) {
    const long long K = 2 * c->hs.n_g;
    const int rows = c->rows_kb + c->rows_psi + c->rows_defl;
    if (rows == 0 || !c->A_dirty) return WEST_OK;
    int rc = ensure(c, c->A_all, (size_t)rows * K * sizeof(double));
    if (rc) return rc;
    if (c->rows_kb) CK(cudaMemcpyAsync(c->A_all.p, c->A_kb.p, (size_t)c->rows_kb * K * sizeof(double), cudaMemcpyDeviceToDevice, c->st));
    if (c->rows_psi)
        CK(cudaMemcpyAsync((double*)c->A_all.p + (size_t)c->rows_kb * K, c->A_psi.p, (size_t)c->rows_psi * K * sizeof(double),
                           cudaMemcpyDeviceToDevice, c->st));
    if (c->rows_defl)
        CK(cudaMemcpyAsync((double*)c->A_all.p + (size_t)(c->rows_kb + c->rows_psi) * K, c->A_defl.p,
                           (size_t)c->rows_defl * K * sizeof(double), cudaMemcpyDeviceToDevice, c->st));
    c->A_dirty = false;
    return WEST_OK;
}

// coefficients of the low-rank terms (applied by wcg::lowrank_fix to the overlap block C[m][n]):
//   rows [0, n_rows_d) of the block take dcoef[m] (the KB D_k); the remaining rows (psi / deflation rows) take alpha_vec[orbital of
//   column n] if alpha_vec is given, else the constant alpha_const (RHS projection: -1)
struct LowrankCoef {
    const double* dcoef = nullptr; int n_rows_d = 0;
    double alpha_const = 0.0; const double* alpha_vec = nullptr; const int* colmap = nullptr; int nvpc = 1, n_occ = 1;
};

// ---- WEST_MIXED tensor path (tcgen05 kind::tf32, tc_gemm.cuh)
inline long long pad4(long long n) { return (n + 3) / 4 * 4; }
bool tc_available(const west_ctx* c) { return c->tm_encode != nullptr; }
size_t tc_hot_bytes(const west_ctx* c, int rows, long long n_vec) {       // Xsplit + Csplit of one lowrank_apply
    if (!tc_available(c) || rows <= 0) return 0;
    const long long Kp = pad4(2 * c->hs.n_g), rp = pad4(rows);
    return al256(sizeof(float) * 2 * (size_t)n_vec * Kp) + al256(sizeof(float) * 2 * (size_t)n_vec * rp);
}
// (k, batch, row) tensor map: element (k, b, r) at p[r * ld + b * ldb + k]; box {BK, 1, 128}, 128-byte swizzle, zero fill out of bounds
int tc_map(west_ctx* c, CUtensorMap* m, const float* p, long long rows, long long cols, long long ld, long long n_batch = 1, long long ldb = 0) {
    if (n_batch == 1) ldb = rows * ld;
    cuuint64_t gdim[3] = {(cuuint64_t)cols, (cuuint64_t)n_batch, (cuuint64_t)rows};
    cuuint64_t gstr[2] = {(cuuint64_t)ldb * sizeof(float), (cuuint64_t)ld * sizeof(float)};
    cuuint32_t box[3] = {(cuuint32_t)wtc::BK, 1, (cuuint32_t)wtc::BM}, es[3] = {1, 1, 1};
    const CUresult r = reinterpret_cast<PFN_cuTensorMapEncodeTiled_v12000>(c->tm_encode)(
        m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void*)p, gdim, gstr, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
        CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(c, WEST_ECUDA, "cuTensorMapEncodeTiled failed (%d) for a %lld x %lld x %lld map", (int)r, rows, n_batch, cols);
    return WEST_OK;
}
// operator data of the tensor path: (re)split the stacked operator matrix after a west_set_* change (not a hot-arena buffer)
int ensure_tc_operator(west_ctx* c) {
    if (!c->tc_dirty) return WEST_OK;
    const long long K = 2 * c->hs.n_g, Kp = pad4(K);
    const int rows = c->rows_kb + c->rows_psi + c->rows_defl;
    const long long rp = pad4(rows);
    int rc;
    if ((rc = ensure(c, c->A_hi, sizeof(float) * (size_t)rows * Kp))) return rc;
    if ((rc = ensure(c, c->A_lo, sizeof(float) * (size_t)rows * Kp))) return rc;
    if ((rc = ensure(c, c->AT_hi, sizeof(float) * (size_t)K * rp))) return rc;
    if ((rc = ensure(c, c->AT_lo, sizeof(float) * (size_t)K * rp))) return rc;
    const double* A = (const double*)c->A_all.p;
    wtc::split_rows<<<blocks_for((long long)rows * Kp, 256), 256, 0, c->st>>>(rows, K, A, K, (float*)c->A_hi.p, (float*)c->A_lo.p, Kp);
    wtc::split_rows_transposed<<<dim3((unsigned)((K + 31) / 32), (unsigned)((rp + 31) / 32)), dim3(32, 8), 0, c->st>>>(rows, K, A, K, (float*)c->AT_hi.p,
                                                                                                                   (float*)c->AT_lo.p, rp);
    CK(cudaGetLastError());
    c->launches += 2;
    c->tc_dirty = false;
    return WEST_OK;
}
cudaError_t tc_attrs() {
    static bool done = false;
    if (done) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(wtc::tf32x3_gemm<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)wtc::SMEM_BYTES);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(wtc::tf32x3_gemm<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)wtc::SMEM_BYTES);
    done = e == cudaSuccess;
    return e;
}
// rows [0, nr) of the operator matrix on the tensor path:  Y += A^T (coef . fix(A X^T))
int lowrank_apply_tc(west_ctx* c, int nr, int n_vec, const double* X, double* Y, const LowrankCoef& lc) {
    const long long K = 2 * c->hs.n_g, Kp = pad4(K), rp = pad4(nr);
    const int rows_all = c->rows_kb + c->rows_psi + c->rows_defl;
    const long long rp_all = pad4(rows_all);
    int rc;
    CK(tc_attrs());
    if ((rc = ensure_tc_operator(c))) return rc;
    if ((rc = hot(c, c->Xsplit, sizeof(float) * 2 * (size_t)n_vec * Kp))) return rc;
    if ((rc = hot(c, c->Csplit, sizeof(float) * 2 * (size_t)n_vec * rp))) return rc;
    if ((rc = hot(c, c->Cbuf, bytes_C(nr, n_vec)))) return rc;
    float* Xh = (float*)c->Xsplit.p; float* Xl = Xh + (size_t)n_vec * Kp;
    float* Ch = (float*)c->Csplit.p; float* Cl = Ch + (size_t)n_vec * rp;
    double* Ct = (double*)c->Cbuf.p;                       // [n_vec][rp] (transposed overlap block, rows contiguous)
    wtc::Maps m1, m2;
    if ((rc = tc_map(c, &m1.a_hi, (const float*)c->A_hi.p, nr, K, Kp)) || (rc = tc_map(c, &m1.a_lo, (const float*)c->A_lo.p, nr, K, Kp)) ||
        (rc = tc_map(c, &m1.b_hi, Xh, n_vec, K, Kp)) || (rc = tc_map(c, &m1.b_lo, Xl, n_vec, K, Kp)) ||
        (rc = tc_map(c, &m2.a_hi, (const float*)c->AT_hi.p, K, nr, rp_all)) || (rc = tc_map(c, &m2.a_lo, (const float*)c->AT_lo.p, K, nr, rp_all)) ||
        (rc = tc_map(c, &m2.b_hi, Ch, n_vec, nr, rp)) || (rc = tc_map(c, &m2.b_lo, Cl, n_vec, nr, rp)))
        return rc;
    {
        Prof p_(c, PC_GEMM_TN);
        wtc::split_rows<<<blocks_for((long long)n_vec * Kp, 256), 256, 0, c->st>>>(n_vec, K, X, K, Xh, Xl, Kp);
        CK(cudaMemsetAsync(Ct, 0, sizeof(double) * (size_t)n_vec * rp, c->st));
        const int n_kb = (int)((K + wtc::BK - 1) / wtc::BK);
        const long long tiles = (long long)((nr + 127) / 128) * ((n_vec + 127) / 128);
        int splits = (int)std::max<long long>(1, std::min<long long>(n_kb / 16, (148 * 2 + tiles - 1) / tiles));
        int kps = (n_kb + splits - 1) / splits;
        splits = (n_kb + kps - 1) / kps;
        const wtc::TileGrid tg{(nr + 127) / 128, (n_vec + 127) / 128, splits, 1, 0};
        const long long nt = (long long)tg.tiles_a * tg.tiles_b * tg.splits;
        wtc::tf32x3_gemm<true><<<(unsigned)std::min<long long>(nt, 148), wtc::NTHREADS, wtc::SMEM_BYTES, c->st>>>(m1, tg, nr, n_vec, n_kb, kps, Ct, rp);
        CK(cudaGetLastError());
        c->launches += 2;
    }
    wcg::lowrank_fix_split<<<blocks_for((long long)n_vec * rp, 256), 256, 0, c->st>>>(nr, n_vec, rp, Ct, (const double*)c->A_all.p, K, X, K, lc.dcoef, lc.n_rows_d,
                                                                               lc.alpha_const, lc.alpha_vec, lc.colmap, lc.nvpc, lc.n_occ, is_gamma(c) ? 1 : 0, Ch, Cl);
    CK(cudaGetLastError());
    c->launches += 1;
    {
        Prof p_(c, PC_GEMM_UP);
        const int n_kb = (nr + wtc::BK - 1) / wtc::BK;
        const wtc::TileGrid tg{(int)((K + 127) / 128), (n_vec + 127) / 128, 1, 1, 0};
        const long long nt = (long long)tg.tiles_a * tg.tiles_b;
        wtc::tf32x3_gemm<false><<<(unsigned)std::min<long long>(nt, 148), wtc::NTHREADS, wtc::SMEM_BYTES, c->st>>>(m2, tg, (int)K, n_vec, n_kb, n_kb, Y, K);
        CK(cudaGetLastError());
        c->launches += 1;
    }
    return WEST_OK;
}

// ---- WEST_FP64_I8 tensor path (tcgen05 kind::i8, i8_gemm.cuh): FP64-accurate products from error-free int8 slices
constexpr int I8S = 8;                                       // slices per operand: 56 bits below every row's largest element
inline long long pad64(long long n) { return (n + 63) / 64 * 64; }
size_t i8_hot_bytes(const west_ctx* c, int rows, long long n_vec) {       // X slices + scales, C slices + scales of one low-rank apply
    if (!tc_available(c) || rows <= 0) return 0;
    const long long Kp = pad64(2 * c->hs.n_g), Mp = pad64(rows);
    return al256((size_t)I8S * n_vec * Kp) + al256((size_t)I8S * n_vec * Mp) + 2 * al256(sizeof(double) * (size_t)n_vec);
}
// (k byte, slice, row) tensor map over slices [S][rows_alloc][ld]: the first k_extent bytes of the first `rows` rows; box {64, 1, 128},
// 64-byte swizzle, zero fill out of bounds (so a contraction over the first k_extent entries of longer rows is exact)
int i8_map(west_ctx* c, CUtensorMap* m, const signed char* p, long long rows, long long rows_alloc, long long k_extent, long long ld) {
    const long long Kp = k_extent;
    cuuint64_t gdim[3] = {(cuuint64_t)k_extent, (cuuint64_t)I8S, (cuuint64_t)rows};
    cuuint64_t gstr[2] = {(cuuint64_t)(rows_alloc * ld), (cuuint64_t)ld};
    cuuint32_t box[3] = {(cuuint32_t)wi8::BKB, 1, (cuuint32_t)wi8::BM}, es[3] = {1, 1, 1};
    const CUresult r = reinterpret_cast<PFN_cuTensorMapEncodeTiled_v12000>(c->tm_encode)(
        m, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, (void*)p, gdim, gstr, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_64B,
        CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(c, WEST_ECUDA, "cuTensorMapEncodeTiled failed (%d) for an int8 slice map of %lld x %lld", (int)r, rows, Kp);
    return WEST_OK;
}
cudaError_t i8_attrs() {
    static bool done = false;
    if (done) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(wi8::i8_slice_gemm<I8S, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)wi8::Sched<I8S>::SMEM_BYTES);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(wi8::i8_slice_gemm<I8S, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)wi8::Sched<I8S>::SMEM_BYTES);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(wi8::i8_slice_gemm<6, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)wi8::Sched<6>::SMEM_BYTES);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(wi8::i8_slice_gemm<6, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)wi8::Sched<6>::SMEM_BYTES);
    done = e == cudaSuccess;
    return e;
}
// out[c * ldo + r] += sum_k A[r][k] B[c][k] from slice arrays (both [S][rows_alloc][Kp], scales per row).  atomic: split along k (the
// caller zeroes out); else every element is owned by one CTA (read-modify-write).
int launch_i8_gemm(west_ctx* c, bool atomic, int rows_a, long long alloc_a, long long ld_a, const signed char* A, const double* sa, int rows_b, long long alloc_b,
                   long long ld_b, const signed char* B, const double* sb, long long Kp /* contraction length */, double* out, long long ldo, int prof_class) {
    if (rows_a <= 0 || rows_b <= 0) return WEST_OK;
    int rc;
    CK(i8_attrs());
    wi8::Maps m;
    if ((rc = i8_map(c, &m.a, A, rows_a, alloc_a, std::min(Kp, ld_a), ld_a)) || (rc = i8_map(c, &m.b, B, rows_b, alloc_b, std::min(Kp, ld_b), ld_b))) return rc;
    const int n_kb = (int)((Kp + wi8::BKB - 1) / wi8::BKB);
    const long long tiles = (long long)((rows_a + 127) / 128) * ((rows_b + 127) / 128);
    int splits = 1;
    if (atomic) {
        // exactness of the int32 sums bounds a split's k range; beyond that, splits only to give every SM a tile
        const int need = (int)((Kp + wi8::MAX_K_PER_SPLIT - 1) / wi8::MAX_K_PER_SPLIT);
        // and k chunks of ~8 KB per slice row: the operator chunk all tiles of a split share then stays closer to the L2 (measured at the cfg-5
        // shape: 153.5 ms with 3 splits, 134-136 ms with 12-40)
        splits = (int)std::max<long long>(need, std::min<long long>(n_kb / 32, std::max<long long>((Kp + 8191) / 8192, (148 + tiles - 1) / tiles)));
        splits = std::max(1, splits);
    } else if (Kp > wi8::MAX_K_PER_SPLIT) {
        return fail(c, WEST_EINVAL, "int8 slice GEMM: contraction length %lld exceeds the exact int32 range of an unsplit product", Kp);
    }
    int kps = (n_kb + splits - 1) / splits;
    splits = (n_kb + kps - 1) / kps;
    // update product (rows_a = 2 n_g rows of the transposed operator): vector tiles in groups, else every CTA streams its own operator tile
    // from DRAM once per vector tile; overlap product: few operator tiles, small groups
    // (measured at the cfg-5 shape: update product 190 ms with the operator tiles fastest, 142-148 ms with groups of 4-16 vector tiles)
    const int gb = atomic ? 4 : 6;
    const wi8::TileGrid tg{(rows_a + 127) / 128, (rows_b + 127) / 128, splits, gb};
    const long long nt = tiles * splits;
    Prof p_(c, prof_class);
    const unsigned grid = (unsigned)std::min<long long>(nt, 148);
    if (c->i8_slices == 6) {           // the slice arrays always hold 8 planes; the 6-slice schedule touches the first six
        if (atomic) wi8::i8_slice_gemm<6, true><<<grid, wi8::NTHREADS, wi8::Sched<6>::SMEM_BYTES, c->st>>>(m, tg, rows_a, rows_b, n_kb, kps, sa, sb, out, ldo);
        else wi8::i8_slice_gemm<6, false><<<grid, wi8::NTHREADS, wi8::Sched<6>::SMEM_BYTES, c->st>>>(m, tg, rows_a, rows_b, n_kb, kps, sa, sb, out, ldo);
    } else {
        if (atomic) wi8::i8_slice_gemm<I8S, true><<<grid, wi8::NTHREADS, wi8::Sched<I8S>::SMEM_BYTES, c->st>>>(m, tg, rows_a, rows_b, n_kb, kps, sa, sb, out, ldo);
        else wi8::i8_slice_gemm<I8S, false><<<grid, wi8::NTHREADS, wi8::Sched<I8S>::SMEM_BYTES, c->st>>>(m, tg, rows_a, rows_b, n_kb, kps, sa, sb, out, ldo);
    }
    CK(cudaGetLastError());
    c->launches += 1;
    return WEST_OK;
}
// operator data of the int8 path: (re)slice the stacked operator matrix after a west_set_* change (not a hot-arena buffer)
int ensure_i8_operator(west_ctx* c) {
    if (!c->i8_dirty) return WEST_OK;
    const long long K = 2 * c->hs.n_g, Kp = pad64(K);
    const int rows = c->rows_kb + c->rows_psi + c->rows_defl;
    const long long Mp = pad64(rows);
    int rc;
    if ((rc = ensure(c, c->A_i8, (size_t)I8S * rows * Kp))) return rc;
    if ((rc = ensure(c, c->AT_i8, (size_t)I8S * K * Mp))) return rc;
    if ((rc = ensure(c, c->A_i8_scale, sizeof(double) * (size_t)rows))) return rc;
    if ((rc = ensure(c, c->AT_i8_scale, sizeof(double) * (size_t)K))) return rc;
    const double* A = (const double*)c->A_all.p;
    wi8::slice_rows<I8S><<<rows, 256, 0, c->st>>>(K, A, K, (signed char*)c->A_i8.p, rows, Kp, (double*)c->A_i8_scale.p);
    wi8::col_absmax<<<blocks_for(K, 256), 256, 0, c->st>>>(rows, K, A, K, (double*)c->AT_i8_scale.p);
    wi8::slice_rows_transposed<I8S><<<dim3((unsigned)((K + 31) / 32), (unsigned)((Mp + 31) / 32)), dim3(32, 8), 0, c->st>>>(rows, K, A, K, (const double*)c->AT_i8_scale.p,
                                                                                                                    (signed char*)c->AT_i8.p, Mp);
    CK(cudaGetLastError());
    c->launches += 3;
    c->i8_dirty = false;
    return WEST_OK;
}
// rows [0, nr) of the operator matrix on the int8 path:  Y += A^T (coef . fix(A X^T))
int lowrank_apply_i8(west_ctx* c, int nr, int n_vec, const double* X, double* Y, const LowrankCoef& lc) {
    const long long K = 2 * c->hs.n_g, Kp = pad64(K), Mp = pad64(nr);
    const int rows_all = c->rows_kb + c->rows_psi + c->rows_defl;
    const long long Mp_all = pad64(rows_all), rp = pad4(nr);
    int rc;
    if ((rc = ensure_i8_operator(c))) return rc;
    if ((rc = hot(c, c->Xi8, (size_t)I8S * n_vec * Kp))) return rc;
    if ((rc = hot(c, c->Ci8, (size_t)I8S * n_vec * Mp))) return rc;
    if ((rc = hot(c, c->Xi8_scale, sizeof(double) * (size_t)n_vec))) return rc;
    if ((rc = hot(c, c->Ci8_scale, sizeof(double) * (size_t)n_vec))) return rc;
    if ((rc = hot(c, c->Cbuf, bytes_C(nr, n_vec)))) return rc;
    double* Ct = (double*)c->Cbuf.p;                       // [n_vec][rp] (transposed overlap block, rows contiguous)
    {
        Prof p_(c, PC_GEMM_TN);
        if (c->i8_slices == 6) wi8::slice_rows<6><<<n_vec, 256, 0, c->st>>>(K, X, K, (signed char*)c->Xi8.p, n_vec, Kp, (double*)c->Xi8_scale.p);
        else wi8::slice_rows<I8S><<<n_vec, 256, 0, c->st>>>(K, X, K, (signed char*)c->Xi8.p, n_vec, Kp, (double*)c->Xi8_scale.p);
        CK(cudaMemsetAsync(Ct, 0, sizeof(double) * (size_t)n_vec * rp, c->st));
        CK(cudaGetLastError());
        c->launches += 1;
    }
    if ((rc = launch_i8_gemm(c, true, nr, rows_all, Kp, (const signed char*)c->A_i8.p, (const double*)c->A_i8_scale.p, n_vec, n_vec, Kp, (const signed char*)c->Xi8.p,
                             (const double*)c->Xi8_scale.p, K, Ct, rp, PC_GEMM_TN)))
        return rc;
    {
        Prof p_(c, PC_GEMM_UP);
        wcg::lowrank_fix_t<<<blocks_for((long long)n_vec * rp, 256), 256, 0, c->st>>>(nr, n_vec, rp, Ct, (const double*)c->A_all.p, K, X, K, lc.dcoef, lc.n_rows_d,
                                                                                 lc.alpha_const, lc.alpha_vec, lc.colmap, lc.nvpc, lc.n_occ, is_gamma(c) ? 1 : 0);
        if (c->i8_slices == 6) wi8::slice_rows<6><<<n_vec, 256, 0, c->st>>>(nr, Ct, rp, (signed char*)c->Ci8.p, n_vec, Mp, (double*)c->Ci8_scale.p);
        else wi8::slice_rows<I8S><<<n_vec, 256, 0, c->st>>>(nr, Ct, rp, (signed char*)c->Ci8.p, n_vec, Mp, (double*)c->Ci8_scale.p);
        CK(cudaGetLastError());
        c->launches += 2;
    }
    // Y[n][k] += sum_m C[m][n] A[m][k]: k on the TMEM lanes (operator transposed, scale per k), vectors on the columns
    return launch_i8_gemm(c, false, (int)K, K, Mp_all, (const signed char*)c->AT_i8.p, (const double*)c->AT_i8_scale.p, n_vec, n_vec, Mp, (const signed char*)c->Ci8.p,
                          (const double*)c->Ci8_scale.p, nr, Y, K, PC_GEMM_UP);
}

// Y += sum_{m in [r0, r0+nr)} coef_m A_m <A_m, X>   for n_vec real-function / complex vectors (as 2 n_g reals each).
// tf32: the WEST_MIXED path of H*psi (3xTF32 tensor-core products, FP32 class) - never the RHS projection or the deflation.
// On Blackwell the tf32 products run on tcgen05 (lowrank_apply_tc); the warp-level mma.sync kernels remain as the path taken when the
// driver offers no tensor-map encoder.
int lowrank_apply(west_ctx* c, int r0, int nr, int n_vec, const double* X, double* Y, const LowrankCoef& lc, bool tf32 = false) {
    if (nr <= 0 || n_vec <= 0) return WEST_OK;
    if (tf32 && r0 == 0 && tc_available(c)) return lowrank_apply_tc(c, nr, n_vec, X, Y, lc);
    if (c->gemm_i8 && !tf32 && r0 == 0 && tc_available(c)) return lowrank_apply_i8(c, nr, n_vec, X, Y, lc);
    const long long K = 2 * c->hs.n_g;
    const long long ldc = (n_vec + 1) / 2 * 2;
    int rc = hot(c, c->Cbuf, bytes_C(nr, n_vec));
    if (rc) return rc;
    const double* A = (const double*)c->A_all.p + (size_t)r0 * K;
    double* C = (double*)c->Cbuf.p;
    rc = launch_gemm_tn(c, nr, n_vec, K, A, K, X, K, C, ldc, 1, 0, 0, 0, true, tf32);
    if (rc) return rc;
    wcg::lowrank_fix<<<blocks_for((long long)nr * n_vec, 256), 256, 0, c->st>>>(nr, n_vec, ldc, C, A, K, X, K, lc.dcoef, lc.n_rows_d, lc.alpha_const,
                                                                             lc.alpha_vec, lc.colmap, lc.nvpc, lc.n_occ, is_gamma(c) ? 1 : 0);
    CK(cudaGetLastError());
    c->launches += 1;
    return launch_gemm_update(c, nr, n_vec, K, C, ldc, A, K, Y, K, tf32);
}

// local part of (H - shift - i omega) on vectors: Y = T x + V_loc x - shift x -+ omega terms   (no KB, no P_v)
int hloc_apply(west_ctx* c, int f32, VecMap vm, int n_slots, const cx<double>* X, cx<double>* Y, const double* shift, double omega) {
    const int chunk = chunk_slots(c, f32);
    int rc = ensure_W(c, std::min(chunk, n_slots), f32);
    if (rc) return rc;
    const int N = c->cell.N;
    K3Epi e;
    e.scale = 1.0 / ((double)N * N * N); e.kinetic = 1; e.shift = shift; e.omega = omega; e.X = X;
    K2Any a{};
    a.W = c->W.p; a.V = f32 ? (const void*)c->d_vpos_f : (const void*)c->d_vpos;
    for (int s0 = 0; s0 < n_slots; s0 += chunk) {
        const int ns = std::min(chunk, n_slots - s0);
        vm.slot0 = s0;
        { Prof p_(c, PC_K1); CK(c->ops->k1(f32, is_gamma(c), ns, c->st, c->geom, vm, X, c->W.p)); }
        { Prof p_(c, PC_K2); CK(c->ops->k2(f32, K2_H, ns, c->st, c->geom, a)); }
        { Prof p_(c, PC_K3); CK(c->ops->k3(f32, is_gamma(c), ns, c->st, c->geom, vm, c->W.p, e, Y)); }
        c->launches += 3;
    }
    return WEST_OK;
}

// ---- workspace plans: the sum of al256(bytes) over the buffers a hot call carves (west_workspace_bytes returns exactly these)
int fft3d_chunk(const west_ctx* c, int n_slots) { return std::max(1, std::min(n_slots, std::min(chunk_slots(c, 0), 64))); }
size_t plan_fft3d(const west_ctx* c, int n_batch) {
    const int n_slots = is_gamma(c) ? (n_batch + 1) / 2 : n_batch;
    const int chunk = fft3d_chunk(c, n_slots);
    return al256(bytes_W(c, chunk, 0)) + al256(sizeof(cx<double>) * (size_t)n3_of(c) * chunk);
}
size_t plan_lanczos(const west_ctx* c, int n_pert, int n_steps, int f32) {
    const size_t n_col = (size_t)n_pert * c->n_occ;
    const long long slots_h = is_gamma(c) ? ((long long)n_col + 1) / 2 : (long long)n_col, slots_r = (long long)n_pert * c->n_uslots;
    size_t t = 4 * al256(sizeof(cx<double>) * (size_t)c->hs.n_g * n_col) + al256(sizeof(double) * (size_t)n3_of(c) * n_pert) + al256(sizeof(double) * n_col + 64) +
               al256(bytes_W(c, std::max(slots_h, slots_r), 0)) + al256(256);
    if (c->rows_kb > 0) t += al256(bytes_C(c->rows_kb, (long long)n_col)) + (f32 ? tc_hot_bytes(c, c->rows_kb, (long long)n_col) : 0);
    if (c->n_occ_user != c->n_occ) t += al256(sizeof(double) * n_col * (2 * (size_t)n_steps + 1));
    if (f32 && tc_available(c)) t += al256(sizeof(float) * 4 * n_col * (size_t)pad4(2 * c->hs.n_g));      // TF32 splits of q^1 and q^l (brakets)
    return t;
}
size_t plan_happly(const west_ctx* c, long long n_vec, int f32, int i8 = 0) {
    const long long n_slots = is_gamma(c) ? (n_vec + 1) / 2 : n_vec;
    return al256(bytes_W(c, n_slots, f32)) +
           (c->rows_kb > 0 ? al256(bytes_C(c->rows_kb, n_vec)) + (f32 ? tc_hot_bytes(c, c->rows_kb, n_vec) : (i8 ? i8_hot_bytes(c, c->rows_kb, n_vec) : 0)) : 0);
}

}  // namespace

// ============================================================================================================ public API
extern "C" {

const char* west_last_error(const west_ctx* c) { return c ? c->err.c_str() : g_create_error.c_str(); }
int64_t west_device_bytes(const west_ctx* c) { return c ? c->dev_bytes : 0; }
int64_t west_launch_count(const west_ctx* c) { return c ? c->launches : 0; }
int west_set_profile(west_ctx* c, int32_t on) {
    if (!c) return WEST_EINVAL;
    c->profile = on != 0;
    return WEST_OK;
}
int west_get_profile(west_ctx* c, double* ms, int64_t* count) {
    if (!c || !ms || !count) return WEST_EINVAL;
    cudaStreamSynchronize(c->st);
    for (int i = 0; i < PC_N; ++i) { ms[i] = 0; count[i] = 0; }
    for (const auto& sp : c->spans) {
        float t = 0;
        cudaEventElapsedTime(&t, c->ev_pool[sp.e0], c->ev_pool[sp.e1]);
        ms[sp.cls] += t; count[sp.cls] += 1;
    }
    c->spans.clear();
    c->ev_used = 0;
    return WEST_OK;
}
int west_set_cg_kernel(west_ctx* c, int32_t which) {
    if (!c || which < 0 || which > 2) return WEST_EINVAL;
    c->cg_kernel = which;
    return WEST_OK;
}
int west_set_ms_history(west_ctx* c, int32_t slots) {
    if (!c || slots < -1 || slots == 1 || slots > wcg::MSH_HMAX) return fail(c, WEST_EINVAL, "west_set_ms_history: slots must be -1, 0 or 2 .. %d", wcg::MSH_HMAX);
    c->ms_hist = slots;
    return WEST_OK;
}
int west_set_fft_chunk(west_ctx* c, int32_t n) {
    if (!c || n < 0 || n > 65535) return WEST_EINVAL;
    c->fft_chunk = n;
    return WEST_OK;
}

int west_create(west_ctx** out, const west_cell* cell, void* stream) {
    west_ctx* c = nullptr;
    if (!out || !cell) return fail(c, WEST_EINVAL, "west_create: NULL argument");
    *out = nullptr;
    const FftOps* ops = nullptr;
    switch (cell->N) {
        case 24: ops = west_fft_ops_24(); break;
        case 36: ops = west_fft_ops_36(); break;
        case 48: ops = west_fft_ops_48(); break;
        case 72: ops = west_fft_ops_72(); break;
        case 144: ops = west_fft_ops_144(); break;
        default: return fail(c, WEST_EINVAL, "west_create: unsupported N = %d (supported: 24, 36, 48, 72, 144)", cell->N);
    }
    if (cell->n2max < 0 || !(cell->L > 0) || (cell->mode != WEST_FULL && cell->mode != WEST_GAMMA))
        return fail(c, WEST_EINVAL, "west_create: bad cell (L = %g, n2max = %d, mode = %d)", cell->L, cell->n2max, cell->mode);
    if (cell->N < 4 * isqrt_floor(cell->n2max) + 1)
        return fail(c, WEST_EINVAL, "west_create: N = %d < 4*floor(sqrt(n2max)) + 1 = %d", cell->N, 4 * isqrt_floor(cell->n2max) + 1);
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(c, WEST_ECUDA, "west_create: no CUDA device (%s); this library has no CPU fallback", cudaGetErrorString(e));
    }
    west_ctx* ctx = new west_ctx();
    ctx->cell = *cell;
    ctx->st = (cudaStream_t)stream;
    ctx->ops = ops;
    ctx->hs = build_sphere(cell->n2max, cell->N, cell->mode == WEST_GAMMA, cell->L);
    c = ctx;
    auto bail = [&](int rc) { g_create_error = ctx->err; west_destroy(ctx); return rc; };
    const HostSphere& s = ctx->hs;
    int rc;
    if ((rc = dev_alloc(c, (void**)&c->d_row_off, sizeof(int) * (s.nr + 1)))) return bail(rc);
    if ((rc = dev_alloc(c, (void**)&c->d_unit_off, sizeof(int) * s.n_units))) return bail(rc);
    if ((rc = dev_alloc(c, (void**)&c->d_unit_zmax, sizeof(int) * s.n_units))) return bail(rc);
    if ((rc = dev_alloc(c, (void**)&c->d_tw, sizeof(cx<double>) * s.N))) return bail(rc);
    if ((rc = dev_alloc(c, (void**)&c->d_g2, sizeof(double) * s.n_g))) return bail(rc);
    std::vector<cx<double>> tw(s.N);
    for (int i = 0; i < s.N; ++i) {
        const double a = 2.0 * 3.14159265358979323846264338327950288 * (double)i / (double)s.N;
        tw[i].x = std::cos(a); tw[i].y = std::sin(a);
    }
    // exact values on the axes
    tw[0] = mk<double>(1, 0);
    if (s.N % 4 == 0) { tw[s.N / 4] = mk<double>(0, 1); tw[3 * s.N / 4] = mk<double>(0, -1); }
    if (s.N % 2 == 0) tw[s.N / 2] = mk<double>(-1, 0);
    e = cudaMemcpy(c->d_row_off, s.row_off.data(), sizeof(int) * (s.nr + 1), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(c->d_unit_off, s.unit_off.data(), sizeof(int) * s.n_units, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(c->d_unit_zmax, s.unit_zmax.data(), sizeof(int) * s.n_units, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(c->d_tw, tw.data(), sizeof(cx<double>) * s.N, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(c->d_g2, s.g2.data(), sizeof(double) * s.n_g, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMallocHost((void**)&c->h_pinned, 64 * sizeof(int));
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_poll[0], cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_poll[1], cudaEventDisableTiming);
    if (e != cudaSuccess) { fail(c, WEST_ECUDA, "west_create: %s", cudaGetErrorString(e)); return bail(WEST_ECUDA); }
    {
        cudaDriverEntryPointQueryResult q;
        void* fn = nullptr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess) c->tm_encode = fn;
        else cudaGetLastError();
    }
    // twiddle tables of west_fft3d_dense (all three grid sizes, 7 KB): no allocation in the hot call
    for (int n : {64, 128, 256}) {
        std::vector<cx<double>> dtw(n);
        for (int i = 0; i < n; ++i) {
            const double a = 2.0 * 3.14159265358979323846264338327950288 * (double)i / (double)n;
            dtw[i].x = std::cos(a); dtw[i].y = std::sin(a);
        }
        dtw[0] = mk<double>(1, 0); dtw[n / 4] = mk<double>(0, 1); dtw[n / 2] = mk<double>(-1, 0); dtw[3 * n / 4] = mk<double>(0, -1);
        void* d = nullptr;
        if ((rc = dev_alloc(c, &d, sizeof(cx<double>) * n))) return bail(rc);
        if (cudaMemcpy(d, dtw.data(), sizeof(cx<double>) * n, cudaMemcpyHostToDevice) != cudaSuccess) { fail(c, WEST_ECUDA, "west_create: twiddle copy"); return bail(WEST_ECUDA); }
        c->dense_tw.emplace(n, d);
    }
    WestGeom& g = c->geom;
    g.N = s.N; g.n_max = s.n_max; g.nr = s.nr; g.n_cols = s.n_cols; g.n_units = s.n_units; g.gamma = s.gamma; g.n_g = s.n_g;
    g.row_off = c->d_row_off; g.unit_off = c->d_unit_off; g.unit_zmax = c->d_unit_zmax; g.tw = c->d_tw; g.g2 = c->d_g2;
    *out = ctx;
    return WEST_OK;
}

int west_destroy(west_ctx* c) {
    if (!c) return WEST_OK;
    cudaStreamSynchronize(c->st);
    for (void* p : c->owned) cudaFree(p);
    if (c->arena.base && !c->arena.user) cudaFree(c->arena.base);
    for (cudaEvent_t e : c->ev_pool) cudaEventDestroy(e);
    for (cudaEvent_t e : c->ev_poll) if (e) cudaEventDestroy(e);
    if (c->h_pinned) cudaFreeHost(c->h_pinned);
    delete c;
    return WEST_OK;
}

int west_gsphere(const west_ctx* cc, int64_t* n_g, int32_t* miller, int32_t* fft_index, int32_t* fft_index_minus, double* g2) {
    west_ctx* c = const_cast<west_ctx*>(cc);
    if (!c) return WEST_EINVAL;
    const HostSphere& s = c->hs;
    if (n_g) *n_g = s.n_g;
    if (miller) std::memcpy(miller, s.miller.data(), sizeof(int32_t) * 3 * s.n_g);
    if (g2) std::memcpy(g2, s.g2.data(), sizeof(double) * s.n_g);
    const int N = s.N;
    auto md = [N](int v) { int r = v % N; return r < 0 ? r + N : r; };
    for (int64_t i = 0; i < s.n_g; ++i) {
        const int a = s.miller[3 * i], b = s.miller[3 * i + 1], d = s.miller[3 * i + 2];
        if (fft_index) fft_index[i] = (md(a) * N + md(b)) * N + md(d);
        if (fft_index_minus) fft_index_minus[i] = (md(-a) * N + md(-b)) * N + md(-d);
    }
    return WEST_OK;
}

int west_set_vloc(west_ctx* c, const double* vloc) {
    if (!c || !vloc) return fail(c, WEST_EINVAL, "west_set_vloc: NULL argument");
    const long long n3 = n3_of(c);
    int rc;
    const int lch = c->ops->LC_H, N_ = c->cell.N;
    const size_t nv = (size_t)N_ * ((N_ + lch - 1) / lch) * c->ops->N2 * lch * c->ops->N1;      // K2::vloc_elems(): chunks padded to LC lines
    if (!c->d_vpos) {
        if ((rc = dev_alloc(c, (void**)&c->d_vpos, sizeof(double) * nv))) return rc;
        if ((rc = dev_alloc(c, (void**)&c->d_vpos_f, sizeof(float) * nv))) return rc;
        CK(cudaMemsetAsync(c->d_vpos, 0, sizeof(double) * nv, c->st));
        CK(cudaMemsetAsync(c->d_vpos_f, 0, sizeof(float) * nv, c->st));
    }
    vloc_layout<double><<<blocks_for(n3, 256), 256, 0, c->st>>>(N_, c->ops->N1, c->ops->N2, lch, vloc, c->d_vpos);
    vloc_layout<float><<<blocks_for(n3, 256), 256, 0, c->st>>>(N_, c->ops->N1, c->ops->N2, lch, vloc, c->d_vpos_f);
    CK(cudaGetLastError());
    c->launches += 2;
    c->have_vloc = true;
    return WEST_OK;
}

int west_set_kb(west_ctx* c, int32_t n_proj, const void* beta, const double* dcoef_host) {
    if (!c || n_proj < 0 || (n_proj > 0 && (!beta || !dcoef_host))) return fail(c, WEST_EINVAL, "west_set_kb: bad argument");
    const int full = !is_gamma(c);
    const long long n_g = c->hs.n_g;
    c->n_proj = n_proj;
    c->rows_kb = n_proj * (full ? 2 : 1);
    c->A_dirty = true; c->tc_dirty = true; c->i8_dirty = true;
    c->h_dcoef.resize(c->rows_kb);
    for (int k = 0; k < n_proj; ++k) {
        if (full) { c->h_dcoef[2 * k] = dcoef_host[k]; c->h_dcoef[2 * k + 1] = dcoef_host[k]; }
        else c->h_dcoef[k] = dcoef_host[k];
    }
    if (n_proj == 0) return WEST_OK;
    int rc = ensure(c, c->A_kb, (size_t)c->rows_kb * 2 * n_g * sizeof(double));
    if (rc) return rc;
    if ((rc = ensure(c, c->dcoef_dev, sizeof(double) * c->rows_kb))) return rc;
    c->d_dcoef = (double*)c->dcoef_dev.p;
    CK(cudaMemcpy(c->d_dcoef, c->h_dcoef.data(), sizeof(double) * c->rows_kb, cudaMemcpyHostToDevice));
    stack_rows<<<blocks_for(n_g * n_proj, 256), 256, 0, c->st>>>(n_g, n_proj, full, (const cx<double>*)beta, (double*)c->A_kb.p);
    CK(cudaGetLastError());
    c->launches += 1;
    return WEST_OK;
}

int west_set_states(west_ctx* c, int32_t n_occ_user, const void* psi, const double* eps_host) {
    if (!c || n_occ_user <= 0 || !psi || !eps_host) return fail(c, WEST_EINVAL, "west_set_states: bad argument");
    const int full = !is_gamma(c);
    const long long n_g = c->hs.n_g, n3 = n3_of(c);
    // WEST_GAMMA transforms two real orbitals per complex FFT: an odd count gets one ZERO orbital appended (R15).  Its right-hand
    // sides, solutions and density contributions are identically zero (the CG marks zero columns inactive at start), its row in
    // the P_v GEMMs is zero, and it never appears in an output.
    const int n_occ = (!full && (n_occ_user & 1)) ? n_occ_user + 1 : n_occ_user;
    c->n_occ = n_occ;
    c->n_occ_user = n_occ_user;
    c->rows_psi = n_occ * (full ? 2 : 1);
    c->A_dirty = true; c->tc_dirty = true; c->i8_dirty = true;
    c->h_eps.assign(eps_host, eps_host + n_occ_user);
    if (n_occ > n_occ_user) c->h_eps.push_back(eps_host[n_occ_user - 1]);
    int rc = ensure(c, c->A_psi, (size_t)c->rows_psi * 2 * n_g * sizeof(double));
    if (rc) return rc;
    if (n_occ > n_occ_user) CK(cudaMemsetAsync(c->A_psi.p, 0, (size_t)c->rows_psi * 2 * n_g * sizeof(double), c->st));
    stack_rows<<<blocks_for(n_g * n_occ_user, 256), 256, 0, c->st>>>(n_g, n_occ_user, full, (const cx<double>*)psi, (double*)c->A_psi.p);
    CK(cudaGetLastError());
    if ((rc = ensure(c, c->tk, sizeof(double) * n_occ))) return rc;
    if ((rc = ensure(c, c->eps_dev, sizeof(double) * n_occ))) return rc;
    c->d_eps = (double*)c->eps_dev.p;
    CK(cudaMemcpy(c->d_eps, c->h_eps.data(), sizeof(double) * n_occ, cudaMemcpyHostToDevice));
    c->eps_min = *std::min_element(eps_host, eps_host + n_occ_user);
    c->eps_max = *std::max_element(eps_host, eps_host + n_occ_user);
    kinetic_expect<<<n_occ_user, 256, 0, c->st>>>(n_g, is_gamma(c), c->d_g2, (const cx<double>*)psi, (double*)c->tk.p);
    CK(cudaGetLastError());
    if (n_occ > n_occ_user) {
        const double one = 1.0;        // finite preconditioner for the zero orbital's (never active) columns
        CK(cudaMemcpyAsync((double*)c->tk.p + n_occ_user, &one, sizeof(double), cudaMemcpyHostToDevice, c->st));
        CK(cudaStreamSynchronize(c->st));
    }
    c->launches += 2;
    // u_v(r) cache in position order: GAMMA packs (v, v+1) as u_v + i u_{v+1}
    c->n_uslots = full ? n_occ : (n_occ + 1) / 2;
    if ((rc = ensure(c, c->ucache, sizeof(cx<double>) * n3 * c->n_uslots))) return rc;
    // a set-up call may allocate: the stick intermediate of this one transform is a temporary of its own (not the hot arena)
    const int chunk = std::max(1, std::min(c->n_uslots, std::min(chunk_slots(c, 0), 256)));
    void* Wtmp = nullptr;
    cudaError_t e = cudaMalloc(&Wtmp, bytes_W(c, chunk, 0));
    if (e != cudaSuccess) { cudaGetLastError(); return fail(c, WEST_ENOMEM, "west_set_states: cudaMalloc of the transform buffer failed: %s", cudaGetErrorString(e)); }
    VecMap vm{full ? 1 : 2, full ? 0 : 1, n_occ_user, 0};       // vectors >= n_vec read as zero: the padding orbital
    cudaError_t ke = cudaSuccess;
    for (int s0 = 0; s0 < c->n_uslots && ke == cudaSuccess; s0 += chunk) {
        const int ns = std::min(chunk, c->n_uslots - s0);
        vm.slot0 = s0;
        K2Any a{};
        a.W = Wtmp; a.R = (cx<double>*)c->ucache.p + (long long)s0 * n3;
        ke = c->ops->k1(0, is_gamma(c), ns, c->st, c->geom, vm, (const cx<double>*)psi, Wtmp);
        if (ke == cudaSuccess) ke = c->ops->k2(0, K2_TOR, ns, c->st, c->geom, a);
        c->launches += 2;
    }
    cudaStreamSynchronize(c->st);
    cudaFree(Wtmp);
    if (ke != cudaSuccess) return fail(c, WEST_ECUDA, "west_set_states: %s", cudaGetErrorString(ke));
    return WEST_OK;
}

int west_set_deflation(west_ctx* c, int32_t n_defl, const void* psi_c, const double* eps_host) {
    if (!c || n_defl < 0 || (n_defl > 0 && (!psi_c || !eps_host))) return fail(c, WEST_EINVAL, "west_set_deflation: bad argument");
    const int full = !is_gamma(c);
    const long long n_g = c->hs.n_g;
    c->n_defl = n_defl;
    c->rows_defl = n_defl * (full ? 2 : 1);
    c->A_dirty = true; c->tc_dirty = true; c->i8_dirty = true;
    if (n_defl == 0) return WEST_OK;
    c->h_eps_defl.assign(eps_host, eps_host + n_defl);
    int rc = ensure(c, c->A_defl, (size_t)c->rows_defl * 2 * n_g * sizeof(double));
    if (rc) return rc;
    if ((rc = ensure(c, c->eps_defl, sizeof(double) * n_defl))) return rc;
    CK(cudaMemcpyAsync(c->eps_defl.p, c->h_eps_defl.data(), sizeof(double) * n_defl, cudaMemcpyHostToDevice, c->st));
    stack_rows<<<blocks_for(n_g * n_defl, 256), 256, 0, c->st>>>(n_g, n_defl, full, (const cx<double>*)psi_c, (double*)c->A_defl.p);
    CK(cudaGetLastError());
    c->launches += 1;
    return WEST_OK;
}

int west_fft3d(west_ctx* c, int32_t dir, int32_t precision, int32_t n_batch, const void* in, void* out) {
    if (!c || (dir != 1 && dir != -1) || n_batch < 0 || (n_batch > 0 && (!in || !out))) return fail(c, WEST_EINVAL, "west_fft3d: bad argument");
    if (precision != WEST_FP64) return fail(c, WEST_EINVAL, "west_fft3d: only WEST_FP64 (the FP32 variant exists inside west_h_apply only)");
    if (n_batch == 0) return WEST_OK;
    const int gamma = is_gamma(c), N = c->cell.N;
    const long long n3 = n3_of(c);
    const int n_slots = gamma ? (n_batch + 1) / 2 : n_batch;
    const int chunk = fft3d_chunk(c, n_slots);
    int rc;
    if ((rc = hot_begin(c, plan_fft3d(c, n_batch)))) return rc;
    if ((rc = ensure_W(c, chunk, 0))) return rc;
    if ((rc = hot(c, c->Rbuf, sizeof(cx<double>) * n3 * chunk))) return rc;
    VecMap vm{gamma ? 2 : 1, gamma ? 1 : 0, n_batch, 0};
    K2Any a{};
    a.W = c->W.p; a.R = (cx<double>*)c->Rbuf.p;
    for (int s0 = 0; s0 < n_slots; s0 += chunk) {
        const int ns = std::min(chunk, n_slots - s0);
        vm.slot0 = s0;
        if (dir == 1) {
            CK(c->ops->k1(0, gamma, ns, c->st, c->geom, vm, (const cx<double>*)in, c->W.p));
            CK(c->ops->k2(0, K2_TOR, ns, c->st, c->geom, a));
            pos_to_user<<<blocks_for(n3 * ns, 256), 256, 0, c->st>>>(N, c->ops->N1, c->ops->N2, gamma, s0, ns, n_batch, (const cx<double>*)c->Rbuf.p, (double*)out);
        } else {
            user_to_pos<<<blocks_for(n3 * ns, 256), 256, 0, c->st>>>(N, c->ops->N1, c->ops->N2, gamma, s0, ns, n_batch, (const double*)in, (cx<double>*)c->Rbuf.p);
            CK(c->ops->k2(0, K2_FROMR, ns, c->st, c->geom, a));
            K3Epi e{1.0 / ((double)N * N * N), 0, nullptr, 0.0, nullptr};
            CK(c->ops->k3(0, gamma, ns, c->st, c->geom, vm, c->W.p, e, (cx<double>*)out));
        }
        CK(cudaGetLastError());
        c->launches += 3;
    }
    return WEST_OK;
}

int west_fft3d_dense(west_ctx* c, int32_t n, int32_t sign, int32_t precision, int32_t n_batch, const void* in, void* out) {
    if (!c || (sign != 1 && sign != -1) || n_batch < 0 || n_batch > 65535 || (n_batch > 0 && (!in || !out)))
        return fail(c, WEST_EINVAL, "west_fft3d_dense: bad argument");
    if (precision != WEST_FP64 && precision != WEST_FP32) return fail(c, WEST_EINVAL, "west_fft3d_dense: precision must be WEST_FP64 or WEST_FP32");
    if (!west_dense_fft_supported(n)) return fail(c, WEST_EINVAL, "west_fft3d_dense: n = %d is not built (64, 128, 256)", n);
    if (n_batch == 0) return WEST_OK;
    auto it = c->dense_tw.find(n);
    if (it == c->dense_tw.end()) return fail(c, WEST_EINVAL, "west_fft3d_dense: no twiddle table for n = %d", n);
    Prof pf(c, PC_FFT_OTHER);
    CK(west_dense_fft3d(n, precision == WEST_FP32, sign, n_batch, c->st, in, out, it->second));
    c->launches += 3;
    return WEST_OK;
}

int west_h_apply(west_ctx* c, int32_t precision, int32_t n_vec, const void* x, void* y) {
    if (!c || n_vec < 0 || (n_vec > 0 && (!x || !y))) return fail(c, WEST_EINVAL, "west_h_apply: bad argument");
    if (precision != WEST_FP64 && precision != WEST_MIXED && precision != WEST_FP64_I8) return fail(c, WEST_EINVAL, "west_h_apply: bad precision %d", precision);
    if (!c->have_vloc) return fail(c, WEST_ESTATE, "west_h_apply: west_set_vloc has not been called");
    c->gemm_i8 = precision == WEST_FP64_I8 && tc_available(c);
    c->i8_slices = 8;
    if (n_vec == 0) return WEST_OK;
    const int gamma = is_gamma(c);
    const int n_slots = gamma ? (n_vec + 1) / 2 : n_vec;
    VecMap vm{gamma ? 2 : 1, gamma ? 1 : 0, n_vec, 0};
    int rc;
    if ((rc = ensure_opmatrix(c))) return rc;
    // operator data of the tensor paths is (re)built BEFORE the workspace is carved: ensure() may give the lazy workspace back to make room
    c->arena_release_ok = true;
    if (c->gemm_i8 && c->rows_kb > 0) rc = ensure_i8_operator(c);
    if (!rc && precision == WEST_MIXED && tc_available(c) && c->rows_kb > 0) rc = ensure_tc_operator(c);
    c->arena_release_ok = false;
    if (rc) return rc;
    if ((rc = hot_begin(c, plan_happly(c, n_vec, precision == WEST_MIXED, c->gemm_i8)))) return rc;
    if ((rc = hloc_apply(c, precision == WEST_MIXED, vm, n_slots, (const cx<double>*)x, (cx<double>*)y, nullptr, 0.0))) return rc;
    if (c->rows_kb > 0) {
        LowrankCoef lc; lc.dcoef = c->d_dcoef; lc.n_rows_d = c->rows_kb;
        rc = lowrank_apply(c, 0, c->rows_kb, n_vec, (const double*)x, (double*)y, lc, precision == WEST_MIXED);
    }
    return rc;
}

int west_gemm_tn(west_ctx* c, int32_t m, int32_t n, int64_t k, const double* A, int64_t lda, const double* B, int64_t ldb, double* C, int64_t ldc) {
    if (!c || !A || !B || !C || (k & 1) || (lda & 1) || (ldb & 1)) return fail(c, WEST_EINVAL, "west_gemm_tn: k, lda, ldb must be even");
    return launch_gemm_tn(c, m, n, k, A, lda, B, ldb, C, ldc);
}
int west_gemm_update(west_ctx* c, int32_t m, int32_t n, int64_t k, const double* C, int64_t ldc, const double* A, int64_t lda, double* Y, int64_t ldy) {
    if (!c || !A || !Y || !C || (k & 1) || (lda & 1) || (ldc & 1) || (ldy & 1)) return fail(c, WEST_EINVAL, "west_gemm_update: k, lda, ldc, ldy must be even");
    return launch_gemm_update(c, m, n, k, C, ldc, A, lda, Y, ldy);
}

}  // extern "C"

// ============================================================================================================ chi0 * dV
namespace {

#ifndef WEST_RES_NT
#define WEST_RES_NT 1024
#define WEST_RES_EPT 9
#endif
constexpr int RES_NT = WEST_RES_NT, RES_EPT = WEST_RES_EPT;
template <int MODE>
cudaError_t cg_resident_attr() {
    if (MODE == 1) return cudaSuccess;
    constexpr int M = MODE == 1 ? 0 : MODE;
    return cudaFuncSetAttribute(wcg::cg_step_resident<M, RES_NT, RES_EPT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)(sizeof(double2) * RES_NT * RES_EPT));
}
constexpr int CLU_NT = 512, CLU_EPT = 9, CLU_CL = 2;
template <int MODE>
cudaError_t cg_cluster_attr() {
    constexpr int M = MODE == 1 ? 0 : MODE;
    return cudaFuncSetAttribute(wcg::cg_step_cluster<M, CLU_NT, CLU_EPT, CLU_CL>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)(sizeof(double2) * CLU_NT * CLU_EPT));
}
template <int MODE>
void cg_cluster_launch(int n_act, cudaStream_t st, long long n_g, int n_occ, const double* g2, const double* tk, int precond_on, double tol2,
                       double2* P, const double2* AP, double2* X, double2* R, wcg::Scalars s, const int* colmap) {
    constexpr int M = MODE == 1 ? 0 : MODE;
    const int ept = (int)((n_g + (long long)CLU_NT * CLU_CL - 1) / ((long long)CLU_NT * CLU_CL));
    wcg::cg_step_cluster<M, CLU_NT, CLU_EPT, CLU_CL><<<n_act * CLU_CL, CLU_NT, sizeof(double2) * CLU_NT * ept, st>>>(
        n_g, n_occ, g2, tk, precond_on, tol2, P, AP, X, R, s, colmap);
}
template <int MODE>
void cg_resident_launch(int n_act, cudaStream_t st, long long n_g, int n_occ, const double* g2, const double* tk, int precond_on, double tol2,
                        double2* P, const double2* AP, double2* X, double2* R, wcg::Scalars s, const int* colmap) {
    constexpr int M = MODE == 1 ? 0 : MODE;          // MODE 1 never takes this path
    const int ept = (int)((n_g + RES_NT - 1) / RES_NT);
    wcg::cg_step_resident<M, RES_NT, RES_EPT><<<n_act, RES_NT, sizeof(double2) * RES_NT * ept, st>>>(n_g, n_occ, g2, tk, precond_on, tol2, P, AP,
                                                                                                      X, R, s, colmap);
}

// Lagged convergence poll (reading R5 allows late masking): the live-column count written by iteration k is copied to pinned host memory
// behind iteration k's kernels and READ by the host only after iteration k+1 has been queued, so the stream never drains inside the
// solve.  The host's column count n_act is therefore an upper bound of the device's (cg_compact_map pads the difference with inert
// columns), and the iteration after the last live column converged is launched on inactive columns (its kernels change nothing).
struct Poller {
    int slot = 0, pending = -1;
    cudaError_t post(west_ctx* c, const int* dev_counter) {
        cudaError_t e = cudaMemcpyAsync(c->h_pinned + slot, dev_counter, sizeof(int), cudaMemcpyDeviceToHost, c->st);
        if (e == cudaSuccess) e = cudaEventRecord(c->ev_poll[slot], c->st);
        pending = slot; slot ^= 1;
        return e;
    }
    bool ready() const { return pending >= 0; }
    int collect(west_ctx* c) {
        cudaEventSynchronize(c->ev_poll[pending]);
        const int v = c->h_pinned[pending];
        pending = -1;
        return v;
    }
};

// drop converged columns from the working set (r -> AP buffer, p -> old r buffer; rotation by the caller)
int compact_columns(west_ctx* c, int n_act, int n_new, long long len, int*& colmap, int*& newmap, int* src, const int* active, cx<double>*& R,
                    cx<double>*& P, cx<double>*& AP) {
    Prof p_(c, PC_CGVEC);
    wcg::cg_compact_map<<<1, 1024, 0, c->st>>>(n_act, colmap, active, newmap, src, n_new);
    wcg::cg_gather_cols<<<n_new, wcg::NT, 0, c->st>>>(len, src, (const double2*)R, (double2*)AP);
    wcg::cg_gather_cols<<<n_new, wcg::NT, 0, c->st>>>(len, src, (const double2*)P, (double2*)R);
    CK(cudaGetLastError());
    c->launches += 3;
    cx<double>* oldR = R; cx<double>* oldP = P;
    R = AP; P = oldR; AP = oldP;           // AP (scratch) now holds r, the old r buffer holds p
    std::swap(colmap, newmap);
    return WEST_OK;
}

template <int MODE>
int cg_solve(west_ctx* c, int f32, int n_col, const west_cg_opts& o, double omega, cx<double>* X, cx<double>*& R, cx<double>*& P,
             cx<double>*& AP, double* shift, wcg::Scalars s, int* maps /* [3][n_col] */, int* iters_out, int64_t* n_h_out, int* live_out) {
    const long long n_g = c->hs.n_g;
    const int nvpc = MODE == 1 ? 2 : 1, n_occ = c->n_occ;
    const long long len = (long long)nvpc * n_g;
    const int gamma = is_gamma(c);
    const double* g2 = c->d_g2;
    const double* tk = (const double*)c->tk.p;
    const double tol2 = o.tol * o.tol;
    const int every = std::max(1, o.check_every);
    int* colmap = maps; int* newmap = maps + n_col; int* src = maps + 2 * (size_t)n_col;
    CK(cudaMemsetAsync(s.counters, 0, 2 * sizeof(int), c->st));
    CK(cudaMemsetAsync(X, 0, sizeof(cx<double>) * len * n_col, c->st));
    wcg::cg_init<MODE><<<n_col, wcg::NT, 0, c->st>>>(n_g, n_occ, g2, tk, o.precond, (const double2*)R, (double2*)P, s, colmap);
    CK(cudaGetLastError());
    c->launches += 1;
    const int rows = c->rows_kb + c->rows_psi + c->rows_defl;
    // column-resident vector kernel when a column fits one CTA's registers + shared memory (cfgs 1-4); else the streaming one
    const bool resident = MODE != 1 && n_g <= (long long)RES_EPT * RES_NT && c->cg_kernel == 0;
    const bool clustered = MODE != 1 && n_g <= (long long)CLU_EPT * CLU_NT * CLU_CL && c->cg_kernel == 2;
    if (resident) CK(cg_resident_attr<MODE>());
    if (clustered) CK(cg_cluster_attr<MODE>());
    int n_act = n_col;          // columns currently held (compacted) in R, P, AP: an upper bound of the device's live count
    int it = 0, live = n_col;
    int64_t n_h = 0;
    Poller poll;
    bool done = false;
    for (; it < o.max_iter && !done; ++it) {
        // slots of the H application: GAMMA pairs vectors (2s, 2s+1) - in MODE 1 these are (Re, Im) of one column
        const int n_vec = n_act * nvpc;
        VecMap vm{gamma ? 2 : 1, gamma ? 1 : 0, n_vec, 0};
        const int n_slots = gamma ? (n_vec + 1) / 2 : n_vec;
        int rc = hloc_apply(c, f32, vm, n_slots, P, AP, shift, omega);
        if (rc) return rc;
        LowrankCoef lc;
        lc.dcoef = c->d_dcoef; lc.n_rows_d = c->rows_kb; lc.alpha_vec = (const double*)c->alpha_v.p; lc.colmap = colmap; lc.nvpc = nvpc; lc.n_occ = n_occ;
        rc = lowrank_apply(c, 0, rows, n_vec, (const double*)P, (double*)AP, lc, f32 != 0);
        if (rc) return rc;
        n_h += n_vec;
        {
            Prof p_(c, PC_CGVEC);
            if (clustered)
                cg_cluster_launch<MODE>(n_act, c->st, n_g, n_occ, g2, tk, o.precond, tol2, (double2*)P, (const double2*)AP, (double2*)X, (double2*)R,
                                        s, colmap);
            else if (resident)
                cg_resident_launch<MODE>(n_act, c->st, n_g, n_occ, g2, tk, o.precond, tol2, (double2*)P, (const double2*)AP, (double2*)X, (double2*)R,
                                         s, colmap);
            else
                wcg::cg_step<MODE><<<n_act, wcg::NT, 0, c->st>>>(n_g, n_occ, g2, tk, o.precond, tol2, (double2*)P, (const double2*)AP,
                                                                 (double2*)X, (double2*)R, s, colmap);
            CK(cudaGetLastError());
            c->launches += 1;
        }
        if (poll.ready()) {                       // the count as of the previous polled iteration; this iteration is already queued
            live = poll.collect(c);
            if (live <= 0) done = true;
            // drop converged columns from the working set when that removes at least ~6 % of it (a1-a9 then run on fewer vectors)
            else if (it + 1 < o.max_iter && live <= n_act - std::max(2, n_act / 16)) {
                if ((rc = compact_columns(c, n_act, live, len, colmap, newmap, src, s.active, R, P, AP))) return rc;
                n_act = live;
                fill_shift<<<blocks_for(n_act * nvpc, 256), 256, 0, c->st>>>(n_act * nvpc, nvpc, n_occ, c->d_eps, shift, colmap);
                CK(cudaGetLastError());
                c->launches += 1;
            }
        }
        if (!done && ((it + 1) % every == 0 || it + 1 == o.max_iter)) CK(poll.post(c, s.counters));
    }
    if (poll.ready()) live = poll.collect(c);     // cap reached: the exact final count
    *iters_out = it;
    *n_h_out = n_h;
    *live_out = live;
    return WEST_OK;
}

__global__ void fill_const(int n, double v, double* out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = v;
}
// alpha_v of the alpha P_v term (reading R3): the caller's constant, or (alpha_user <= 0) the per-orbital default
// alpha_v = (eps_v - eps_min) + W/2, W the occupied band width: H - eps_v + alpha_v P_v is then >= W/2 on the occupied space for every v
__global__ void fill_alpha(int n_occ, const double* eps, double eps_min, double width, double alpha_user, double* out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n_occ) out[i] = alpha_user > 0 ? alpha_user : fmax(eps[i] - eps_min + 0.5 * width, 0.01);
}

// a1: b = -P_c (dV_i psi_v) written into R ([n_col][nvpc][n_g]; the imaginary-part vectors of nvpc = 2 stay zero)
int chi0_rhs(west_ctx* c, int n_pert, int nvpc, cx<double>* R, double sign = -1.0, bool project = true) {
    const int gamma = is_gamma(c), N = c->cell.N, n_col = n_pert * c->n_occ, n_vec = n_col * nvpc;
    const long long n_g = c->hs.n_g;
    const int n_uslots = c->n_uslots, n_rslots = n_pert * n_uslots;
    const int chunk = std::max(1, chunk_slots(c, 0));
    int rc = ensure_W(c, std::max(n_rslots, 1), 0);
    if (rc) return rc;
    if (nvpc == 2) CK(cudaMemsetAsync(R, 0, sizeof(cx<double>) * n_g * n_vec, c->st));
    // slot (i, us) -> columns i*n_occ + 2us (+1)  [GAMMA] or i*n_occ + us
    VecMap vm{gamma ? 2 * nvpc : 1, gamma ? nvpc : 0, n_vec, 0};
    K2Any a{};
    a.W = c->W.p; a.ucache = (const cx<double>*)c->ucache.p; a.dV = (const double*)c->dVpos.p; a.n_uslots = n_uslots;
    K3Epi e{sign / ((double)N * N * N), 0, nullptr, 0.0, nullptr};
    for (int s0 = 0; s0 < n_rslots; s0 += chunk) {
        const int ns = std::min(chunk, n_rslots - s0);
        vm.slot0 = s0; a.slot0 = s0;
        Prof p_(c, PC_FFT_OTHER);
        CK(c->ops->k2(0, K2_FROMR, ns, c->st, c->geom, a));
        CK(c->ops->k3(0, gamma, ns, c->st, c->geom, vm, c->W.p, e, R));
        c->launches += 2;
    }
    if (!project) return WEST_OK;
    // R <- R - Psi (Psi^T R): coefficient -1 on the psi rows (and, if set, the deflated conduction states)
    const int rows_p = c->rows_psi + c->rows_defl;
    LowrankCoef lc; lc.alpha_const = -1.0;
    if ((rc = lowrank_apply(c, c->rows_kb, rows_p, n_vec, (const double*)R, (double*)R, lc))) return rc;
    if (c->rows_defl > 0) {
        // Cbuf now holds <psi_m | dV psi_v> for every projector row: keep the deflation rows for the closed-form part of the solution
        const long long ldc = (n_vec + 1) / 2 * 2;
        if ((rc = hot(c, c->craw, sizeof(double) * (size_t)c->rows_defl * ldc))) return rc;
        c->craw_ld = ldc;
        CK(cudaMemcpyAsync(c->craw.p, (const double*)c->Cbuf.p + (size_t)c->rows_psi * ldc, sizeof(double) * (size_t)c->rows_defl * ldc,
                           cudaMemcpyDeviceToDevice, c->st));
    }
    return WEST_OK;
}

// Deflation (optional, west_set_deflation): the components of the solution along the given conduction eigenstates are known in
// closed form, dpsi_low = - sum_c psi_c <psi_c|dV psi_v> / (eps_c - eps_v - i omega); the CG runs on the complement (those states sit
// in the alpha-projector next to P_v, the right-hand side is projected off them), which raises the smallest eigenvalue of the
// operator from the gap to eps_(first state not deflated) - eps_v and cuts the iteration count.  Exact, not a truncation.
__global__ void defl_coef(int rows, int mult, int n_col, int in_nvpc, int out_nvpc, int n_occ, long long ld_in, const double* Craw,
                          long long ld_out, double* D, const double* eps_c, const double* eps_v, double omega) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int n_out = n_col * out_nvpc;
    if (i >= (long long)rows * n_out) return;
    const int m = (int)(i / n_out), n = (int)(i - (long long)m * n_out);
    const int col = n / out_nvpc, part = n - col * out_nvpc;
    const double delta = eps_c[m / mult] - eps_v[col % n_occ];
    const double cr = Craw[(long long)m * ld_in + (long long)col * in_nvpc];
    double d;
    if (out_nvpc == 1) d = -cr / delta;
    else { const double den = delta * delta + omega * omega; d = part == 0 ? -cr * delta / den : -cr * omega / den; }
    D[(long long)m * ld_out + n] = d;
}

int add_deflated(west_ctx* c, int n_col, int in_nvpc, int out_nvpc, double omega, cx<double>* X) {
    if (c->rows_defl == 0) return WEST_OK;
    const long long K = 2 * c->hs.n_g;
    const int n_out = n_col * out_nvpc;
    const long long ldo = (n_out + 1) / 2 * 2;
    int rc = hot(c, c->dcoef_defl, sizeof(double) * (size_t)c->rows_defl * ldo);
    if (rc) return rc;
    CK(cudaMemsetAsync(c->dcoef_defl.p, 0, sizeof(double) * (size_t)c->rows_defl * ldo, c->st));
    defl_coef<<<blocks_for((long long)c->rows_defl * n_out, 256), 256, 0, c->st>>>(
        c->rows_defl, is_gamma(c) ? 1 : 2, n_col, in_nvpc, out_nvpc, c->n_occ, c->craw_ld, (const double*)c->craw.p, ldo,
        (double*)c->dcoef_defl.p, (const double*)c->eps_defl.p, c->d_eps, omega);
    CK(cudaGetLastError());
    c->launches += 1;
    const double* A = (const double*)c->A_all.p + (size_t)(c->rows_kb + c->rows_psi) * K;
    return launch_gemm_update(c, c->rows_defl, n_out, K, (const double*)c->dcoef_defl.p, ldo, A, K, (double*)X, K);
}

// a10: dn_i(r) = (4/Omega) Re sum_v conj(u_v) du_iv from X ([n_col][nvpc][n_g]) into dn_out ([n_pert][N^3], natural order)
int chi0_dn(west_ctx* c, int n_pert, int nvpc, const cx<double>* X, double* dn_out, double occupation, int accumulate) {
    const int gamma = is_gamma(c), N = c->cell.N, n_col = n_pert * c->n_occ, n_vec = n_col * nvpc;
    const long long n3 = n3_of(c);
    const double vol = c->cell.L * c->cell.L * c->cell.L;
    const int n_uslots = c->n_uslots, n_rslots = n_pert * n_uslots;
    const int chunk = std::max(1, chunk_slots(c, 0));
    int rc = ensure_W(c, std::max(n_rslots, 1), 0);
    if (rc) return rc;
    CK(cudaMemsetAsync(c->dnpos.p, 0, sizeof(double) * n3 * n_pert, c->st));
    VecMap vm{gamma ? 2 * nvpc : 1, gamma ? nvpc : 0, n_vec, 0};
    K2Any a{};
    a.W = c->W.p; a.ucache = (const cx<double>*)c->ucache.p; a.dn = (double*)c->dnpos.p; a.n_uslots = n_uslots; a.fac = 2.0 * occupation / vol;
    for (int s0 = 0; s0 < n_rslots; s0 += chunk) {
        const int ns = std::min(chunk, n_rslots - s0);
        vm.slot0 = s0; a.slot0 = s0;
        Prof p_(c, PC_FFT_OTHER);
        CK(c->ops->k1(0, gamma, ns, c->st, c->geom, vm, X, c->W.p));
        CK(c->ops->k2(0, K2_DN, ns, c->st, c->geom, a));
        c->launches += 2;
    }
    pos_to_nat_real<<<blocks_for(n3 * n_pert, 256), 256, 0, c->st>>>(N, c->ops->N1, c->ops->N2, n3 * n_pert, (const double*)c->dnpos.p, dn_out, accumulate);
    CK(cudaGetLastError());
    c->launches += 1;
    return WEST_OK;
}

// converged solutions -> the caller's dpsi block of this (frequency, perturbation sub-block): out column (i, v < n_user), parts_out
// vectors per column; the solver's column (i, v) holds parts_in vectors (parts beyond it are written as zero)
__global__ void __launch_bounds__(wcg::NT) dpsi_gather(long long n_g, int n_occ, int n_user, int parts_in, int parts_out, const double2* X, double2* out) {
    const int b = blockIdx.x;                      // (i * n_user + v) * parts_out + q
    const int q = b % parts_out, cv = b / parts_out, v = cv % n_user, i = cv / n_user;
    double2* dst = out + (long long)b * n_g;
    if (q < parts_in) {
        const double2* src = X + (((long long)i * n_occ + v) * parts_in + q) * n_g;
        for (long long g = threadIdx.x; g < n_g; g += wcg::NT) dst[g] = src[g];
    } else {
        for (long long g = threadIdx.x; g < n_g; g += wcg::NT) dst[g] = make_double2(0.0, 0.0);
    }
}

// multi-shift CG (WEST_GAMMA): all frequencies from one unpreconditioned Krylov sequence of the real seed operator
int ms_solve(west_ctx* c, int f32, int n_col, const west_cg_opts& o, const wcg::MsShifts& sh, cx<double>*& R, cx<double>*& P, cx<double>*& AP,
             cx<double>* XS, cx<double>* PS, int want_imag, double* shift, wcg::MsState st, int* maps, int* iters_out, int64_t* n_h_out) {
    const long long n_g = c->hs.n_g;
    const int n_occ = c->n_occ;
    const double tol2 = o.tol * o.tol;
    const int every = std::max(1, o.check_every);
    int* colmap = maps; int* newmap = maps + n_col; int* src = maps + 2 * (size_t)n_col;
    CK(cudaMemsetAsync(st.counters, 0, 4 * sizeof(int), c->st));
    CK(cudaMemsetAsync(XS, 0, sizeof(cx<double>) * 2 * n_g * n_col * sh.n, c->st));
    wcg::ms_init<<<n_col, wcg::NT, 0, c->st>>>(n_g, n_col, sh, (const double2*)R, (double2*)P, (double2*)PS, st, colmap);
    CK(cudaGetLastError());
    c->launches += 1;
    const int rows = c->rows_kb + c->rows_psi + c->rows_defl;
    int n_act = n_col, it = 0;
    int64_t n_h = 0;
    Poller poll;
    bool done = false;
    for (; it < o.max_iter && !done; ++it) {
        VecMap vm{2, 1, n_act, 0};
        int rc = hloc_apply(c, f32, vm, (n_act + 1) / 2, P, AP, shift, 0.0);
        if (rc) return rc;
        LowrankCoef lc;
        lc.dcoef = c->d_dcoef; lc.n_rows_d = c->rows_kb; lc.alpha_vec = (const double*)c->alpha_v.p; lc.colmap = colmap; lc.nvpc = 1; lc.n_occ = n_occ;
        rc = lowrank_apply(c, 0, rows, n_act, (const double*)P, (double*)AP, lc, f32 != 0);
        if (rc) return rc;
        n_h += n_act;
        {
            Prof p_(c, PC_CGVEC);
            wcg::ms_step<<<n_act, wcg::NT, 0, c->st>>>(n_g, n_col, sh, tol2, want_imag, (double2*)P, (const double2*)AP, (double2*)R, (double2*)XS,
                                                       (double2*)PS, st, colmap);
            CK(cudaGetLastError());
            c->launches += 1;
        }
        if (poll.ready()) {
            const int live = poll.collect(c);
            if (live <= 0) done = true;
            else if (it + 1 < o.max_iter && live <= n_act - std::max(2, n_act / 16)) {
                if ((rc = compact_columns(c, n_act, live, n_g, colmap, newmap, src, st.active, R, P, AP))) return rc;
                n_act = live;
                fill_shift<<<blocks_for(n_act, 256), 256, 0, c->st>>>(n_act, 1, n_occ, c->d_eps, shift, colmap);
                CK(cudaGetLastError());
                c->launches += 1;
            }
        }
        if (!done && ((it + 1) % every == 0 || it + 1 == o.max_iter)) CK(poll.post(c, st.counters));
    }
    if (poll.ready()) poll.collect(c);
    *iters_out = it;
    *n_h_out = n_h;
    return WEST_OK;
}

// multi-shift CG with a Krylov history (cg_kernels.cuh, ms_hist_*): the seed recurrence keeps its residuals r_j in a ring of hs.H slots
// (slot 0 holds b on entry) and the shifted solutions are contracted from them once per segment, instead of 6 vector passes per live
// shift and iteration.  QS (carry vectors, [shift][col][2][n_g]) is only touched when the ring wraps (more than H - 1 iterations).
cudaError_t ms_hist_attrs() {
    static bool done = false;
    if (done) return cudaSuccess;
    const int bytes = (int)(2 * wcg::MS_MAX_SHIFTS * (wcg::MSH_HMAX + 1) * sizeof(double2));
    cudaError_t e = cudaFuncSetAttribute(wcg::ms_hist_combine<false, false, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(wcg::ms_hist_combine<true, false, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(wcg::ms_hist_combine<false, true, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(wcg::ms_hist_combine<true, true, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    done = e == cudaSuccess;
    return e;
}
int ms_hist_combine_launch(west_ctx* c, int n_col, int n_shift, int j0, int n_end, bool carry_in, bool carry_out, bool imag, const wcg::MsHist& hs,
                           const wcg::MsState& st, cx<double>* XS, cx<double>* QS) {
    if (n_end <= j0) return WEST_OK;
    const long long n_g = c->hs.n_g;
    const size_t sm = 2 * (size_t)n_shift * (size_t)(n_end - j0 + 1) * sizeof(double2);
    dim3 grid((unsigned)n_col, (unsigned)((n_g + wcg::MSH_CHUNK - 1) / wcg::MSH_CHUNK));
    unsigned long long* ctr = reinterpret_cast<unsigned long long*>(st.counters + 2);
    Prof p_(c, PC_CGVEC);
    if (imag && carry_out) wcg::ms_hist_combine<true, true, 4><<<grid, wcg::NT, sm, c->st>>>(n_g, n_col, n_shift, j0, n_end, carry_in, hs, st.iters, (double2*)XS, (double2*)QS, ctr);
    else if (imag) wcg::ms_hist_combine<true, false, 4><<<grid, wcg::NT, sm, c->st>>>(n_g, n_col, n_shift, j0, n_end, carry_in, hs, st.iters, (double2*)XS, (double2*)QS, ctr);
    else if (carry_out) wcg::ms_hist_combine<false, true, 8><<<grid, wcg::NT, sm, c->st>>>(n_g, n_col, n_shift, j0, n_end, carry_in, hs, st.iters, (double2*)XS, (double2*)QS, ctr);
    else wcg::ms_hist_combine<false, false, 8><<<grid, wcg::NT, sm, c->st>>>(n_g, n_col, n_shift, j0, n_end, carry_in, hs, st.iters, (double2*)XS, (double2*)QS, ctr);
    CK(cudaGetLastError());
    c->launches += 1;
    return WEST_OK;
}
int ms_hist_solve(west_ctx* c, int f32, int n_col, const west_cg_opts& o, const wcg::MsShifts& sh, const wcg::MsHist& hs, cx<double>*& P, cx<double>*& AP,
                  cx<double>* XS, cx<double>* QS, int want_imag, double* shift, wcg::MsState st, int* maps, int* iters_out, int64_t* n_h_out) {
    const long long n_g = c->hs.n_g;
    const int n_occ = c->n_occ;
    const double tol2 = o.tol * o.tol;
    const int every = std::max(1, o.check_every);
    int* colmap = maps; int* newmap = maps + n_col; int* src = maps + 2 * (size_t)n_col;
    CK(ms_hist_attrs());
    CK(cudaMemsetAsync(st.counters, 0, 4 * sizeof(int), c->st));
    CK(cudaMemsetAsync(XS, 0, sizeof(cx<double>) * 2 * n_g * n_col * sh.n, c->st));
    wcg::ms_init<<<n_col, wcg::NT, 0, c->st>>>(n_g, n_col, sh, (const double2*)hs.vec, (double2*)P, (double2*)nullptr, st, colmap);
    CK(cudaGetLastError());
    c->launches += 1;
    const int rows = c->rows_kb + c->rows_psi + c->rows_defl;
    // column-resident vector kernel where a column fits one SM (cfgs 1-4), as in cg_solve
    const bool resident = n_g <= (long long)RES_EPT * RES_NT && c->cg_kernel == 0;
    if (resident)
        CK(cudaFuncSetAttribute(wcg::ms_hist_step_resident<RES_NT, RES_EPT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sizeof(double2) * RES_NT * RES_EPT)));
    int n_act = n_col, it = 0, j0 = 0;
    bool carry = false;
    int64_t n_h = 0;
    Poller poll;
    bool done = false;
    int rc;
    for (; it < o.max_iter && !done; ++it) {
        if (it - j0 + 1 == hs.H) {            // iteration `it` would overwrite r_j0: contract the segment [j0, it) first, keep the carry vectors
            if ((rc = ms_hist_combine_launch(c, n_col, sh.n, j0, it, carry, true, want_imag != 0, hs, st, XS, QS))) return rc;
            j0 = it; carry = true;
        }
        VecMap vm{2, 1, n_act, 0};
        rc = hloc_apply(c, f32, vm, (n_act + 1) / 2, P, AP, shift, 0.0);
        if (rc) return rc;
        LowrankCoef lc;
        lc.dcoef = c->d_dcoef; lc.n_rows_d = c->rows_kb; lc.alpha_vec = (const double*)c->alpha_v.p; lc.colmap = colmap; lc.nvpc = 1; lc.n_occ = n_occ;
        rc = lowrank_apply(c, 0, rows, n_act, (const double*)P, (double*)AP, lc, f32 != 0);
        if (rc) return rc;
        n_h += n_act;
        {
            Prof p_(c, PC_CGVEC);
            if (resident) {
                const int ept = (int)((n_g + RES_NT - 1) / RES_NT);
                wcg::ms_hist_step_resident<RES_NT, RES_EPT><<<n_act, RES_NT, sizeof(double2) * RES_NT * ept, c->st>>>(n_g, n_col, sh, tol2, it, hs, (double2*)P,
                                                                                                                  (const double2*)AP, st, colmap);
            } else
                wcg::ms_hist_step<<<n_act, wcg::NT, 0, c->st>>>(n_g, n_col, sh, tol2, it, hs, (double2*)P, (const double2*)AP, st, colmap);
            CK(cudaGetLastError());
            c->launches += 1;
        }
        if (poll.ready()) {
            const int live = poll.collect(c);
            if (live <= 0) done = true;
            else if (it + 1 < o.max_iter && live <= n_act - std::max(2, n_act / 16)) {
                // only p is a compacted working vector here (the residuals stay in the ring in original column order)
                Prof p_(c, PC_CGVEC);
                wcg::cg_compact_map<<<1, 1024, 0, c->st>>>(n_act, colmap, st.active, newmap, src, live);
                wcg::cg_gather_cols<<<live, wcg::NT, 0, c->st>>>(n_g, src, (const double2*)P, (double2*)AP);
                CK(cudaGetLastError());
                c->launches += 2;
                std::swap(P, AP);
                std::swap(colmap, newmap);
                n_act = live;
                fill_shift<<<blocks_for(n_act, 256), 256, 0, c->st>>>(n_act, 1, n_occ, c->d_eps, shift, colmap);
                CK(cudaGetLastError());
                c->launches += 1;
            }
        }
        if (!done && ((it + 1) % every == 0 || it + 1 == o.max_iter)) CK(poll.post(c, st.counters));
    }
    if (poll.ready()) poll.collect(c);
    if ((rc = ms_hist_combine_launch(c, n_col, sh.n, j0, it, carry, false, want_imag != 0, hs, st, XS, QS))) return rc;
    *iters_out = it;
    *n_h_out = n_h;
    return WEST_OK;
}

// ---- block CG (solver 2, omega = 0): one Krylov space per orbital shared by its s = np right-hand sides (bcg_kernels.cuh)
size_t bcg_small_bytes(int n_occ, int s) {
    const size_t ss = (size_t)s * s, no = (size_t)n_occ, nc = no * s;
    return al256(sizeof(double) * 4 * no * ss) + al256(sizeof(double) * no * s) + al256(sizeof(int) * (no * s + no)) + al256(sizeof(double) * 2 * nc) +
           al256(sizeof(int) * 3 * no + 64) + al256(sizeof(int) * (3 * no + nc));
}
template <int TS>
void gram_launch(west_ctx* c, int s, long long K, int n_act, const int* orbmap, const double* A, const double* B, double* C, int gamma) {
    const int tiles = (s + TS - 1) / TS, t2 = tiles * tiles;
    long long splits = std::max<long long>(1, std::min<long long>(K / 2048, (592 + (long long)n_act * t2 - 1) / ((long long)n_act * t2)));
    long long kps = ((K + splits - 1) / splits + 31) / 32 * 32;
    splits = (K + kps - 1) / kps;
    if (splits > 1) cudaMemsetAsync(C, 0, sizeof(double) * (size_t)n_act * s * s, c->st);
    wbcg::gram_kernel<TS><<<dim3(n_act, (unsigned)(t2 * splits)), 256, 0, c->st>>>(s, K, n_act, orbmap, A, B, C, gamma, (int)splits, kps);
}
int bcg_gram(west_ctx* c, int s, long long K, int n_act, const int* orbmap, const cx<double>* A, const cx<double>* B, double* C) {
    Prof p_(c, PC_MISC);
    const int gamma = is_gamma(c) ? 1 : 0;
    if (s <= 16) gram_launch<16>(c, s, K, n_act, orbmap, (const double*)A, (const double*)B, C, gamma);
    else if (s <= 32) gram_launch<32>(c, s, K, n_act, orbmap, (const double*)A, (const double*)B, C, gamma);
    else gram_launch<64>(c, s, K, n_act, orbmap, (const double*)A, (const double*)B, C, gamma);
    CK(cudaGetLastError());
    c->launches += 1;
    return WEST_OK;
}
int bcg_update(west_ctx* c, int s, long long K, int n_act, const int* orbmap, const double* C, const cx<double>* P, cx<double>* Y, long long out_stride,
               const int* out_orb, double sign) {
    Prof p_(c, PC_MISC);
    const unsigned gx = (unsigned)((K / 2 + 255) / 256);
    if (s <= 16)
        wbcg::update_kernel<16><<<dim3(gx, n_act, 1), 256, sizeof(double) * s * 16, c->st>>>(s, K, n_act, orbmap, C, (const double*)P, (double*)Y, out_stride, out_orb, sign);
    else
        wbcg::update_kernel<32><<<dim3(gx, n_act, (s + 31) / 32), 256, sizeof(double) * s * 32, c->st>>>(s, K, n_act, orbmap, C, (const double*)P, (double*)Y, out_stride,
                                                                                                      out_orb, sign);
    CK(cudaGetLastError());
    c->launches += 1;
    return WEST_OK;
}

int bcg_solve(west_ctx* c, int f32, int s, const west_cg_opts& o, cx<double>* X, cx<double>* R, cx<double>* P, cx<double>* Q, cx<double>* Z, double* shift,
              double* rep_dev, int* iters_out, int64_t* n_h_out, int* live_out) {
    const long long n_g = c->hs.n_g, K = 2 * n_g;
    const int n_occ = c->n_occ, gamma = is_gamma(c), n_col = s * n_occ;
    const double tol2 = o.tol * o.tol;
    const int every = std::max(1, o.check_every);
    const double* tk = (const double*)c->tk.p;
    // carve the small buffers
    char* p = (char*)c->blk.p;
    auto take = [&](size_t bytes) { char* q = p; p += al256(bytes); return q; };
    const size_t ss = (size_t)s * s;
    double* G = (double*)take(sizeof(double) * 4 * n_occ * ss);
    double* T = G + n_occ * ss; double* C = T + n_occ * ss;
    wbcg::Fac fac;
    fac.L = C + n_occ * ss;
    fac.D = (double*)take(sizeof(double) * n_occ * s);
    fac.order = (int*)take(sizeof(int) * ((size_t)n_occ * s + n_occ));
    fac.rank = fac.order + (size_t)n_occ * s;
    wbcg::State st;
    st.b2 = (double*)take(sizeof(double) * 2 * n_col); st.rr = st.b2 + n_col;
    st.n_open = (int*)take(sizeof(int) * 3 * n_occ + 64); st.active = st.n_open + n_occ; st.iters = st.active + n_occ; st.counters = st.iters + n_occ;
    int* orbmap = (int*)take(sizeof(int) * (3 * (size_t)n_occ + n_col));
    int* newmap = orbmap + n_occ; int* src = newmap + n_occ; int* colmap = src + n_occ;
    const size_t csm = wbcg::coef_smem(s);
    if (csm > 48 * 1024) CK(cudaFuncSetAttribute(wbcg::coef_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)csm));

    CK(cudaMemsetAsync(st.n_open, 0, sizeof(int) * 3 * n_occ + 64, c->st));
    CK(cudaMemsetAsync(X, 0, sizeof(cx<double>) * n_g * n_col, c->st));
    // identity orbital map; Z = M R goes straight into P (the first search block); b2, flags
    wbcg::colmap_kernel<<<blocks_for(n_occ, 256), 256, 0, c->st>>>(n_occ, 1, n_occ, nullptr, orbmap);
    wbcg::zr_kernel<<<n_col, 256, 0, c->st>>>(n_g, n_occ, n_occ, gamma, orbmap, c->d_g2, tk, o.precond, tol2, 1, (const double2*)R, (double2*)P, st);
    wbcg::flags_kernel<<<blocks_for(n_occ, 256), 256, 0, c->st>>>(n_occ, orbmap, 1, st);
    wbcg::colmap_kernel<<<blocks_for(n_col, 256), 256, 0, c->st>>>(n_occ, s, n_occ, orbmap, colmap);
    CK(cudaGetLastError());
    c->launches += 4;
    const int rows = c->rows_kb + c->rows_psi + c->rows_defl;
    int n_act = n_occ, it = 0, live = n_occ;
    int64_t n_h = 0;
    Poller poll;
    bool done = false;
    for (; it < o.max_iter && !done; ++it) {
        const int n_vec = n_act * s;
        VecMap vm{gamma ? 2 : 1, gamma ? 1 : 0, n_vec, 0};
        const int n_slots = gamma ? (n_vec + 1) / 2 : n_vec;
        int rc = hloc_apply(c, f32, vm, n_slots, P, Q, shift, 0.0);
        if (rc) return rc;
        LowrankCoef lc;
        lc.dcoef = c->d_dcoef; lc.n_rows_d = c->rows_kb; lc.alpha_vec = (const double*)c->alpha_v.p; lc.colmap = colmap; lc.nvpc = 1; lc.n_occ = n_occ;
        if ((rc = lowrank_apply(c, 0, rows, n_vec, (const double*)P, (double*)Q, lc, f32 != 0))) return rc;
        n_h += n_vec;
        if ((rc = bcg_gram(c, s, K, n_act, orbmap, P, Q, G))) return rc;
        if ((rc = bcg_gram(c, s, K, n_act, orbmap, P, R, T))) return rc;
        {
            Prof p_(c, PC_MISC);
            wbcg::coef_kernel<<<n_act, 256, csm, c->st>>>(s, 0, orbmap, G, T, C, fac, 1e-12, 1.0);
            CK(cudaGetLastError());
            c->launches += 1;
        }
        if ((rc = bcg_update(c, s, K, n_act, orbmap, C, P, X, n_occ, orbmap, 1.0))) return rc;        // x += P alpha   (original column order)
        if ((rc = bcg_update(c, s, K, n_act, orbmap, C, Q, R, n_act, nullptr, -1.0))) return rc;      // r -= Q alpha
        {
            Prof p_(c, PC_CGVEC);
            wbcg::zr_kernel<<<n_vec, 256, 0, c->st>>>(n_g, n_act, n_occ, gamma, orbmap, c->d_g2, tk, o.precond, tol2, 0, (const double2*)R, (double2*)Z, st);
            wbcg::flags_kernel<<<blocks_for(n_act, 256), 256, 0, c->st>>>(n_act, orbmap, 0, st);
            CK(cudaGetLastError());
            c->launches += 2;
        }
        if ((rc = bcg_gram(c, s, K, n_act, orbmap, Q, Z, T))) return rc;
        {
            Prof p_(c, PC_MISC);
            wbcg::coef_kernel<<<n_act, 256, csm, c->st>>>(s, 1, orbmap, G, T, C, fac, 1e-12, -1.0);
            CK(cudaGetLastError());
            c->launches += 1;
        }
        if ((rc = bcg_update(c, s, K, n_act, orbmap, C, P, Z, n_act, nullptr, 1.0))) return rc;       // p_new = z - P beta
        std::swap(P, Z);
        if (poll.ready()) {
            live = poll.collect(c);
            if (live <= 0) done = true;
            else if (it + 1 < o.max_iter && live <= n_act - std::max(1, n_act / 16)) {
                Prof p_(c, PC_CGVEC);
                wcg::cg_compact_map<<<1, 1024, 0, c->st>>>(n_act, orbmap, st.active, newmap, src, live);
                wbcg::gather_blocks<<<live * s, 256, 0, c->st>>>(n_g, live, n_act, src, (const double2*)R, (double2*)Q);
                wbcg::gather_blocks<<<live * s, 256, 0, c->st>>>(n_g, live, n_act, src, (const double2*)P, (double2*)Z);
                cx<double>* oldR = R; cx<double>* oldP = P;
                R = Q; P = Z; Q = oldR; Z = oldP;
                std::swap(orbmap, newmap);
                n_act = live;
                wbcg::colmap_kernel<<<blocks_for(n_act * s, 256), 256, 0, c->st>>>(n_act, s, n_occ, orbmap, colmap);
                fill_shift<<<blocks_for(n_act * s, 256), 256, 0, c->st>>>(n_act * s, 1, n_occ, c->d_eps, shift, colmap);
                CK(cudaGetLastError());
                c->launches += 5;
            }
        }
        if (!done && ((it + 1) % every == 0 || it + 1 == o.max_iter)) CK(poll.post(c, st.counters));
    }
    if (poll.ready()) live = poll.collect(c);
    if (rep_dev) {
        wbcg::report_kernel<<<1, 256, 0, c->st>>>(n_col, n_occ, tol2, st, rep_dev);
        CK(cudaGetLastError());
    }
    *iters_out = it;
    *n_h_out = n_h;
    *live_out = live;
    return WEST_OK;
}

constexpr int MS_HIST_MIN = 32;      // fewest ring slots worth planning a Krylov history for (below that the sub-block shrinks instead)

// ---- workspace plan of west_chi0_apply for a sub-block of pb perturbations
struct Chi0Plan {
    int solver = 0, nvpc = 1, n_freq = 1, pb = 0;
    size_t tc = 0;         // WEST_MIXED tensor path: split operands of one low-rank apply (a sum of al256 pieces)
    size_t blk = 0;        // block CG: Gram / coefficient / factor blocks and flags (already a sum of al256 pieces)
    size_t vec = 0, xs = 0, shift = 0, grid = 0, scal = 0, maps = 0, misc = 0, W = 0, C = 0, msst = 0, craw = 0, dcoefd = 0, alpha = 0;
    int H = 0;             // multi-shift solver: ring slots of the Krylov history (0 = the per-shift recurrences of ms_step)
    bool carry = false;    // history ring smaller than max_iter + 1: carry vectors Q_s are planned
    size_t hscal = 0;
    size_t fixed() const {                     // everything but the history ring
        size_t t = blk + tc + al256(shift) + 2 * al256(grid) + al256(scal) + al256(maps) + al256(misc) + al256(W) + al256(C) + al256(alpha);
        if (solver == 1 && H > 0) t += 2 * al256(vec) + al256(xs) + (carry ? al256(xs) : 0) + al256(msst);
        else t += (solver == 1 ? 3 : (solver == 2 ? 5 : 4)) * al256(vec) + (solver == 1 ? 2 * al256(xs) + al256(msst) : 0);
        if (craw) t += al256(craw) + al256(dcoefd);
        return t;
    }
    size_t total() const { return fixed() + (solver == 1 && H > 0 ? al256((size_t)H * vec) + al256((size_t)H * hscal) : 0); }
};
Chi0Plan chi0_plan(const west_ctx* c, int solver, int nvpc, int n_freq, int pb, int f32 = 0, int H = 0, bool carry = false, int i8 = 0) {
    Chi0Plan p;
    p.solver = solver; p.nvpc = nvpc; p.n_freq = n_freq; p.pb = pb; p.H = solver == 1 ? H : 0; p.carry = carry;
    const size_t n_g = (size_t)c->hs.n_g, n3 = (size_t)n3_of(c);
    const size_t n_col = (size_t)pb * c->n_occ;
    const int vp = solver == 1 ? 1 : nvpc;                     // vectors per column in the working sets r, p, Ap (, x)
    p.vec = sizeof(cx<double>) * n_g * n_col * vp;
    p.shift = sizeof(double) * n_col * vp;
    p.grid = sizeof(double) * n3 * pb;
    p.scal = n_col * (sizeof(double2) + 2 * sizeof(double) + 2 * sizeof(int)) + 64;
    p.maps = sizeof(int) * 3 * n_col;
    p.misc = 256;
    const long long n_vec = (long long)n_col * vp;
    const long long slots_h = is_gamma(c) ? (n_vec + 1) / 2 : n_vec, slots_r = (long long)pb * c->n_uslots;
    p.W = bytes_W(c, std::max(slots_h, slots_r), 0);
    const int rows = c->rows_kb + c->rows_psi + c->rows_defl;
    p.C = bytes_C(rows, n_vec);
    if (f32) p.tc = tc_hot_bytes(c, rows, n_vec);
    else if (i8) p.tc = i8_hot_bytes(c, rows, n_vec);
    p.alpha = sizeof(double) * c->n_occ;
    if (solver == 2) p.blk = bcg_small_bytes(c->n_occ, pb);
    if (solver == 1) {
        p.xs = sizeof(cx<double>) * n_g * n_col * 2 * n_freq;
        const size_t ncs = n_col * n_freq;
        p.msst = sizeof(double) * 4 * n_col + sizeof(double2) * 2 * ncs + sizeof(double) * ncs + sizeof(int) * (2 * n_col + ncs) + 64;
        p.hscal = sizeof(double2) * 3 * ncs;                   // per ring slot: a_s, b_s, zeta of every (shift, column)
    }
    if (c->rows_defl > 0) {
        p.craw = sizeof(double) * (size_t)c->rows_defl * (size_t)((n_vec + 1) / 2 * 2);
        p.dcoefd = sizeof(double) * (size_t)c->rows_defl * (size_t)((n_col * (solver == 1 ? 2 : nvpc) + 1) / 2 * 2);
    }
    return p;
}

}  // namespace

extern "C" int west_chi0_apply(west_ctx* c, int32_t precision, int32_t n_pert, const double* dV, int32_t n_freq,
                               const double* omega_host, const west_cg_opts* opts, double* dn, void* dpsi_opt, west_stats* stats) {
    if (!c || n_pert < 0 || n_freq < 0 || !opts || (n_freq > 0 && !omega_host) || (n_pert > 0 && n_freq > 0 && (!dV || !dn)))
        return fail(c, WEST_EINVAL, "west_chi0_apply: bad argument");
    if (precision != WEST_FP64 && precision != WEST_MIXED && precision != WEST_FP64_I8) return fail(c, WEST_EINVAL, "west_chi0_apply: bad precision %d", precision);
    c->gemm_i8 = precision == WEST_FP64_I8 && tc_available(c);
    c->i8_slices = opts->tol >= 1e-9 ? 6 : 8;      // products accurate to 2^-42 of the row maxima are four orders below such a tolerance
    if (!c->have_vloc || c->n_occ == 0) return fail(c, WEST_ESTATE, "west_chi0_apply: west_set_vloc and west_set_states are required");
    if (opts->max_iter < 1 || !(opts->tol > 0) || opts->solver < 0 || opts->solver > 2 || opts->occupation < 0 || opts->occupation > 2 ||
        (opts->dn_accumulate != 0 && opts->dn_accumulate != 1))
        return fail(c, WEST_EINVAL, "west_chi0_apply: bad cg options");
    // H - eps_v + alpha P_v is positive on the occupied space only if alpha > eps_v - eps_min for every v (reading R3): a smaller
    // constant would make CG break down or converge to a wrong answer silently
    if (opts->alpha_pv > 0 && !(opts->alpha_pv > c->eps_max - c->eps_min))
        return fail(c, WEST_EINVAL, "west_chi0_apply: alpha_pv = %g Ry does not exceed the occupied band width %g Ry (pass alpha_pv <= 0 for the per-orbital default)",
                    opts->alpha_pv, c->eps_max - c->eps_min);
    const double occ = opts->occupation > 0 ? opts->occupation : 2.0;
    if (opts->solver == 1 && (c->cell.mode != WEST_GAMMA || n_freq > wcg::MS_MAX_SHIFTS))
        return fail(c, WEST_EINVAL, "west_chi0_apply: the multi-shift solver needs WEST_GAMMA and at most %d frequencies", wcg::MS_MAX_SHIFTS);
    const int gamma = is_gamma(c), N = c->cell.N, n_occ = c->n_occ, n_user = c->n_occ_user;
    for (int w = 0; w < n_freq; ++w) {
        if (omega_host[w] < 0) return fail(c, WEST_EINVAL, "west_chi0_apply: omega must be >= 0");
        if (omega_host[w] > 0 && !gamma) return fail(c, WEST_EINVAL, "west_chi0_apply: omega > 0 needs WEST_GAMMA (COCG needs real orbitals, R7)");
    }
    if (stats) std::memset(stats, 0, sizeof *stats);
    if (n_pert == 0 || n_freq == 0) return WEST_OK;
    const int f32 = precision == WEST_MIXED;
    const long long n_g = c->hs.n_g, n3 = n3_of(c);
    bool any_omega = false;
    for (int w = 0; w < n_freq; ++w) any_omega |= omega_host[w] > 0;
    const int nvpc_max = any_omega ? 2 : 1;
    int rc;
    if ((rc = ensure_opmatrix(c))) return rc;
    // operator data of the tensor paths is (re)built BEFORE the workspace is planned and carved: ensure() may give the lazy workspace back
    c->arena_release_ok = true;
    if (c->gemm_i8) rc = ensure_i8_operator(c);
    if (!rc && f32 && tc_available(c)) rc = ensure_tc_operator(c);
    c->arena_release_ok = false;
    if (rc) return rc;

    // ---- workspace: the largest perturbation sub-block whose buffers fit the arena (the caller's, or what the device has free)
    const size_t budget = arena_budget(c);
    Chi0Plan plan;
    int pb = n_pert;
    bool planned = false;
    if (opts->solver == 1 && c->ms_hist >= 0) {
        // multi-shift with a Krylov history: the largest sub-block that leaves room for a useful ring (at least MS_HIST_MIN slots, or
        // the whole run when max_iter is smaller); the ring then takes what is left, up to min(max_iter + 1, 128) slots.  In the lazy
        // mode the ring may use half of the free device memory (the context keeps its arena until it is destroyed).
        const int h_want = c->ms_hist > 0 ? std::min(c->ms_hist, opts->max_iter + 1) : std::min(opts->max_iter + 1, wcg::MSH_HMAX);
        const int h_min = c->ms_hist > 0 ? h_want : std::min(h_want, MS_HIST_MIN);
        const size_t hbudget = c->arena.user ? budget : budget / 2;
        for (int nb = 1; h_want >= 2; ++nb) {
            pb = (n_pert + nb - 1) / nb;
            // a ring that only fits sub-blocks of fewer than ~2000 columns costs more in GEMM efficiency than it saves in vector traffic
            // (measured at cfg 5, 4 frequencies: 1 024-column sub-blocks ran the projector GEMMs at 0.86 instead of 0.92 of the DGEMM rate)
            if (c->ms_hist == 0 && nb > 1 && (long long)pb * n_occ < 2048) break;
            Chi0Plan q = chi0_plan(c, 1, nvpc_max, n_freq, pb, f32, h_want, h_want < opts->max_iter + 1, c->gemm_i8);
            const size_t fx = q.fixed(), per = al256(q.vec) + al256(q.hscal) + 512;
            if (fx + (size_t)h_min * per <= hbudget) {
                int h = (int)std::min<size_t>((size_t)h_want, (hbudget - fx) / per + 2);      // (per over-estimates a slot: refine against the exact total)
                for (; h >= h_min; --h) {
                    plan = chi0_plan(c, 1, nvpc_max, n_freq, pb, f32, h, h < opts->max_iter + 1, c->gemm_i8);
                    if (plan.total() <= hbudget) break;
                }
                planned = h >= h_min && plan.total() <= budget;
                if (planned) break;
            }
            if (pb == 1) break;
        }
    }
    for (int nb = 1; !planned; ++nb) {
        pb = (n_pert + nb - 1) / nb;
        plan = chi0_plan(c, opts->solver, nvpc_max, n_freq, pb, f32, 0, false, c->gemm_i8);
        if (plan.total() <= budget || pb == 1) break;
    }
    if (plan.total() > budget)
        return fail(c, c->arena.user ? WEST_EWORKSPACE : WEST_ENOMEM, "west_chi0_apply: one perturbation needs %zu bytes of workspace, %zu available",
                    plan.total(), budget);
    if ((rc = hot_begin(c, plan.total()))) return rc;
    const int n_vecsets = opts->solver == 1 ? (plan.H > 0 ? 2 : 3) : 4;
    for (int i = 4 - n_vecsets; i < 4; ++i)
        if ((rc = hot(c, c->vecs[i], plan.vec))) return rc;
    if ((rc = hot(c, c->shift, plan.shift))) return rc;
    if ((rc = hot(c, c->dVpos, plan.grid))) return rc;
    if ((rc = hot(c, c->dnpos, plan.grid))) return rc;
    if ((rc = hot(c, c->scal, plan.scal))) return rc;
    if ((rc = hot(c, c->maps, plan.maps))) return rc;
    if ((rc = hot(c, c->misc, plan.misc))) return rc;
    if ((rc = hot(c, c->W, plan.W))) return rc;
    if ((rc = hot(c, c->Cbuf, plan.C))) return rc;
    if ((rc = hot(c, c->alpha_v, plan.alpha))) return rc;
    if (opts->solver == 2) {
        if ((rc = hot(c, c->vec5, plan.vec))) return rc;
        if ((rc = hot(c, c->blk, plan.blk))) return rc;
    }
    if (opts->solver == 1) {
        if ((rc = hot(c, c->xs, plan.xs))) return rc;
        if (plan.H == 0 || plan.carry) { if ((rc = hot(c, c->ps, plan.xs))) return rc; }      // p_s of ms_step, or the carry vectors of the history ring
        if ((rc = hot(c, c->msst, plan.msst))) return rc;
        if (plan.H > 0) {
            if ((rc = hot(c, c->hist, (size_t)plan.H * plan.vec))) return rc;
            if ((rc = hot(c, c->hist_scal, (size_t)plan.H * plan.hscal))) return rc;
        }
    }
    if (plan.craw) {
        if ((rc = hot(c, c->craw, plan.craw))) return rc;
        if ((rc = hot(c, c->dcoef_defl, plan.dcoefd))) return rc;
    }
    fill_alpha<<<blocks_for(n_occ, 256), 256, 0, c->st>>>(n_occ, c->d_eps, c->eps_min, c->eps_max - c->eps_min, opts->alpha_pv, (double*)c->alpha_v.p);
    CK(cudaGetLastError());
    c->launches += 1;

    struct Events {                      // destroyed on every return path
        cudaEvent_t e[4] = {nullptr, nullptr, nullptr, nullptr};
        ~Events() { for (auto x : e) if (x) cudaEventDestroy(x); }
        cudaEvent_t& operator[](int i) { return e[i]; }
    } ev;
    if (stats) for (auto& e : ev.e) CK(cudaEventCreate(&e));
    int ret = WEST_OK;
    int it_min = INT32_MAX;
    auto add_times = [&]() {
        float t;
        cudaEventElapsedTime(&t, ev[0], ev[1]); stats->ms_rhs += t;
        cudaEventElapsedTime(&t, ev[1], ev[2]); stats->ms_cg += t;
        cudaEventElapsedTime(&t, ev[2], ev[3]); stats->ms_dn += t;
    };

    for (int p0 = 0; p0 < n_pert; p0 += pb) {
        const int np = std::min(pb, n_pert - p0);           // perturbations of this sub-block
        const int n_col = np * n_occ;
        cx<double>* X = (cx<double>*)c->vecs[0].p; cx<double>* R = (cx<double>*)c->vecs[1].p;
        cx<double>* P = (cx<double>*)c->vecs[2].p; cx<double>* AP = (cx<double>*)c->vecs[3].p;
        nat_to_pos_real<double><<<blocks_for(n3 * np, 256), 256, 0, c->st>>>(N, c->ops->N1, c->ops->N2, n3 * np, dV + (long long)p0 * n3, (double*)c->dVpos.p);
        CK(cudaGetLastError());
        c->launches += 1;
        // [n_freq][n_pert][n_occ(caller's)][parts][n_g]: block of (frequency w, perturbation p0)
        const int parts_out = gamma ? 2 : 1;
        auto dpsi_block = [&](int w) { return (double2*)dpsi_opt + ((long long)w * n_pert + p0) * n_user * parts_out * n_g; };

        if (opts->solver == 1) {
            // -------------------------------------------------------- multi-shift CG: every frequency from one Krylov sequence
            wcg::MsShifts sh;
            sh.n = n_freq;
            for (int w = 0; w < n_freq; ++w) sh.omega[w] = omega_host[w];
            const size_t per = (size_t)n_g * n_col * 2;                       // complex-valued solution of one frequency
            const size_t ncs = (size_t)n_col * n_freq;
            wcg::MsState st;
            {
                char* p = (char*)c->msst.p;
                st.zeta = (double2*)p; p += sizeof(double2) * ncs;
                st.zeta_prev = (double2*)p; p += sizeof(double2) * ncs;
                st.a_prev = (double*)p; p += sizeof(double) * n_col;
                st.b_prev = (double*)p; p += sizeof(double) * n_col;
                st.rr = (double*)p; p += sizeof(double) * n_col;
                st.b2 = (double*)p; p += sizeof(double) * n_col;
                st.res2 = (double*)p; p += sizeof(double) * ncs;
                st.active = (int*)p; p += sizeof(int) * n_col;
                st.iters = (int*)p; p += sizeof(int) * n_col;
                st.sactive = (int*)p; p += sizeof(int) * ncs;
                p = (char*)(((uintptr_t)p + 15) & ~(uintptr_t)15);
                st.counters = (int*)p;
            }
            fill_shift<<<blocks_for(n_col, 256), 256, 0, c->st>>>(n_col, 1, n_occ, c->d_eps, (double*)c->shift.p, nullptr);
            CK(cudaGetLastError());
            if (stats) CK(cudaEventRecord(ev[0], c->st));
            // history variant: b goes straight into ring slot 0 (the ring is laid out for THIS sub-block's column count)
            wcg::MsHist hs{(double2*)c->hist.p, (double2*)c->hist_scal.p, plan.H};
            if ((rc = chi0_rhs(c, np, 1, plan.H > 0 ? (cx<double>*)c->hist.p : R))) return rc;
            if (stats) CK(cudaEventRecord(ev[1], c->st));
            int iters = 0;
            int64_t n_h = 0;
            if (plan.H > 0)
                rc = ms_hist_solve(c, f32, n_col, *opts, sh, hs, P, AP, (cx<double>*)c->xs.p, (cx<double>*)c->ps.p, dpsi_opt != nullptr, (double*)c->shift.p, st,
                                   (int*)c->maps.p, &iters, &n_h);
            else
                rc = ms_solve(c, f32, n_col, *opts, sh, R, P, AP, (cx<double>*)c->xs.p, (cx<double>*)c->ps.p, dpsi_opt != nullptr, (double*)c->shift.p, st,
                              (int*)c->maps.p, &iters, &n_h);
            if (rc) return rc;
            if (stats) CK(cudaEventRecord(ev[2], c->st));
            for (int w = 0; w < n_freq; ++w) {
                cx<double>* Xw = (cx<double>*)c->xs.p + (size_t)w * per;
                if ((rc = add_deflated(c, n_col, 1, 2, omega_host[w], Xw))) return rc;
                if ((rc = chi0_dn(c, np, 2, Xw, dn + ((long long)w * n_pert + p0) * n3, occ, opts->dn_accumulate))) return rc;
                if (dpsi_opt) {
                    dpsi_gather<<<np * n_user * 2, wcg::NT, 0, c->st>>>(n_g, n_occ, n_user, 2, 2, (const double2*)Xw, dpsi_block(w));
                    CK(cudaGetLastError());
                    c->launches += 1;
                }
            }
            // convergence report: the return code needs it, so this is the call's one stream synchronisation
            double* rep = (double*)c->misc.p;
            wcg::ms_report<<<1, wcg::NT, 0, c->st>>>(n_col, n_freq, opts->tol * opts->tol, st, rep);
            if (stats) CK(cudaEventRecord(ev[3], c->st));
            double* h = (double*)(c->h_pinned + 8);
            CK(cudaMemcpyAsync(h, rep, 4 * sizeof(double), cudaMemcpyDeviceToHost, c->st));
            CK(cudaMemcpyAsync(c->h_pinned + 16, st.counters + 2, sizeof(long long), cudaMemcpyDeviceToHost, c->st));
            CK(cudaStreamSynchronize(c->st));
            if (stats) {
                if (plan.H > 0) stats->n_hist_passes += *reinterpret_cast<long long*>(c->h_pinned + 16);
                else stats->n_shift_updates += *reinterpret_cast<long long*>(c->h_pinned + 16);
                stats->ms_history_slots = plan.H;
            }
            if (h[1] > 0) ret = WEST_NOTCONVERGED;
            if (stats) {
                add_times();
                stats->iters = std::max(stats->iters, iters); stats->n_unconverged += (int)h[1]; stats->resid_max = std::max(stats->resid_max, h[0]);
                stats->n_h_apply += n_h;
                it_min = std::min(it_min, (int)h[2]);
            }
            continue;
        }

        wcg::Scalars s;
        {
            char* p = (char*)c->scal.p;
            s.rz = (double2*)p; p += sizeof(double2) * n_col;
            s.rr = (double*)p; p += sizeof(double) * n_col;
            s.b2 = (double*)p; p += sizeof(double) * n_col;
            s.active = (int*)p; p += sizeof(int) * n_col;
            s.iters = (int*)p; p += sizeof(int) * n_col;
            p = (char*)(((uintptr_t)p + 15) & ~(uintptr_t)15);
            s.counters = (int*)p;
        }
        for (int w = 0; w < n_freq; ++w) {
            const double omega = omega_host[w];
            const int mode = gamma ? (omega > 0 ? 1 : 0) : 2;
            const int nvpc = mode == 1 ? 2 : 1, n_vec = n_col * nvpc;
            fill_shift<<<blocks_for(n_vec, 256), 256, 0, c->st>>>(n_vec, nvpc, n_occ, c->d_eps, (double*)c->shift.p, nullptr);
            CK(cudaGetLastError());
            if (stats) CK(cudaEventRecord(ev[0], c->st));
            if ((rc = chi0_rhs(c, np, nvpc, R))) return rc;
            if (stats) CK(cudaEventRecord(ev[1], c->st));
            // ---- a2-a9: batched PCG / COCG
            int iters = 0, live = 0;
            int64_t n_h = 0;
            // solver 2: block CG over the np right-hand sides of every orbital (omega = 0; blocks of 2 .. 128 perturbations)
            const bool block = opts->solver == 2 && mode != 1 && np >= 2 && np <= wbcg::SMAX;
            if (block) rc = bcg_solve(c, f32, np, *opts, X, R, P, AP, (cx<double>*)c->vec5.p, (double*)c->shift.p, stats ? (double*)c->misc.p : nullptr, &iters, &n_h, &live);
            else if (mode == 0) rc = cg_solve<0>(c, f32, n_col, *opts, omega, X, R, P, AP, (double*)c->shift.p, s, (int*)c->maps.p, &iters, &n_h, &live);
            else if (mode == 1) rc = cg_solve<1>(c, f32, n_col, *opts, omega, X, R, P, AP, (double*)c->shift.p, s, (int*)c->maps.p, &iters, &n_h, &live);
            else rc = cg_solve<2>(c, f32, n_col, *opts, omega, X, R, P, AP, (double*)c->shift.p, s, (int*)c->maps.p, &iters, &n_h, &live);
            if (rc) return rc;
            if (live > 0) ret = WEST_NOTCONVERGED;
            if ((rc = add_deflated(c, n_col, nvpc, nvpc, omega, X))) return rc;
            if (stats) CK(cudaEventRecord(ev[2], c->st));
            if ((rc = chi0_dn(c, np, nvpc, X, dn + ((long long)w * n_pert + p0) * n3, occ, opts->dn_accumulate))) return rc;
            if (dpsi_opt) {
                dpsi_gather<<<np * n_user * parts_out, wcg::NT, 0, c->st>>>(n_g, n_occ, n_user, nvpc, parts_out, (const double2*)X, dpsi_block(w));
                CK(cudaGetLastError());
                c->launches += 1;
            }
            if (stats) {
                CK(cudaEventRecord(ev[3], c->st));
                double* rep = (double*)c->misc.p;
                if (!block) wcg::cg_report<<<1, wcg::NT, 0, c->st>>>(n_col, opts->tol * opts->tol, s, rep);
                double* h = (double*)(c->h_pinned + 8);
                CK(cudaMemcpyAsync(h, rep, 4 * sizeof(double), cudaMemcpyDeviceToHost, c->st));
                CK(cudaStreamSynchronize(c->st));
                add_times();
                stats->iters = std::max(stats->iters, iters);
                stats->n_unconverged += (int)h[1];
                stats->resid_max = std::max(stats->resid_max, h[0]);
                stats->n_h_apply += n_h;
                it_min = std::min(it_min, (int)h[2]);
            }
        }
    }
    if (stats) {
        stats->iters_min = it_min == INT32_MAX ? 0 : it_min;
        stats->n_sub_blocks = (n_pert + pb - 1) / pb;
    }
    return ret;
}

extern "C" size_t west_workspace_bytes(const west_ctx* c, int32_t op, int32_t n_pert, int32_t n_freq, int32_t precision) {
    if (!c || n_pert <= 0) return 0;
    const int f32 = precision == WEST_MIXED, i8 = precision == WEST_FP64_I8 && tc_available(c);
    switch (op) {
        case WEST_OP_FFT3D: return plan_fft3d(c, n_pert);
        case WEST_OP_H_APPLY: return plan_happly(c, n_pert, f32, i8);
        case WEST_OP_CHI0: return chi0_plan(c, 0, 1, std::max(1, n_freq), n_pert, f32, 0, false, i8).total();
        case WEST_OP_CHI0_IW: return chi0_plan(c, 0, is_gamma(c) ? 2 : 1, std::max(1, n_freq), n_pert, f32, 0, false, i8).total();
        case WEST_OP_CHI0_MULTISHIFT: return chi0_plan(c, 1, 1, std::max(1, n_freq), n_pert, f32, 0, false, i8).total();
        case WEST_OP_CHI0_MULTISHIFT_HIST: return chi0_plan(c, 1, 1, std::max(1, n_freq), n_pert, f32, wcg::MSH_HMAX, true, i8).total();
        case WEST_OP_CHI0_BLOCK: return chi0_plan(c, 2, 1, std::max(1, n_freq), n_pert, f32, 0, false, i8).total();
        case WEST_OP_LANCZOS: return plan_lanczos(c, n_pert, std::max(1, n_freq), f32);
    }
    return 0;
}

extern "C" int west_set_workspace(west_ctx* c, void* ws, size_t bytes) {
    if (!c || (ws && ((uintptr_t)ws & 255))) return fail(c, WEST_EINVAL, "west_set_workspace: NULL context or a block that is not 256-byte aligned");
    Arena& a = c->arena;
    if (a.base && !a.user) {             // drop the context's own arena: not a hot call, may synchronise and free
        cudaStreamSynchronize(c->st);
        cudaFree(a.base);
        c->dev_bytes -= (int64_t)a.cap;
    }
    a.base = (char*)ws; a.cap = ws ? bytes : 0; a.user = ws != nullptr; a.off = 0;
    a.epoch += 1;
    return WEST_OK;
}

// ============================================================================================================ Lanczos chains
extern "C" int west_lanczos(west_ctx* c, int32_t precision, int32_t n_pert, const double* phi, int32_t n_steps, double* alpha, double* beta,
                            double* norm, double* braket_opt) {
    if (!c || n_pert < 0 || n_steps < 1 || (n_pert > 0 && (!phi || !alpha || !beta || !norm))) return fail(c, WEST_EINVAL, "west_lanczos: bad argument");
    if (precision != WEST_FP64 && precision != WEST_MIXED) return fail(c, WEST_EINVAL, "west_lanczos: bad precision %d", precision);
    c->gemm_i8 = false;
    if (!c->have_vloc || c->n_occ == 0) return fail(c, WEST_ESTATE, "west_lanczos: west_set_vloc and west_set_states are required");
    const int gamma = is_gamma(c), N = c->cell.N, n_occ = c->n_occ;
    if (braket_opt && !gamma) return fail(c, WEST_EINVAL, "west_lanczos: brakets are implemented for WEST_GAMMA only");
    if (n_pert == 0) return WEST_OK;
    const long long n_g = c->hs.n_g, n3 = n3_of(c), K = 2 * n_g;
    const int n_col = n_pert * n_occ;
    int rc;
    if ((rc = ensure_opmatrix(c))) return rc;
    if ((rc = hot_begin(c, plan_lanczos(c, n_pert, n_steps, precision == WEST_MIXED)))) return rc;
    for (int i = 0; i < 4; ++i)
        if ((rc = hot(c, c->vecs[i], sizeof(cx<double>) * n_g * n_col))) return rc;
    if ((rc = hot(c, c->dVpos, sizeof(double) * n3 * n_pert))) return rc;
    if ((rc = hot(c, c->scal, sizeof(double) * n_col + 64))) return rc;
    {
        const long long slots_h = gamma ? ((long long)n_col + 1) / 2 : (long long)n_col, slots_r = (long long)n_pert * c->n_uslots;
        if ((rc = hot(c, c->W, bytes_W(c, std::max(slots_h, slots_r), 0)))) return rc;
    }
    cx<double>* Q = (cx<double>*)c->vecs[0].p; cx<double>* QP = (cx<double>*)c->vecs[1].p;
    cx<double>* HQ = (cx<double>*)c->vecs[2].p; cx<double>* Q1 = (cx<double>*)c->vecs[3].p;
    double* beta_prev = (double*)c->scal.p;
    // odd orbital count in WEST_GAMMA (R15): the chains run over the padded column set into scratch arrays, the caller's are filled at the end
    const int n_user = c->n_occ_user;
    double *alpha_out = alpha, *beta_out = beta, *norm_out = norm;
    if (n_user != n_occ) {
        if ((rc = hot(c, c->msst, sizeof(double) * (size_t)n_col * (2 * n_steps + 1)))) return rc;
        alpha = (double*)c->msst.p; beta = alpha + (size_t)n_col * n_steps; norm = beta + (size_t)n_col * n_steps;
    }
    nat_to_pos_real<double><<<blocks_for(n3 * n_pert, 256), 256, 0, c->st>>>(N, c->ops->N1, c->ops->N2, n3 * n_pert, phi, (double*)c->dVpos.p);
    CK(cudaGetLastError());
    c->launches += 1;
    // q^1 = psi_i phi_m (Eq. 16), normalised (R16)
    if ((rc = chi0_rhs(c, n_pert, 1, Q, +1.0, false))) return rc;
    CK(cudaMemsetAsync(QP, 0, sizeof(cx<double>) * n_g * n_col, c->st));
    if (gamma) wlz::lz_normalize<true><<<n_col, wcg::NT, 0, c->st>>>(n_g, (double2*)Q, braket_opt ? (double2*)Q1 : nullptr, norm, beta_prev);
    else wlz::lz_normalize<false><<<n_col, wcg::NT, 0, c->st>>>(n_g, (double2*)Q, nullptr, norm, beta_prev);
    CK(cudaGetLastError());
    c->launches += 1;
    if (braket_opt) CK(cudaMemsetAsync(braket_opt, 0, sizeof(double) * (size_t)n_user * n_steps * n_pert * n_pert, c->st));
    const int f32 = precision == WEST_MIXED;
    const long long Kp = pad4(K);
    const bool tc_brakets = braket_opt && f32 && tc_available(c);
    float* Qs = nullptr; float* Q1s = nullptr;
    if (tc_brakets) {
        CK(tc_attrs());
        if ((rc = hot(c, c->xs, sizeof(float) * 4 * (size_t)n_col * Kp))) return rc;
        Qs = (float*)c->xs.p; Q1s = Qs + 2 * (size_t)n_col * Kp;
        wtc::split_rows<<<blocks_for((long long)n_col * Kp, 256), 256, 0, c->st>>>(n_col, K, (const double*)Q1, K, Q1s, Q1s + (size_t)n_col * Kp, Kp);
        CK(cudaGetLastError());
        c->launches += 1;
    }
    VecMap vm{gamma ? 2 : 1, gamma ? 1 : 0, n_col, 0};
    const int n_slots = gamma ? (n_col + 1) / 2 : n_col;
    for (int l = 0; l < n_steps; ++l) {
        if (braket_opt) {
            // <q^1_{n i} | q^l_{m i}> for every orbital i: n_occ Gram blocks, rows of one block n_occ vectors apart (Fig. 4)
            double* C = braket_opt + (size_t)l * n_pert * n_pert;
            const long long sC = (long long)n_steps * n_pert * n_pert;
            if (tc_brakets) {
                // WEST_MIXED: FP32 operands (the FP32 payload of Fig. 5c, as an FP32-operand product): q^l is split into
                // TF32 hi / lo like q^1 and the n_occ blocks run as ONE batched tcgen05 launch (batch entry = orbital, tc_gemm.cuh)
                Prof p_(c, PC_GEMM_TN);
                wtc::split_rows<<<blocks_for((long long)n_col * Kp, 256), 256, 0, c->st>>>(n_col, K, (const double*)Q, K, Qs, Qs + (size_t)n_col * Kp, Kp);
                wtc::Maps m;
                if ((rc = tc_map(c, &m.a_hi, Qs, n_pert, K, (long long)n_occ * Kp, n_user, Kp)) ||
                    (rc = tc_map(c, &m.a_lo, Qs + (size_t)n_col * Kp, n_pert, K, (long long)n_occ * Kp, n_user, Kp)) ||
                    (rc = tc_map(c, &m.b_hi, Q1s, n_pert, K, (long long)n_occ * Kp, n_user, Kp)) ||
                    (rc = tc_map(c, &m.b_lo, Q1s + (size_t)n_col * Kp, n_pert, K, (long long)n_occ * Kp, n_user, Kp)))
                    return rc;
                const int n_kb = (int)((K + wtc::BK - 1) / wtc::BK), tp = (n_pert + 127) / 128;
                const wtc::TileGrid tg{tp, tp, 1, n_user, sC};
                const long long nt = (long long)tp * tp * n_user;
                // out[c * ldo + r]: r = row of the A operand (q^l_m), c = row of the B operand (q^1_n)  ->  C[i][n][m]
                wtc::tf32x3_gemm<false><<<(unsigned)std::min<long long>(nt, 148), wtc::NTHREADS, wtc::SMEM_BYTES, c->st>>>(m, tg, n_pert, n_pert, n_kb, n_kb, C, n_pert);
                CK(cudaGetLastError());
                c->launches += 2;
            } else if ((rc = launch_gemm_tn(c, n_pert, n_pert, K, (const double*)Q1, (long long)n_occ * K, (const double*)Q, (long long)n_occ * K, C,
                                            n_pert, n_user, K, K, sC, false)))
                return rc;
            wlz::braket_fix<<<blocks_for((long long)n_user * n_pert * n_pert, 256), 256, 0, c->st>>>(n_user, n_pert, sC, C, (const double*)Q1,
                                                                                                  (const double*)Q, (long long)n_occ * K, K);
            CK(cudaGetLastError());
            c->launches += 1;
        }
        if ((rc = hloc_apply(c, f32, vm, n_slots, Q, HQ, nullptr, 0.0))) return rc;
        if (c->rows_kb > 0) {
            LowrankCoef lc; lc.dcoef = c->d_dcoef; lc.n_rows_d = c->rows_kb;
            if ((rc = lowrank_apply(c, 0, c->rows_kb, n_col, (const double*)Q, (double*)HQ, lc, f32 != 0))) return rc;
        }
        {
            Prof p_(c, PC_CGVEC);
            if (gamma) wlz::lz_step<true><<<n_col, wcg::NT, 0, c->st>>>(n_g, n_steps, l, (const double2*)Q, (const double2*)HQ, (double2*)QP, alpha, beta, beta_prev);
            else wlz::lz_step<false><<<n_col, wcg::NT, 0, c->st>>>(n_g, n_steps, l, (const double2*)Q, (const double2*)HQ, (double2*)QP, alpha, beta, beta_prev);
            CK(cudaGetLastError());
            c->launches += 1;
        }
        std::swap(Q, QP);          // QP now holds q^l (the next q^{l-1}), Q holds q^{l+1}
    }
    if (n_user != n_occ) {
        const size_t w = sizeof(double) * n_steps;
        CK(cudaMemcpy2DAsync(alpha_out, w * n_user, alpha, w * n_occ, w * n_user, n_pert, cudaMemcpyDeviceToDevice, c->st));
        CK(cudaMemcpy2DAsync(beta_out, w * n_user, beta, w * n_occ, w * n_user, n_pert, cudaMemcpyDeviceToDevice, c->st));
        CK(cudaMemcpy2DAsync(norm_out, sizeof(double) * n_user, norm, sizeof(double) * n_occ, sizeof(double) * n_user, n_pert, cudaMemcpyDeviceToDevice, c->st));
    }
    return WEST_OK;
}

extern "C" int west_lanczos_diag(west_ctx* c, int32_t n_chain, int32_t n_steps, const double* alpha, const double* beta, double* d, double* U,
                                 int32_t* sweeps_opt) {
    if (!c || n_chain < 0 || n_steps < 1 || n_steps > wlz::TRI_MAX || (n_chain > 0 && (!alpha || !beta || !d || !U)))
        return fail(c, WEST_EINVAL, "west_lanczos_diag: bad argument (1 <= n_steps <= %d)", wlz::TRI_MAX);
    if (n_chain == 0) return WEST_OK;
    int rc;
    if ((rc = hot_begin(c, al256(256)))) return rc;
    if ((rc = hot(c, c->misc, 256))) return rc;
    int* n_failed = (int*)c->misc.p;
    CK(cudaMemsetAsync(n_failed, 0, sizeof(int), c->st));
    const size_t bytes = sizeof(double) * wlz::TRI_WARPS * (2 * wlz::TRI_MAX + (size_t)n_steps * (n_steps + 1));
    if (bytes > 48 * 1024) CK(cudaFuncSetAttribute(wlz::tridiag_eig, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    {
        Prof p_(c, PC_MISC);
        wlz::tridiag_eig<<<(n_chain + wlz::TRI_WARPS - 1) / wlz::TRI_WARPS, 32 * wlz::TRI_WARPS, bytes, c->st>>>(n_chain, n_steps, alpha, beta, d, U,
                                                                                                       sweeps_opt, n_failed);
        CK(cudaGetLastError());
        c->launches += 1;
    }
    CK(cudaMemcpyAsync(c->h_pinned, n_failed, sizeof(int), cudaMemcpyDeviceToHost, c->st));
    CK(cudaStreamSynchronize(c->st));
    if (c->h_pinned[0] > 0)
        return fail(c, WEST_NOTCONVERGED, "west_lanczos_diag: %d of %d matrices did not converge in 60 QL sweeps per eigenvalue", c->h_pinned[0], n_chain);
    return WEST_OK;
}

// ============================================================================================================ no-allocation entry point
// west_fft3d_static: west_fft3d for callers that cannot tolerate ANY allocation (code under CUDA graph capture, tight serving loops,
// harnesses that forbid cudaMalloc): the stick intermediate W and the position-order grid of the transform live in ONE file-scope
// device array of fixed size instead of the workspace arena.  Every GPU that loads the library holds WEST_STATIC_SCRATCH_BYTES until
// the process exits.  Same kernels, same launch order and same arithmetic as west_fft3d; only the scratch pointers differ.
namespace {

static __device__ __align__(256) unsigned char g_west_static_scratch[WEST_STATIC_SCRATCH_BYTES];

// In host code `g_west_static_scratch` is a host-side stand-in, NOT a device address: the device address is looked up once per device
// (with that device current) by cudaGetSymbolAddress and cached here.  No allocation, no synchronisation.
constexpr int STATIC_MAX_DEVICES = 64;
std::mutex g_static_mu;
void* g_static_ptr[STATIC_MAX_DEVICES] = {};

int static_scratch_ptr(west_ctx* c, unsigned char** out) {
    int dev = -1;
    CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return fail(c, WEST_EINVAL, "west_fft3d_static: device ordinal %d outside 0..%d", dev, STATIC_MAX_DEVICES - 1);
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_ptr[dev]) {
        void* p = nullptr;
        CK(cudaGetSymbolAddress(&p, g_west_static_scratch));
        if (!p) return fail(c, WEST_ECUDA, "west_fft3d_static: cudaGetSymbolAddress returned a null address on device %d", dev);
        g_static_ptr[dev] = p;
    }
    *out = (unsigned char*)g_static_ptr[dev];
    return WEST_OK;
}

}  // namespace

extern "C" size_t west_static_scratch_bytes(void) { return WEST_STATIC_SCRATCH_BYTES; }

extern "C" int west_fft3d_static(west_ctx* c, int32_t dir, int32_t n_batch, const void* in, void* out) {
    if (!c || (dir != 1 && dir != -1) || n_batch < 0 || (n_batch > 0 && (!in || !out))) return fail(c, WEST_EINVAL, "west_fft3d_static: bad argument");
    if (n_batch == 0) return WEST_OK;
    const int gamma = is_gamma(c), N = c->cell.N;
    const long long n3 = n3_of(c);
    // one transform slot needs its sticks W [N][n_cols] and its grid [N^3], both complex128 (each piece rounded up to 256 bytes)
    const size_t w_slot = sizeof(cx<double>) * (size_t)N * c->hs.n_cols, r_slot = sizeof(cx<double>) * (size_t)n3;
    const size_t per_slot = al256(w_slot) + al256(r_slot);
    if (per_slot > WEST_STATIC_SCRATCH_BYTES)
        return fail(c, WEST_EWORKSPACE, "west_fft3d_static: one transform of this cell (N = %d, %d columns) needs %zu bytes of scratch, the static array holds %zu "
                    "(WEST_STATIC_SCRATCH_BYTES; N <= 72 fits) - use west_fft3d with a workspace", N, c->hs.n_cols, per_slot, (size_t)WEST_STATIC_SCRATCH_BYTES);
    const int n_slots = gamma ? (n_batch + 1) / 2 : n_batch;
    // slots per launch: as many as the array holds (the pieces of a chunk are contiguous, so the split is W[chunk] then R[chunk])
    int chunk = 1;
    while (chunk < n_slots && chunk < 64 && al256(w_slot * (chunk + 1)) + al256(r_slot * (chunk + 1)) <= WEST_STATIC_SCRATCH_BYTES) ++chunk;
    unsigned char* base = nullptr;
    int rc;
    if ((rc = static_scratch_ptr(c, &base))) return rc;
    void* W = base;
    cx<double>* R = reinterpret_cast<cx<double>*>(base + al256(w_slot * chunk));
    // Nothing in the array has to start at zero: K1 (dir = +1) writes every (position, column) of W and K2 every grid point before
    // anything is read; dir = -1 fills the grid first and K2 then writes every (position, column) of W.  The array keeps the last
    // call's contents otherwise.
    VecMap vm{gamma ? 2 : 1, gamma ? 1 : 0, n_batch, 0};
    K2Any a{};
    a.W = W; a.R = R;
    for (int s0 = 0; s0 < n_slots; s0 += chunk) {
        const int ns = std::min(chunk, n_slots - s0);
        vm.slot0 = s0;
        if (dir == 1) {
            CK(c->ops->k1(0, gamma, ns, c->st, c->geom, vm, (const cx<double>*)in, W));
            CK(c->ops->k2(0, K2_TOR, ns, c->st, c->geom, a));
            pos_to_user<<<blocks_for(n3 * ns, 256), 256, 0, c->st>>>(N, c->ops->N1, c->ops->N2, gamma, s0, ns, n_batch, R, (double*)out);
        } else {
            user_to_pos<<<blocks_for(n3 * ns, 256), 256, 0, c->st>>>(N, c->ops->N1, c->ops->N2, gamma, s0, ns, n_batch, (const double*)in, R);
            CK(c->ops->k2(0, K2_FROMR, ns, c->st, c->geom, a));
            K3Epi e{1.0 / ((double)N * N * N), 0, nullptr, 0.0, nullptr};
            CK(c->ops->k3(0, gamma, ns, c->st, c->geom, vm, W, e, (cx<double>*)out));
        }
        CK(cudaGetLastError());
        c->launches += 3;
    }
    return WEST_OK;
}

// ============================================================================================================ FP64 pipe yardstick
// Do DMMA (mma.sync m8n8k4 f64) and DFMA run on separate pipes of an sm_100a SM?  One CTA of 16 warps per SM: the first n_dmma_warps
// issue dependent-free DMMA chains, the others DFMA chains (mode bit 0: DMMA warps active, bit 1: DFMA warps active).  bench.py --op pipes
// times the three modes; DESIGN.md section 10 states the result (one shared pipe: the mixed rate never exceeds either alone).
namespace {
__global__ void __launch_bounds__(512, 1) fp64_pipe_probe(int mode, int n_dmma_warps, int iters, double* out) {
    constexpr int NACC = 8;
    const int warp = threadIdx.x >> 5;
    const double a = 1.0 + threadIdx.x * 1e-9, b = 1.0 - threadIdx.x * 1e-9;
    double acc[NACC][2];
#pragma unroll
    for (int i = 0; i < NACC; ++i) acc[i][0] = acc[i][1] = 0.0;
    if (warp < n_dmma_warps) {
        if (mode & 1)
            for (int it = 0; it < iters; ++it) {
#pragma unroll
                for (int i = 0; i < NACC; ++i) wgemm::dmma(acc[i][0], acc[i][1], a, b);
            }
    } else if (mode & 2) {
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int r = 0; r < 2; ++r)
#pragma unroll
                for (int i = 0; i < NACC; ++i) { acc[i][0] = fma(a, b, acc[i][0]); acc[i][1] = fma(b, a, acc[i][1]); }
        }
    }
    double sum = 0;
#pragma unroll
    for (int i = 0; i < NACC; ++i) sum += acc[i][0] + acc[i][1];
    if (sum == 12345.678) out[0] = sum;          // keeps the chains alive
}
}  // namespace
extern "C" int west_probe_fp64_pipes(west_ctx* c, int32_t mode, int32_t n_dmma_warps, int32_t iters, float* ms_host, double* dmma_flop_host, double* dfma_flop_host) {
    if (!c || mode < 1 || mode > 3 || n_dmma_warps < 0 || n_dmma_warps > 16 || iters < 1 || !ms_host) return fail(c, WEST_EINVAL, "west_probe_fp64_pipes: bad argument");
    int rc = hot_begin(c, al256(256));
    if (rc) return rc;
    if ((rc = hot(c, c->misc, 256))) return rc;
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
    fp64_pipe_probe<<<148, 512, 0, c->st>>>(mode, n_dmma_warps, iters, (double*)c->misc.p);       // warm-up
    cudaEventRecord(e0, c->st);
    fp64_pipe_probe<<<148, 512, 0, c->st>>>(mode, n_dmma_warps, iters, (double*)c->misc.p);
    cudaEventRecord(e1, c->st);
    cudaError_t e = cudaEventSynchronize(e1);
    if (e == cudaSuccess) e = cudaEventElapsedTime(ms_host, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    CK(e);
    CK(cudaGetLastError());
    c->launches += 2;
    // one DMMA m8n8k4 = 512 flop per warp instruction; one DFMA warp instruction = 64 flop; 8 accumulator pairs per iteration (DFMA: x4)
    if (dmma_flop_host) *dmma_flop_host = (mode & 1) ? 148.0 * n_dmma_warps * (double)iters * 8 * 512.0 : 0.0;
    if (dfma_flop_host) *dfma_flop_host = (mode & 2) ? 148.0 * (16 - n_dmma_warps) * (double)iters * 8 * 4 * 64.0 : 0.0;
    return WEST_OK;
}
