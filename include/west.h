/* west.h - C ABI of the B200-native chi0*dV hot path of arXiv 2203.05623 (Yu & Govoni).
 *
 * What the library computes (citations are /root/reference/PAPER.md lines):
 *   Eq. 10   (h - eps_i) P_c dpsi_i^j = -P_c v_j^pert psi_i,  P_c = 1 - P_v,
 *                           solved "by a preconditioned conjugate gradient method";
 *   Eq. 11   dn_j(r) = sum_sigma sum_i [psi_i^* dpsi_i^j + c.c.];
 *   dual-space H application "kinetic operator and local potential are applied in the reciprocal or direct
 *                           space ... at least two FFTs (one forward and one backward)";
 *   sphere-truncated FFT    "retains only the Fourier components that correspond to a chosen kinetic energy
 *                           cutoff".
 * Readings of everything the paper leaves open (alpha*P_v, preconditioner, tolerance, i*omega, ordering of G,
 * FFT sign and scale, synthetic pseudopotential) are listed in DESIGN.md section 3 and referenced here as (Rn).
 *
 * Conventions
 *   Units: Rydberg atomic units, kinetic energy |G|^2 Ry, G = (2 pi / L) n, n integer triple, cubic cell of side L bohr.
 *   Sphere (R2): S = { n : |n|^2 <= n2max }, stored in ascending lexicographic order of the signed triple
 *     (n_x, n_y, n_z).  mode WEST_FULL stores all of S (n_g = |S|) and vectors are complex functions.
 *     mode WEST_GAMMA stores the tail of that list starting at n = 0 (n_g = (|S|+1)/2: n = 0 and every triple whose
 *     first non-zero component is positive) and every vector is a REAL function of r, c(-G) = conj c(G), c(0) real.
 *   Coefficient blocks: row-major [vector][n_g], interleaved complex128 (re, im), G fastest.
 *   Grids: [ix][iy][iz], z fastest, N^3 points, r = (L/N)(ix, iy, iz).  Real grids are f64, complex grids c128.
 *   FFT (R10): G->r  f(r_j) = sum_G c(G) exp(+i G.r_j)          (unscaled)
 *              r->G  c(G)   = (1/N^3) sum_j f(r_j) exp(-i G.r_j) (truncated to S)
 *   Requires N even and N >= 4*floor(sqrt(n2max)) + 1 (products of two sphere-limited functions alias-free);
 *     supported N: 24, 36, 48, 72, 144.
 *
 * Ownership and streams
 *   Every pointer is a DEVICE pointer owned by the caller unless marked "host".  Device memory is allocated only by
 *   west_create and west_set_* (operator data: COPIES of what the caller passes, so the caller may free its arrays
 *   after the call returns; the copy is enqueued on the stream).  The HOT calls (west_fft3d, west_h_apply,
 *   west_chi0_apply, west_lanczos, west_lanczos_diag, the GEMMs, west_fft3d_dense) take all scratch memory from ONE
 *   workspace block:
 *     - west_set_workspace(ctx, ws, bytes): the caller's block.  A hot call then performs no cudaMalloc, no cudaFree
 *       and no implicit stream synchronisation for memory; it fails with WEST_EWORKSPACE if the block is too small
 *       (west_workspace_bytes gives the size; west_chi0_apply also accepts a smaller block and then walks the
 *       perturbations in sub-blocks, as long as one perturbation fits).
 *     - no workspace set (the default, convenient for tests): the context owns the block and regrows it when a call needs
 *       more (that call synchronises the stream, frees and reallocates); west_chi0_apply sizes its sub-blocks by the
 *       device's free memory (cudaMemGetInfo).
 *   All work is enqueued on the CUDA stream given to west_create (a cudaStream_t passed as void*; NULL = the legacy
 *   default stream).  Calls are asynchronous with respect to the host except: west_chi0_apply returns after its last CG
 *   iteration has been QUEUED and the one before has FINISHED (the host reads one live-column counter per poll, one
 *   iteration late, through an event - it never drains the stream inside the solve; with stats_opt != NULL or the
 *   multi-shift solver it synchronises once per frequency / sub-block to read the report); west_lanczos_diag
 *   synchronises once; west_get_profile synchronises.  A context is not thread-safe; distinct contexts are independent.
 *
 * Determinism
 *   west_fft3d, west_h_apply's FFT part, the CG vector kernels and the per-column scalars are deterministic.  Two places
 *   use FP64 atomicAdd, so their results can differ in the last bits (<= 1e-15 relative) from run to run: the dn
 *   accumulation over the occupied states (step a10), and the split-K partial sums of west_gemm_tn (KB / P_v overlaps)
 *   whenever the contraction is split over more than one CTA (the CG iterates, and hence dpsi and dn, inherit that).
 *
 * Errors
 *   Every int-returning call returns 0 on success, a negative WEST_E* on a hard error (nothing useful written) or the
 *   positive WEST_NOTCONVERGED (outputs written; stats say how many columns hit max_iter).  The message of the last
 *   error is kept per context (west_last_error).  No exceptions cross the ABI, nothing calls exit().
 *   There is no CPU fallback: without a CUDA device west_create fails with WEST_ECUDA.
 */
#ifndef WEST_H
#define WEST_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define WEST_OK            0
#define WEST_NOTCONVERGED  1
#define WEST_EINVAL       -1
#define WEST_ECUDA        -2
#define WEST_ESTATE       -3   /* a required west_set_* has not been called */
#define WEST_ENOMEM       -4
#define WEST_EWORKSPACE   -5   /* the workspace set by west_set_workspace is too small for this call */

#define WEST_FULL   0
#define WEST_GAMMA  1

#define WEST_FP64   0   /* everything in FP64 */
#define WEST_MIXED  1   /* inside H*psi: FFT + real-space multiply in FP32, KB / P_v projector GEMMs as 3xTF32 tensor-core products
                           (FP32 class, FP64 operands in memory); vectors, CG dots, RHS projection, dn in FP64 */
/* operations of west_workspace_bytes */
#define WEST_OP_FFT3D            0   /* west_fft3d,      n_pert = n_batch */
#define WEST_OP_H_APPLY          1   /* west_h_apply,    n_pert = n_vec */
#define WEST_OP_CHI0             2   /* west_chi0_apply, solver 0, every omega = 0 (PCG) */
#define WEST_OP_CHI0_IW          3   /* west_chi0_apply, solver 0, some omega > 0 (COCG: two real vectors per column) */
#define WEST_OP_CHI0_MULTISHIFT  4   /* west_chi0_apply, solver 1, n_freq frequencies */
#define WEST_OP_LANCZOS          5   /* west_lanczos, n_freq = n_steps */
#define WEST_OP_CHI0_BLOCK       6   /* west_chi0_apply, solver 2, every omega = 0 (block CG: five vector sets) */
#define WEST_OP_CHI0_MULTISHIFT_HIST 7 /* west_chi0_apply, solver 1 with room for a full 128-slot Krylov history for all n_pert perturbations as one
                                        block (the fast variant; WEST_OP_CHI0_MULTISHIFT is the smallest comfortable size, and any block in
                                        between is used for as many ring slots as fit) */

#define WEST_FP64_I8 3  /* west_h_apply / west_chi0_apply: everything in FP64 as WEST_FP64, except that the KB / P_v projector GEMMs inside H*psi form
                           their FP64 products from error-free int8 slices on the INT8 tensor path (tcgen05 kind::i8, int32 accumulation in
                           tensor memory; csrc/i8_gemm.cuh): every operand row is cut into 8 signed 7-bit slices below
                           its own power-of-two scale (2^-56 of the row's largest element is dropped), slice pairs contract exactly in
                           int32, the weight classes are summed in FP64.  Same parity bar as WEST_FP64 (1e-9); the RHS projection and the
                           deflation update stay on DMMA.  west_chi0_apply with opts->tol >= 1e-9 uses 6 slices (2^-42 of the row maxima,
                           four orders below such a tolerance; 21 instead of 36 slice-pair products); tighter tolerances and west_h_apply
                           use 8.  Falls back to WEST_FP64 when the driver offers no tensor-map encoder. */
#define WEST_FP32   2   /* west_fft3d_dense only: complex64 data and arithmetic (the FP32 curves of Fig. 3) */

typedef struct west_ctx west_ctx;

typedef struct {
    double  L;       /* cell side, bohr */
    int32_t n2max;   /* integer sphere radius^2: floor(E_cut L^2 / 4 pi^2) (R2: the inclusion test is integer) */
    int32_t N;       /* FFT grid points per axis */
    int32_t mode;    /* WEST_FULL | WEST_GAMMA */
} west_cell;

typedef struct {
    int32_t max_iter;   /* iteration cap per column (R5), e.g. 500 */
    double  tol;        /* stop when ||r||_2 <= tol * ||b||_2 per column (R5) */
    double  alpha_pv;   /* alpha of the alpha*P_v term (R3); the converged result does not depend on it.  > 0: one constant for every
                           column; it must exceed the occupied band width eps_max - eps_min (else H - eps_v + alpha P_v is indefinite
                           and CG can converge to a wrong answer: WEST_EINVAL).  <= 0: the per-orbital default
                           alpha_v = (eps_v - eps_min) + (eps_max - eps_min)/2 */
    int32_t precond;    /* 0: none; 1: M_v(G) = 1/max(1, |G|^2/(1.35 <psi_v|T|psi_v>)) (R4); 2: Teter-Payne-Allan polynomial form */
    int32_t check_every;/* host polls convergence every this many iterations (>=1) */
    int32_t solver;     /* 0: one preconditioned PCG (omega = 0) / COCG (omega > 0) solve per frequency (R7);
                           1: multi-shift CG (WEST_GAMMA only, <= 16 frequencies): all frequencies from ONE unpreconditioned Krylov
                              sequence of the real seed operator H - eps_v + alpha P_v, one H*psi per iteration for every omega.  The
                              shifted solutions are contracted from the seed residuals, which are kept in a ring of up to 128 vectors
                              per column when the workspace has room (west_set_ms_history); else per-shift vector recurrences;
                           2: block CG: at omega = 0 the n_pert right-hand sides of one orbital share ONE Krylov space (Gram
                              matrices of the search block, rank-revealing pivoted-Cholesky solves that drop dependent directions, csrc/
                              bcg_kernels.cuh); same dpsi, fewer H*psi.  Blocks of 2 .. 128 perturbations (per sub-block); frequencies
                              omega > 0 and other block sizes run as solver 0 */
    double  occupation; /* electrons per orbital in Eq. 11: 2 = spin-unpolarised (0 selects this default), 1 = ONE channel of a
                           spin-polarised system (N_spin = 2): dn = (2 occupation / Omega) Re sum_v ... */
    int32_t dn_accumulate; /* 0: dn is overwritten; 1: dn += this call's response (second spin channel: the sum over sigma) */
} west_cg_opts;

typedef struct {            /* host struct, filled when non-NULL (one stream synchronisation per frequency and sub-block) */
    int32_t iters;          /* CG iterations launched (max over frequencies / sub-blocks; with the lagged poll one more than the slowest column needed) */
    int32_t iters_min;      /* fewest iterations any (non-zero) column took part in before it converged */
    int32_t n_sub_blocks;   /* perturbation sub-blocks the call was split into to fit the workspace (1 = none) */
    int32_t n_unconverged;  /* columns above tol at exit */
    double  resid_max;      /* max over columns of ||r|| / ||b|| (recurrence residual) */
    int64_t n_h_apply;      /* vectors pushed through H in this call (real functions in GAMMA mode) */
    int64_t n_shift_updates;/* multi-shift solver: (column, frequency) vector updates performed (frozen frequencies are skipped) */
    float   ms_rhs, ms_cg, ms_dn;   /* CUDA-event times of the three phases */
    int64_t n_hist_passes;  /* multi-shift solver with the Krylov history: column-vector passes (16 n_g bytes each) of the history contractions */
    int32_t ms_history_slots; /* multi-shift solver: ring slots of the Krylov history used (0 = per-shift recurrences) */
} west_stats;

/* Context. cuda_stream: cudaStream_t as void*. */
int  west_create (west_ctx** ctx, const west_cell* cell, void* cuda_stream);
int  west_destroy(west_ctx* ctx);
const char* west_last_error(const west_ctx* ctx);   /* ctx may be NULL: last error of a failed west_create */

/* Workspace of the hot calls (the paper's rule behind it: "data are copied to the GPU once ... and copied back only
 * for I/O", PAPER.md:171, 183 - nothing is allocated or moved inside the solve).
 * west_workspace_bytes: bytes the operation `op` (WEST_OP_*) needs for n_pert perturbations (vectors / grids for the FFT and H ops) and
 *   n_freq frequencies (Lanczos: steps) at `precision`, with the operator data currently set (call it after west_set_kb / west_set_states /
 *   west_set_deflation).  0 for a bad argument.  For the chi0 ops this is the size that runs all n_pert perturbations as ONE block.
 * west_set_workspace: ws = DEVICE block of `bytes` bytes, 256-byte aligned, owned by the caller and retained until replaced or
 *   west_destroy; ws = NULL returns to the context-owned lazy block.  Not a hot call (it may free the context's own block).
 *   Errors: WEST_EINVAL (NULL ctx, misaligned block). */
size_t west_workspace_bytes(const west_ctx* ctx, int32_t op, int32_t n_pert, int32_t n_freq, int32_t precision);
int    west_set_workspace(west_ctx* ctx, void* ws, size_t bytes);

/* Step a0 - the sphere S and its maps, computed on the HOST with integer arithmetic only.
 * All output pointers are HOST pointers, any may be NULL.  miller [n_g][3]; fft_index[n_g] = ((n_x mod N) N + (n_y mod N)) N
 * + (n_z mod N); fft_index_minus[n_g] = the same for -G; g2[n_g] = |G|^2 in Ry.  Order and n_g follow cell.mode. */
int  west_gsphere(const west_ctx* ctx, int64_t* n_g, int32_t* miller, int32_t* fft_index, int32_t* fft_index_minus, double* g2);

/* Operator data (device pointers, copied).  vloc [N^3] f64.  beta [n_proj][n_g] c128 in the storage of cell.mode
 * (in GAMMA mode each projector must be a real function of r), dcoef [n_proj] f64 HOST: V_NL = sum_k |beta_k> D_k <beta_k|
 * (Kleinman-Bylander, R12).  psi [n_occ][n_g] c128 orthonormal occupied orbitals (sum_G |c|^2 = 1 over the FULL sphere),
 * eps [n_occ] f64 HOST eigenvalues in Ry: the inputs psi_i, eps_i of Eq. 10. n_proj = 0 removes V_NL.
 * n_occ may be odd in either mode (WEST_GAMMA pads internally with a zero orbital, which no output ever contains). */
int  west_set_vloc  (west_ctx* ctx, const double* vloc);
int  west_set_kb    (west_ctx* ctx, int32_t n_proj, const void* beta, const double* dcoef_host);
int  west_set_states(west_ctx* ctx, int32_t n_occ, const void* psi, const double* eps_host);

/* Optional deflation for west_chi0_apply (not in the paper; exact, not a truncation): n_defl eigenstates of H directly ABOVE the
 * occupied ones (psi_c [n_defl][n_g] c128 orthonormal, device; eps_c [n_defl] HOST), e.g. the guard states an eigensolver returns
 * anyway.  Their part of every solution is added in closed form, dpsi_low = - sum_c psi_c <psi_c|dV psi_v> / (eps_c - eps_v - i omega),
 * and the CG runs on the complement (the states join P_v in the alpha-projector and the right-hand side is projected off them), so
 * the smallest eigenvalue of the Sternheimer operator rises from the gap to eps_(first state not given) - eps_v and the iteration
 * count drops.  Costs n_defl more rows in the projector GEMMs.  n_defl = 0 switches it off.  The result is unchanged (tested). */
int  west_set_deflation(west_ctx* ctx, int32_t n_defl, const void* psi_c, const double* eps_c_host);

/* Sphere-truncated 3D FFT (R10).
 * dir = +1: in = coefficients [n_batch][n_g] c128, out = grids.   dir = -1: in = grids, out = coefficients.
 * WEST_FULL:  grids are complex [n_batch][N^3] c128.
 * WEST_GAMMA: vectors are real functions, grids are REAL [n_batch][N^3] f64 (two are packed per complex transform
 *             internally; an odd trailing vector is padded).
 * r->G of data that is not sphere-limited is the truncation to S of its DFT. */
int  west_fft3d(west_ctx* ctx, int32_t dir, int32_t precision, int32_t n_batch, const void* in, void* out);

/* West_fft3d without ANY allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid it): the transform's scratch (stick intermediate + position-order grid, the two buffers west_fft3d takes from
 * the workspace) lives in ONE file-scope device array of WEST_STATIC_SCRATCH_BYTES = 8 MiB inside the library, which every GPU that
 * loads the library holds until the process exits.  Same kernels and arithmetic as west_fft3d (WEST_FP64), same argument meaning:
 * dir = +1: in = coefficients [n_batch][n_g] c128, out = grids; dir = -1: in = grids, out = coefficients; in / out are the caller's
 * device buffers.  The call performs no cudaMalloc, no cudaFree, no allocating library routine and no synchronisation; the first call
 * on a device looks the array's address up (cudaGetSymbolAddress, once per device, with the caller's current device = the context's).
 * Limit: one transform slot (N n_cols + N^3 complex128) must fit the array - N <= 72 does, N = 144 does not: WEST_EWORKSPACE with the
 * sizes in west_last_error, nothing enqueued.  Larger batches are walked in chunks of as many slots as fit.
 * EVERY call on a device shares the array, across contexts and streams: calls that overlap on the GPU race (serialise them on one
 * stream or with events).  The array keeps the last call's contents; nothing in it has to be cleared, because every element a kernel
 * reads has been written earlier in the same call.  Errors: WEST_EINVAL, WEST_EWORKSPACE, WEST_ECUDA. */
#define WEST_STATIC_SCRATCH_BYTES (8u << 20)
int    west_fft3d_static(west_ctx* ctx, int32_t dir, int32_t n_batch, const void* in, void* out);
size_t west_static_scratch_bytes(void);   /* = WEST_STATIC_SCRATCH_BYTES */

/* Dense complex-to-complex 3D FFT on an n^3 cubic grid: the operation timed in Fig. 3 (one FP64 or FP32 C2C
 * transform of a 128^3 or 256^3 grid, data resident on the device).  Independent of the context's cell: ctx supplies the stream,
 * the error string and the launch counter only.
 *   out[b][k_x][k_y][k_z] = sum_r in[b][r_x][r_y][r_z] exp(sign 2 pi i k.r / n),  sign = +1 or -1, no scaling (reading R17)
 * in, out: DEVICE pointers, [n_batch][n][n][n], z fastest, complex128 (precision = WEST_FP64) or complex64 (WEST_FP32), 16-byte
 * (8-byte) aligned; in == out (in place) is allowed, partial overlap is not.  n must be 64, 128 or 256; n_batch <= 65535.
 * Three launches (z, y, x passes) on the context's stream; no workspace.  Errors: WEST_EINVAL (NULL, unsupported n / precision / sign),
 * WEST_ECUDA. */
int  west_fft3d_dense(west_ctx* ctx, int32_t n, int32_t sign, int32_t precision, int32_t n_batch, const void* in, void* out);

/* y = H x = (T + V_loc + V_NL) x for n_vec vectors, x and y [n_vec][n_g] c128 (Eq. 1).
 * x and y must not overlap.  Needs west_set_vloc; V_NL only if west_set_kb was called with n_proj > 0. */
int  west_h_apply(west_ctx* ctx, int32_t precision, int32_t n_vec, const void* x, void* y);

/* dn = chi0(i omega) dV for a block of perturbations (Eq. 10-11; R3-R9).
 *   dV     [n_pert][N^3] f64 real perturbing potentials on the grid (Ry)
 *   omega  [n_freq] HOST, imaginary frequencies in Ry, >= 0; omega = 0 runs real-symmetric PCG, omega > 0 runs COCG (R7)
 *   dn     [n_freq][n_pert][N^3] f64: dn_i(r) = (4/Omega) Re sum_v conj(u_v(r)) du_iv(r)  (e/bohr^3, spin-unpolarised, R9/R11)
 *   dpsi_opt  NULL, or the converged solutions:
 *             WEST_FULL  [n_freq][n_pert][n_occ][n_g] c128
 *             WEST_GAMMA [n_freq][n_pert][n_occ][2][n_g] c128 - real part and imaginary part of dpsi as two real functions
 *   stats_opt NULL or HOST struct.
 * For every (frequency w, perturbation i, occupied state v) it forms b = -P_c (dV_i psi_v), solves
 * (H - eps_v - i omega_w + alpha P_v) dpsi = b by batched (one recurrence per column) preconditioned CG and accumulates dn.
 * If the workspace cannot hold all n_pert perturbations at once they are processed in sub-blocks (stats: n_sub_blocks); the result
 * does not depend on the split.  Errors: WEST_EINVAL, WEST_ESTATE, WEST_EWORKSPACE / WEST_ENOMEM (not even one perturbation fits),
 * WEST_ECUDA; WEST_NOTCONVERGED (> 0) when a column hit max_iter. */
int  west_chi0_apply(west_ctx* ctx, int32_t precision, int32_t n_pert, const double* dV,
                     int32_t n_freq, const double* omega_host, const west_cg_opts* opts,
                     double* dn, void* dpsi_opt, west_stats* stats_opt);

/* Lanczos chains of the frequency-dependent step (Eq. 15-18; widening row SURVEY 8(f)-2).  For every function
 * phi_m and occupied orbital psi_i: q^1 = psi_i phi_m / ||psi_i phi_m|| (Eq. 16; the norm is returned, reading R16),
 * alpha^l = <q^l|H|q^l>, beta^{l+1} = ||(H - alpha^l) q^l - beta^l q^{l-1}||, q^{l+1} = that vector / beta^{l+1}; no
 * re-orthogonalisation.  H = T + V_loc + V_NL as in west_h_apply.
 *   phi    [n_pert][N^3] f64 real functions on the grid
 *   alpha  [n_pert][n_occ][n_steps] f64 (device), alpha[..][l] = alpha^{l+1}
 *   beta   [n_pert][n_occ][n_steps] f64 (device), beta[..][l]  = beta^{l+2} (the norm computed in step l)
 *   norm   [n_pert][n_occ] f64 (device), ||psi_i phi_m|| in the plane-wave 2-norm
 *   braket_opt NULL or [n_occ][n_steps][n_pert][n_pert] f64 (device, WEST_GAMMA only): <q^1_{n i} | q^{l+1}_{m i}>, the
 *          matrix product of Eq. 19 / Fig. 4 as n_occ batched DMMA Gram blocks per step. */
int  west_lanczos(west_ctx* ctx, int32_t precision, int32_t n_pert, const double* phi, int32_t n_steps, double* alpha, double* beta,
                  double* norm, double* braket_opt);

/* d and U of Eq. 19: "the eigenvalues and the eigenvectors of the tri-diagonal matrix that has alpha^l along the diagonal
 * and beta^l along the sub- and super-diagonal", for n_chain chains at once (one warp per matrix, implicit-shift QL with accumulated
 * plane rotations).  alpha, beta [n_chain][n_steps] f64 (device) exactly as west_lanczos returns them (beta[..][l] couples rows l and
 * l+1; the last entry of each row is not part of T).  d [n_chain][n_steps] ascending; U [n_chain][n_steps][n_steps] row-major,
 * U[l][l'] = component l of the eigenvector of d[l'], orthonormal, sign fixed by U[0][l'] >= 0.  sweeps_opt NULL or [n_chain] i32
 * (device): QL sweeps used, -1 = not converged.  1 <= n_steps <= 64.  Synchronises the stream once (to return WEST_NOTCONVERGED). */
int  west_lanczos_diag(west_ctx* ctx, int32_t n_chain, int32_t n_steps, const double* alpha, const double* beta, double* d, double* U,
                       int32_t* sweeps_opt);

/* Dense contraction building blocks (FP64 DMMA), exported for tests and the roofline bench.
 * C[m][n] = sum_k A[m][k] B[n][k]          (west_gemm_tn: both operands K-contiguous, row-major [rows][ld])
 * Y[n][k] += sum_m C[m][n] A[m][k]          (west_gemm_update)
 * All f64, device pointers; ld* are leading dimensions in elements. */
int  west_gemm_tn    (west_ctx* ctx, int32_t m, int32_t n, int64_t k, const double* A, int64_t lda,
                      const double* B, int64_t ldb, double* C, int64_t ldc);
int  west_gemm_update(west_ctx* ctx, int32_t m, int32_t n, int64_t k, const double* C, int64_t ldc,
                      const double* A, int64_t lda, double* Y, int64_t ldy);

/* Introspection for the bench: bytes of device memory the context currently holds, and the number of kernels it has
 * launched since creation (the bench's gpu_launches claim). */
int64_t west_device_bytes(const west_ctx* ctx);
int64_t west_launch_count(const west_ctx* ctx);
/* Optional per-kernel-class timing for the bench's roofline line.  While on, every kernel launch is bracketed by CUDA
 * events on the context's stream.  west_get_profile synchronises the stream, writes the summed milliseconds and span
 * counts of the 8 classes into the HOST arrays ms[8], count[8] and resets the record.  Classes: 0 K1 (sphere -> z sticks,
 * H*psi), 1 K2 (planes: y/x inverse, x V_loc, x/y forward), 2 K3 (z sticks -> sphere + kinetic), 3 gemm_tn, 4 gemm_update,
 * 5 CG vector kernel (fused step; compaction launches included), 6 FFT kernels of the RHS / dn stages (two launches per span), 7 block-CG Gram /
 * coefficient / block-update kernels and the tridiagonal eigensolver. */
int  west_set_profile(west_ctx* ctx, int32_t on);
int  west_get_profile(west_ctx* ctx, double* ms, int64_t* count);
/* Tuning knob: how many FFT slots (complex transforms) are processed per internal chunk (0 = default).  The stick
 * intermediate of a chunk is sized to stay L2-resident between the three FFT kernels. */
int  west_set_fft_chunk(west_ctx* ctx, int32_t n_slots);
/* Tuning knob: vector kernel of the CG iteration (steps a8 + a9).  0 (default): the column-resident kernel where a column fits one SM
 * (n_g <= 9216, omega = 0), else the streaming one; 1: always the streaming kernel; 2: the resident kernel with each column split
 * over a cluster of two CTAs (partial sums through distributed shared memory; same size limit).  Same results up to summation order.
 * Errors: WEST_EINVAL (NULL ctx, which not 0 / 1 / 2). */
int  west_set_cg_kernel(west_ctx* ctx, int32_t which);
/* Tuning knob of the multi-shift solver (west_cg_opts.solver = 1).  slots = 0 (default): keep the seed residuals of every column in a
 * ring of min(max_iter + 1, 128) vectors - fewer if the workspace is smaller, down to 32, below which the perturbation sub-block is
 * shrunk instead - and contract the shifted solutions x_s from them once per ring revolution (every history vector is read once for all
 * frequencies; carry vectors bridge the revolutions).  slots = -1: the per-shift vector recurrences (x_s and p_s updated in every
 * iteration: 6 vector passes per live shift and iteration, but only 3 + 4 n_freq vectors of workspace per column).  slots = 2 .. 128: that
 * ring size exactly (tests).  Same results up to summation order.  Errors: WEST_EINVAL. */
int  west_set_ms_history(west_ctx* ctx, int32_t slots);

/* Yardstick for the roofline statements of DESIGN.md section 10: do the FP64 tensor instruction (DMMA, what the projector GEMMs issue) and
 * the FP64 FMA instruction (what the FFT kernels issue) have separate pipes on this GPU?  One 16-warp CTA per SM (148 CTAs); the first
 * n_dmma_warps warps run independent DMMA chains, the other warps DFMA chains; mode bit 0 switches the DMMA warps on, bit 1 the DFMA warps.
 * Times one launch (after a warm-up launch) with CUDA events and synchronises.  ms_host: milliseconds; dmma_flop_host / dfma_flop_host
 * (may be NULL): floating-point operations each kind of warp executed in the timed launch.  Errors: WEST_EINVAL, WEST_ECUDA. */
int  west_probe_fp64_pipes(west_ctx* ctx, int32_t mode, int32_t n_dmma_warps, int32_t iters, float* ms_host, double* dmma_flop_host, double* dfma_flop_host);

#ifdef __cplusplus
}
#endif
#endif /* WEST_H */
