"""Thin ctypes binding of include/west.h: same names, argument marshalling only.

Device buffers are torch CUDA tensors (PyTorch is the allocator and stream provider); their ``data_ptr()`` is what crosses
the C ABI.  Host arrays are numpy.  Nothing here computes: every step of the path runs in libwest.so's kernels, and the
import fails loudly if the library is missing (no CPU fallback).
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libwest.so")

WEST_OK, WEST_NOTCONVERGED = 0, 1
WEST_EINVAL, WEST_ECUDA, WEST_ESTATE, WEST_ENOMEM, WEST_EWORKSPACE = -1, -2, -3, -4, -5
WEST_OP_FFT3D, WEST_OP_H_APPLY, WEST_OP_CHI0, WEST_OP_CHI0_IW, WEST_OP_CHI0_MULTISHIFT, WEST_OP_LANCZOS, WEST_OP_CHI0_BLOCK, WEST_OP_CHI0_MULTISHIFT_HIST = 0, 1, 2, 3, 4, 5, 6, 7
WEST_FULL, WEST_GAMMA = 0, 1
WEST_FP64, WEST_MIXED, WEST_FP32, WEST_FP64_I8 = 0, 1, 2, 3


class west_cell(C.Structure):
    _fields_ = [("L", C.c_double), ("n2max", C.c_int32), ("N", C.c_int32), ("mode", C.c_int32)]


class west_cg_opts(C.Structure):
    _fields_ = [("max_iter", C.c_int32), ("tol", C.c_double), ("alpha_pv", C.c_double), ("precond", C.c_int32),
                ("check_every", C.c_int32), ("solver", C.c_int32), ("occupation", C.c_double), ("dn_accumulate", C.c_int32)]


class west_stats(C.Structure):
    _fields_ = [("iters", C.c_int32), ("iters_min", C.c_int32), ("n_sub_blocks", C.c_int32), ("n_unconverged", C.c_int32), ("resid_max", C.c_double), ("n_h_apply", C.c_int64), ("n_shift_updates", C.c_int64),
                ("ms_rhs", C.c_float), ("ms_cg", C.c_float), ("ms_dn", C.c_float), ("n_hist_passes", C.c_int64), ("ms_history_slots", C.c_int32)]


EXPORTS = ["west_create", "west_destroy", "west_last_error", "west_gsphere", "west_set_vloc", "west_set_kb", "west_set_states", "west_set_deflation",
           "west_fft3d", "west_fft3d_static", "west_static_scratch_bytes", "west_fft3d_dense", "west_h_apply", "west_chi0_apply", "west_lanczos", "west_lanczos_diag", "west_gemm_tn", "west_gemm_update", "west_device_bytes",
           "west_launch_count", "west_workspace_bytes", "west_set_workspace", "west_set_fft_chunk", "west_set_cg_kernel", "west_set_ms_history", "west_probe_fp64_pipes", "west_set_profile", "west_get_profile"]


def load_library():
    if not os.path.exists(LIB_PATH):
        raise ImportError("%s is missing: run `python -m paper_2203_05623_b200.build` (there is no CPU fallback)" % LIB_PATH)
    lib = C.CDLL(LIB_PATH)
    vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    lib.west_create.argtypes = [C.POINTER(vp), C.POINTER(west_cell), vp]
    lib.west_destroy.argtypes = [vp]
    lib.west_last_error.argtypes = [vp]
    lib.west_last_error.restype = C.c_char_p
    lib.west_gsphere.argtypes = [vp, C.POINTER(i64), vp, vp, vp, vp]
    lib.west_set_vloc.argtypes = [vp, vp]
    lib.west_set_kb.argtypes = [vp, i32, vp, vp]
    lib.west_set_states.argtypes = [vp, i32, vp, vp]
    lib.west_set_deflation.argtypes = [vp, i32, vp, vp]
    lib.west_fft3d.argtypes = [vp, i32, i32, i32, vp, vp]
    lib.west_fft3d_dense.argtypes = [vp, i32, i32, i32, i32, vp, vp]
    lib.west_fft3d_static.argtypes = [vp, i32, i32, vp, vp]
    lib.west_static_scratch_bytes.argtypes = []
    lib.west_static_scratch_bytes.restype = C.c_size_t
    lib.west_h_apply.argtypes = [vp, i32, i32, vp, vp]
    lib.west_chi0_apply.argtypes = [vp, i32, i32, vp, i32, vp, C.POINTER(west_cg_opts), vp, vp, C.POINTER(west_stats)]
    lib.west_lanczos.argtypes = [vp, i32, i32, vp, i32, vp, vp, vp, vp]
    lib.west_lanczos_diag.argtypes = [vp, i32, i32, vp, vp, vp, vp, vp]
    lib.west_gemm_tn.argtypes = [vp, i32, i32, i64, vp, i64, vp, i64, vp, i64]
    lib.west_gemm_update.argtypes = [vp, i32, i32, i64, vp, i64, vp, i64, vp, i64]
    lib.west_device_bytes.argtypes = [vp]
    lib.west_device_bytes.restype = i64
    lib.west_launch_count.argtypes = [vp]
    lib.west_launch_count.restype = i64
    lib.west_workspace_bytes.argtypes = [vp, i32, i32, i32, i32]
    lib.west_workspace_bytes.restype = C.c_size_t
    lib.west_set_workspace.argtypes = [vp, vp, C.c_size_t]
    lib.west_set_fft_chunk.argtypes = [vp, i32]
    lib.west_set_cg_kernel.argtypes = [vp, i32]
    lib.west_set_ms_history.argtypes = [vp, i32]
    lib.west_probe_fp64_pipes.argtypes = [vp, i32, i32, i32, C.POINTER(C.c_float), C.POINTER(dbl), C.POINTER(dbl)]
    lib.west_set_profile.argtypes = [vp, i32]
    lib.west_get_profile.argtypes = [vp, vp, vp]
    for name in EXPORTS:
        getattr(lib, name)
        if name not in ("west_last_error", "west_device_bytes", "west_launch_count", "west_workspace_bytes", "west_static_scratch_bytes"):
            getattr(lib, name).restype = C.c_int
    return lib


class WestError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("west error %d: %s" % (code, msg))
        self.code = code


def _dev(t, dtype=None):
    """device pointer of a contiguous CUDA tensor"""
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError("expected a CUDA torch tensor")
    if not t.is_contiguous():
        raise ValueError("tensor must be contiguous")
    if dtype is not None and t.dtype != dtype:
        raise TypeError("expected dtype %s, got %s" % (dtype, t.dtype))
    return C.c_void_p(t.data_ptr())


class West:
    """One west_ctx.  Method names follow the C entry points (west_ prefix dropped)."""

    def __init__(self, L, n2max, N, mode, stream=None):
        import torch
        self.lib = load_library()
        self.cell = west_cell(float(L), int(n2max), int(N), int(mode))
        self.ctx = C.c_void_p()
        if stream is None:
            stream = torch.cuda.current_stream()
        self.stream = stream
        rc = self.lib.west_create(C.byref(self.ctx), C.byref(self.cell), C.c_void_p(stream.cuda_stream))
        if rc != 0:
            raise WestError(rc, (self.lib.west_last_error(None) or b"").decode())
        n_g = C.c_int64()
        self._ck(self.lib.west_gsphere(self.ctx, C.byref(n_g), None, None, None, None))
        self.n_g = int(n_g.value)
        self.N, self.mode, self.L = int(N), int(mode), float(L)
        self.n_occ = None          # set by set_states
        self._ws = None            # the caller's workspace tensor (kept alive while it is set)

    def _ck(self, rc):
        if rc < 0:
            raise WestError(rc, (self.lib.west_last_error(self.ctx) or b"").decode())
        return rc

    def close(self):
        if self.ctx:
            self.lib.west_destroy(self.ctx)
            self.ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def gsphere(self):
        miller = np.empty((self.n_g, 3), dtype=np.int32)
        idx = np.empty(self.n_g, dtype=np.int32)
        idxm = np.empty(self.n_g, dtype=np.int32)
        g2 = np.empty(self.n_g, dtype=np.float64)
        n = C.c_int64()
        self._ck(self.lib.west_gsphere(self.ctx, C.byref(n), miller.ctypes.data, idx.ctypes.data, idxm.ctypes.data, g2.ctypes.data))
        return miller, idx, idxm, g2

    def set_vloc(self, vloc):
        import torch
        assert vloc.numel() == self.N ** 3
        self._ck(self.lib.west_set_vloc(self.ctx, _dev(vloc, torch.float64)))

    def set_kb(self, beta, dcoef):
        import torch
        d = np.ascontiguousarray(dcoef, dtype=np.float64)
        n_proj = 0 if beta is None else int(beta.shape[0])
        if n_proj:
            assert beta.shape[1] == self.n_g and len(d) == n_proj
        self._ck(self.lib.west_set_kb(self.ctx, n_proj, _dev(beta, torch.complex128) if n_proj else None, d.ctypes.data if n_proj else None))

    def set_states(self, psi, eps):
        import torch
        e = np.ascontiguousarray(eps, dtype=np.float64)
        assert psi.shape[1] == self.n_g and len(e) == psi.shape[0]
        self._ck(self.lib.west_set_states(self.ctx, int(psi.shape[0]), _dev(psi, torch.complex128), e.ctypes.data))
        self.n_occ = int(psi.shape[0])

    def set_deflation(self, psi_c, eps_c):
        """n_defl eigenstates directly above the occupied ones (or None / empty to switch deflation off)."""
        import torch
        n = 0 if psi_c is None else int(psi_c.shape[0])
        e = np.ascontiguousarray(eps_c if n else [], dtype=np.float64)
        self._ck(self.lib.west_set_deflation(self.ctx, n, _dev(psi_c, torch.complex128) if n else None, e.ctypes.data if n else None))

    def fft3d(self, dir, x, out=None, precision=WEST_FP64):
        import torch
        N = self.N
        n_batch = int(x.shape[0])
        if dir == 1:
            assert x.shape[1] == self.n_g
            if out is None:
                out = torch.empty((n_batch, N, N, N), dtype=torch.float64 if self.mode == WEST_GAMMA else torch.complex128, device=x.device)
            self._ck(self.lib.west_fft3d(self.ctx, 1, precision, n_batch, _dev(x, torch.complex128), _dev(out)))
        else:
            if out is None:
                out = torch.empty((n_batch, self.n_g), dtype=torch.complex128, device=x.device)
            self._ck(self.lib.west_fft3d(self.ctx, -1, precision, n_batch, _dev(x, torch.float64 if self.mode == WEST_GAMMA else torch.complex128), _dev(out, torch.complex128)))
        return out

    def fft3d_static(self, dir, x, out):
        """west_fft3d_static: the sphere-truncated FFT with its scratch in the library's fixed static device array (no allocation of any
        kind in the call; `out` must be supplied by the caller).  Calls that overlap on the GPU race on that array."""
        import torch
        n_batch = int(x.shape[0])
        grid_dt = torch.float64 if self.mode == WEST_GAMMA else torch.complex128
        if dir == 1:
            assert x.shape[1] == self.n_g and tuple(out.shape) == (n_batch, self.N, self.N, self.N)
            self._ck(self.lib.west_fft3d_static(self.ctx, 1, n_batch, _dev(x, torch.complex128), _dev(out, grid_dt)))
        else:
            assert tuple(x.shape[1:]) == (self.N, self.N, self.N) and tuple(out.shape) == (n_batch, self.n_g)
            self._ck(self.lib.west_fft3d_static(self.ctx, -1, n_batch, _dev(x, grid_dt), _dev(out, torch.complex128)))
        return out

    def fft3d_dense(self, x, sign, out=None):
        """Dense C2C FFT of x [n_batch][n][n][n] (complex128 -> WEST_FP64, complex64 -> WEST_FP32); out=x runs in place."""
        import torch
        assert x.dim() == 4 and x.shape[1] == x.shape[2] == x.shape[3] and x.dtype in (torch.complex128, torch.complex64)
        if out is None:
            out = torch.empty_like(x)
        prec = WEST_FP64 if x.dtype == torch.complex128 else WEST_FP32
        self._ck(self.lib.west_fft3d_dense(self.ctx, int(x.shape[1]), int(sign), prec, int(x.shape[0]), _dev(x, x.dtype), _dev(out, x.dtype)))
        return out

    def h_apply(self, x, out=None, precision=WEST_FP64):
        import torch
        assert x.shape[1] == self.n_g
        if out is None:
            out = torch.empty_like(x)
        self._ck(self.lib.west_h_apply(self.ctx, precision, int(x.shape[0]), _dev(x, torch.complex128), _dev(out, torch.complex128)))
        return out

    def workspace_bytes(self, op, n_pert, n_freq=1, precision=WEST_FP64):
        return int(self.lib.west_workspace_bytes(self.ctx, int(op), int(n_pert), int(n_freq), int(precision)))

    def set_workspace(self, ws):
        """ws: a CUDA uint8 tensor the caller owns (hot calls then never allocate), or None for the context-owned lazy block."""
        import torch
        if ws is None:
            self._ck(self.lib.west_set_workspace(self.ctx, None, 0))
        else:
            self._ck(self.lib.west_set_workspace(self.ctx, _dev(ws, torch.uint8), int(ws.numel())))
        self._ws = ws

    def chi0_apply(self, dV, omegas, tol=1e-12, max_iter=500, alpha_pv=0.0, precond=1, check_every=4, precision=WEST_FP64, solver=0,
                   dn=None, want_dpsi=False, n_occ=None, want_stats=True, occupation=2.0, accumulate=False):
        """alpha_pv <= 0 selects the library's per-orbital default (west.h).  occupation / accumulate: the sum over spin channels
        of Eq. 11 (one context per channel, occupation=1, the second call with accumulate=True and the first call's dn); see
        chi0_apply_spin."""
        import torch
        N = self.N
        n_pert = int(dV.shape[0])
        assert tuple(dV.shape[1:]) == (N, N, N)
        om = np.ascontiguousarray(omegas, dtype=np.float64)
        n_freq = len(om)
        if dn is None:
            dn = torch.empty((n_freq, n_pert, N, N, N), dtype=torch.float64, device=dV.device)
        assert tuple(dn.shape) == (n_freq, n_pert, N, N, N), "dn must be [n_freq][n_pert][N][N][N]"
        dpsi = None
        if want_dpsi:
            # the library writes with the orbital count given to set_states: size the block from that
            assert self.n_occ is not None and (n_occ is None or int(n_occ) == self.n_occ), "n_occ differs from set_states"
            n_occ = self.n_occ
            shape = (n_freq, n_pert, n_occ, 2, self.n_g) if self.mode == WEST_GAMMA else (n_freq, n_pert, n_occ, self.n_g)
            dpsi = torch.empty(shape, dtype=torch.complex128, device=dV.device)
        opts = west_cg_opts(int(max_iter), float(tol), float(alpha_pv), int(precond), int(check_every), int(solver), float(occupation), int(bool(accumulate)))
        st = west_stats()
        rc = self._ck(self.lib.west_chi0_apply(self.ctx, precision, n_pert, _dev(dV, torch.float64), n_freq, om.ctypes.data, C.byref(opts),
                                               _dev(dn, torch.float64), _dev(dpsi) if dpsi is not None else None,
                                               C.byref(st) if want_stats else None))
        stats = {k: getattr(st, k) for k, _ in west_stats._fields_}
        stats["rc"] = rc
        return dn, dpsi, stats

    @staticmethod
    def chi0_apply_spin(channels, dV, omegas, **kw):
        """N_spin = 2: channels = [West_up, West_down], each holding its own V_loc^sigma, projectors and
        occupied orbitals.  dn = sum over channels, each with one electron per orbital.  alpha_pv may be a pair (one per channel).
        Returns dn and the list of per-channel stats."""
        alpha = kw.pop("alpha_pv", 0.0)
        alphas = list(alpha) if isinstance(alpha, (list, tuple)) else [alpha] * len(channels)
        dn, stats = None, []
        for k, w in enumerate(channels):
            dn, _, st = w.chi0_apply(dV, omegas, dn=dn, occupation=1.0, accumulate=k > 0, alpha_pv=alphas[k], **kw)
            stats.append(st)
        return dn, stats

    def lanczos(self, phi, n_steps, n_occ, want_brakets=False, precision=WEST_FP64):
        """alpha, beta [n_pert][n_occ][n_steps], norm [n_pert][n_occ], brakets [n_occ][n_steps][n_pert][n_pert] or None."""
        import torch
        n_pert = int(phi.shape[0])
        dev = phi.device
        alpha = torch.empty((n_pert, n_occ, n_steps), dtype=torch.float64, device=dev)
        beta = torch.empty_like(alpha)
        norm = torch.empty((n_pert, n_occ), dtype=torch.float64, device=dev)
        br = torch.empty((n_occ, n_steps, n_pert, n_pert), dtype=torch.float64, device=dev) if want_brakets else None
        self._ck(self.lib.west_lanczos(self.ctx, precision, n_pert, _dev(phi, torch.float64), int(n_steps), _dev(alpha), _dev(beta),
                                       _dev(norm), _dev(br) if br is not None else None))
        return alpha, beta, norm, br

    def lanczos_diag(self, alpha, beta, want_sweeps=False):
        """d [..., n_steps] ascending and U [..., n_steps, n_steps] (columns = eigenvectors, U[..., 0, :] >= 0) of the tridiagonal
        matrices of Eq. 19; alpha, beta [..., n_steps] as returned by lanczos()."""
        import torch
        n = int(alpha.shape[-1])
        n_chain = int(alpha.numel() // n) if n else 0
        d = torch.empty_like(alpha)
        U = torch.empty(tuple(alpha.shape) + (n,), dtype=torch.float64, device=alpha.device)
        sw = torch.empty(tuple(alpha.shape[:-1]), dtype=torch.int32, device=alpha.device) if want_sweeps else None
        self._ck(self.lib.west_lanczos_diag(self.ctx, n_chain, n, _dev(alpha, torch.float64), _dev(beta, torch.float64), _dev(d), _dev(U),
                                            _dev(sw) if sw is not None else None))
        return (d, U, sw) if want_sweeps else (d, U)

    def gemm_tn(self, A, B, out=None):
        """C[m][n] = sum_k A[m][k] B[n][k], f64 row-major."""
        import torch
        m, k = A.shape
        n = B.shape[0]
        if out is None:
            out = torch.empty((m, n), dtype=torch.float64, device=A.device)
        self._ck(self.lib.west_gemm_tn(self.ctx, m, n, k, _dev(A, torch.float64), A.stride(0), _dev(B, torch.float64), B.stride(0),
                                       _dev(out, torch.float64), out.stride(0)))
        return out

    def gemm_update(self, Cm, A, Y):
        """Y[n][k] += sum_m C[m][n] A[m][k]."""
        import torch
        m, k = A.shape
        n = Y.shape[0]
        self._ck(self.lib.west_gemm_update(self.ctx, m, n, k, _dev(Cm, torch.float64), Cm.stride(0), _dev(A, torch.float64), A.stride(0),
                                           _dev(Y, torch.float64), Y.stride(0)))
        return Y

    def device_bytes(self):
        return int(self.lib.west_device_bytes(self.ctx))

    def launch_count(self):
        return int(self.lib.west_launch_count(self.ctx))

    def set_cg_kernel(self, which):
        self._ck(self.lib.west_set_cg_kernel(self.ctx, int(which)))

    def set_ms_history(self, slots):
        self._ck(self.lib.west_set_ms_history(self.ctx, int(slots)))

    def probe_fp64_pipes(self, mode, n_dmma_warps, iters=20000):
        """(ms, DMMA flop, DFMA flop) of one launch of the FP64 pipe yardstick (west.h)"""
        ms, fd, ff = C.c_float(), C.c_double(), C.c_double()
        self._ck(self.lib.west_probe_fp64_pipes(self.ctx, int(mode), int(n_dmma_warps), int(iters), C.byref(ms), C.byref(fd), C.byref(ff)))
        return ms.value, fd.value, ff.value

    def set_fft_chunk(self, n):
        self._ck(self.lib.west_set_fft_chunk(self.ctx, int(n)))

    PROFILE_CLASSES = ("k1_g2r_z", "k2_planes", "k3_r2g_z", "gemm_tn", "gemm_update", "cg_vec", "fft_rhs_dn", "misc")

    def set_profile(self, on):
        self._ck(self.lib.west_set_profile(self.ctx, 1 if on else 0))

    def get_profile(self):
        ms = np.zeros(8, dtype=np.float64)
        cnt = np.zeros(8, dtype=np.int64)
        self._ck(self.lib.west_get_profile(self.ctx, ms.ctypes.data, cnt.ctypes.data))
        return {k: {"ms": float(ms[i]), "spans": int(cnt[i])} for i, k in enumerate(self.PROFILE_CLASSES)}
