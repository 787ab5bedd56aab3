#!/usr/bin/env python
"""bench.py - throughput of the chi0*dV hot path (Eq. 10-11 of arXiv 2203.05623) on B200, one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg5] [--impl reference]

A step = one west_chi0_apply over the workload's perturbation block: RHS (a1), batched PCG to the stated tolerance with
the dual-space H*psi, KB / P_v GEMMs and fused vector updates (a2-a9), and the dn accumulation (a10).
metric  = chi0*dV perturbations/s (perturbation x frequency solves per second, whole job, all ranks); the line also carries
          H*psi applications/s.
Default workload = cfg5, the largest single-GPU configuration of BASELINE.json (144^3 grid, 72 703 Gamma plane waves, 1024 states,
batches of 16 perturbations), at omega = 0.  The same line carries "workloads": sub-records for cfg2, cfg3, cfg4 and for cfg5's four
imaginary frequencies (a few steps each, own ms_per_step / roofline / clocks); --no-sub skips them.
The headline is timed WITHOUT the per-kernel profiler; kernel_ms_per_step comes from one extra, untimed step.
N > 1   = weak scaling: every rank holds the full orbitals and its own block of perturbations, no collective on the
          data path ("images"); value = all ranks' perturbations / max-over-ranks time.
--impl reference = the CPU oracle (oracle/) timed on a bounded sample of the same workload, on the host cores, on its own inputs.
--op happly | gemm | lanczos | pdep | fft | spin = single-operation benches (metric 1 of BASELINE.json, yardsticks, widening rows).
Inputs are seeded and synthetic (synth/); the occupied orbitals come from the library's own GPU eigensolver (set-up,
untimed).  Nothing here reads /root/reference.
"""
import argparse
import csv
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

TOL = 1e-8          # CG stopping tolerance of the throughput runs (reading R5)
MAX_ITER = 300
SUB_STEPS, SUB_WARMUP = 3, 1     # timed / warm-up steps of every sub-record (the kernels are warm from the headline by then)
T_START = time.time()
SUB_DEADLINE_S = 1400.0          # a sub-record is skipped (and says so) if the run has already taken this long: the line must still be printed


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg5")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-sub", action="store_true", help="skip the cfg2 / cfg3 / cfg4 / cfg5-imaginary-frequency sub-records")
    ap.add_argument("--omegas", default="default", help="default: omega = 0 for cfg1/2/4/5, the 8 frequencies for cfg3; 'all': every frequency the "
                                                        "config lists (cfg5: 0 and its 4 imaginary ones); 'iw': only the imaginary ones; or a comma list in Ry")
    ap.add_argument("--chunk", type=int, default=0, help="FFT slots per chunk (0 = library default)")
    ap.add_argument("--check-every", type=int, default=1, help="CG convergence poll / compaction period")
    ap.add_argument("--precond", type=int, default=1, help="0 none, 1 R4 default, 2 Teter-Payne-Allan")
    ap.add_argument("--solver", type=int, default=-1, help="0 per-frequency PCG/COCG, 1 multi-shift CG, 2 block CG; -1 = 1 when more than one frequency, else 0")
    ap.add_argument("--op", default="chi0", choices=["chi0", "happly", "gemm", "lanczos", "pdep", "fft", "spin", "pipes"],
                    help="chi0 = the hot path (default); happly = west_h_apply alone (H*psi/s, kernel classes); gemm = the projector GEMM shapes "
                         "against cuBLAS; lanczos = Eq. 15-19 chains; pdep = Davidson shell for chi0bar; fft = the dense C2C FFT of Fig. 3 "
                         "(--workload fft128 | fft256, --precision); spin = N_spin = 2 chi0 (widening rows)")
    ap.add_argument("--precision", default="fp64", choices=["fp64", "fp32", "mixed", "i8"], help="--op fft: fp64 | fp32; --op happly / gemm: fp64 | mixed | i8 (FP64 from int8 slices, WEST_FP64_I8); --op chi0: i8 overrides the workload's precision")
    ap.add_argument("--n-vec", type=int, default=0, help="--op happly / gemm: number of vectors (0 = the workload's CG-loop width)")
    ap.add_argument("--deflate", type=int, default=0, help="number of conduction eigenstates handed to west_set_deflation (0 = off)")
    ap.add_argument("--n-pert", type=int, default=0, help="override the perturbation count (0 = the config's)")
    ap.add_argument("--alpha-factor", type=float, default=0.0, help="alpha_pv = factor x (eps_Nv - eps_1), reading R3 (the result does not depend on it; "
                                                                         "must exceed 1); 0 = the library's per-orbital default alpha_v = (eps_v - eps_1) + W/2")
    ap.add_argument("--cg-kernel", type=int, default=0, help="west_set_cg_kernel: 0 automatic (column-resident where it fits), 1 streaming, 2 column split over a 2-CTA cluster")
    ap.add_argument("--ms-history", type=int, default=0, help="west_set_ms_history: 0 automatic Krylov-history ring of the multi-shift solver, -1 per-shift recurrences, 2..128 fixed ring size")
    ap.add_argument("--workspace", type=int, default=1, help="1: the bench allocates west_workspace_bytes and hands it over (no allocation in the timed calls); 0: lazy context-owned block")
    return ap.parse_args()


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def sm_clock_mhz():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return float(json.load(open(p)).get("sm_max_mhz", 1965.0))
    return 1965.0


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index = index
        self.stop_flag = threading.Event()
        self.rows = []

    def run(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        while not self.stop_flag.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + q, "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([x.strip() for x in out.split(",")])
            except Exception:
                pass
            self.stop_flag.wait(0.2)

    def finish(self):
        self.stop_flag.set()
        self.join()
        return self.summary()

    def summary(self):
        sm = [float(r[0]) for r in self.rows if r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) > 2 + i and r[2 + i].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons,
                "samples": len(self.rows)}


def omegas_for(a, cfg, workload):
    if a.omegas == "default":
        return list(cfg["omegas"]) if workload == "cfg3" else [0.0]
    if a.omegas == "all":
        return list(cfg["omegas"])
    if a.omegas == "iw":
        return [x for x in cfg["omegas"] if x > 0]
    return [float(x) for x in a.omegas.split(",")]


def build_inputs(cfg):
    """Seeded synthetic cell (synth/): potentials, projectors on the library's own sphere, perturbations."""
    import synth
    atoms = synth.atoms_for(cfg)
    vloc = synth.vloc_for(cfg, atoms)
    return atoms, vloc


def setup_gpu(cfg, n_pert, chunk, verbose, n_defl=0, vloc_add=None, alpha_factor=0.0):
    import torch
    import synth
    import paper_2203_05623_b200 as wb
    from paper_2203_05623_b200 import eigs
    mode = wb.WEST_GAMMA if cfg["mode"] == "gamma" else wb.WEST_FULL
    w = wb.West(cfg["L"], cfg["n2max"], cfg["N"], mode)
    if chunk:
        w.set_fft_chunk(chunk)
    miller, _, _, g2 = w.gsphere()
    atoms, vloc = build_inputs(cfg)
    if vloc_add is not None:
        vloc = vloc + vloc_add
    beta, dcoef = synth.kb_projectors(miller, cfg["L"], atoms, 0.8, cfg["projectors"])
    if mode == wb.WEST_GAMMA:
        # synth normalises over the rows it is given (the half sphere); rescale to sum over the FULL sphere = 1
        nrm = np.sqrt(2.0 * np.sum(np.abs(beta) ** 2, axis=1) - np.abs(beta[:, 0]) ** 2)
        beta = beta / nrm[:, None]
    dev = torch.device("cuda")
    w.set_vloc(torch.from_numpy(vloc).to(dev))
    w.set_kb(torch.from_numpy(np.ascontiguousarray(beta)).to(dev), dcoef)
    t0 = time.time()
    n_occ = cfg["n_occ"]
    eps, psi, res = eigs.lowest_states(w, n_occ + n_defl, tol=1e-10, verbose=False)
    gap = float(eps[n_occ] - eps[n_occ - 1])
    if n_defl:
        w.set_deflation(psi[n_occ:n_occ + n_defl].contiguous(), eps[n_occ:n_occ + n_defl])
        psi = psi[:n_occ].contiguous()
    if verbose:
        print("# %s eigensolver: %.1f s, residual %.2e, gap %.4f Ry" % (cfg["name"], time.time() - t0, res, gap), file=sys.stderr)
    w.set_states(psi, eps[:cfg["n_occ"]])
    width = float(eps[cfg["n_occ"] - 1] - eps[0])
    alpha = max(alpha_factor * width, 0.01) if alpha_factor > 0 else 0.0        # 0: per-orbital default inside the library
    dV = synth.perturbations(cfg, n_pert=n_pert)
    return w, dV, alpha, dict(eps=eps, psi=psi, gap=gap, res=res, miller=miller, vloc=vloc, beta=beta, dcoef=dcoef, width=width)


def alpha_of(alpha, aux, v):
    """the alpha_v the library used for orbital v (west.h: alpha_pv <= 0 selects (eps_v - eps_min) + W/2)"""
    return alpha if alpha > 0 else max(float(aux["eps"][v] - aux["eps"][0]) + 0.5 * aux["width"], 0.01)


# ------------------------------------------------------------------------------------------------ oracle side (CPU legs, parity sample)
class OracleSide:
    """The oracle's view of a bench cell: its own sphere, its own matrix-free H; the orbitals are the bench's inputs (re-checked
    here as eigenvectors of the ORACLE's H before anything is compared or timed)."""

    def __init__(self, cfg, aux):
        from oracle import gsphere as ogs
        from oracle import hamiltonian as oham
        self.cfg, self.aux = cfg, aux
        L, N = cfg["L"], cfg["N"]
        self.m = ogs.enumerate_sphere(cfg["n2max"])
        self.idx = ogs.fft_index(self.m, N)
        self.g2 = ogs.g2_of(self.m, L)
        self.minus = ogs.index_of_minus(self.m)
        self.gamma = cfg["mode"] == "gamma"
        self.ogs = ogs
        psi = aux["psi"].cpu().numpy()
        self.U = (ogs.expand_half_to_full(psi, self.m) if self.gamma else psi).T.copy()          # [n_g_full, n_occ]
        beta = ogs.expand_half_to_full(aux["beta"], self.m) if self.gamma else aux["beta"]
        self.eps = aux["eps"]
        self.apply_H = lambda y: oham.apply_h(y, self.m, L, N, aux["vloc"], beta, aux["dcoef"])
        r = self.apply_H(self.U[:, 0]) - self.eps[0] * self.U[:, 0]
        assert np.linalg.norm(r) < 1e-6, "orbitals are not eigenvectors of the oracle's H"

    def full(self, c_half):
        return self.ogs.expand_half_to_full(c_half, self.m) if self.gamma else c_half

    def rhs(self, dV_i, v):
        from oracle import chi0 as ochi0
        b = ochi0.rhs_vectors(self.U[:, v:v + 1], dV_i[None], self.idx, self.cfg["N"])[0, 0]
        return b

    def true_residual(self, dV_i, v, x, omega, alpha_v):
        """|| (H - eps_v - i omega + alpha P_v) x + P_c dV_i psi_v || / || rhs ||  (Eq. 10, with SURVEY Appendix A's shift)"""
        U = self.U
        b = self.rhs(dV_i, v)
        rhs = -(b - U @ (U.conj().T @ b))
        A = self.apply_H(x) - (self.eps[v] + 1j * omega) * x + alpha_v * (U @ (U.conj().T @ x))
        return float(np.linalg.norm(A - rhs) / np.linalg.norm(rhs))


def cpu_h_apply_leg(cfg, osd, n_vec):
    """SURVEY 8(d) CPU leg (i): the oracle's matrix-free H*psi (numpy.fft + dense projector products) over n_vec random vectors."""
    rng = np.random.Generator(np.random.PCG64(99))
    n = len(osd.m)
    x = rng.standard_normal((n_vec, n)) + 1j * rng.standard_normal((n_vec, n))
    t0 = time.time()
    osd.apply_H(x)
    dt = time.time() - t0
    return {"h_apply_per_s": n_vec / dt, "n_vec": n_vec, "seconds": dt, "what": "oracle.hamiltonian.apply_h on %d random full-sphere vectors (%d coefficients)" % (n_vec, n)}


def cpu_sum_over_states_leg():
    """SURVEY 8(d) CPU leg (ii): the plain definition - dense H, LAPACK eigh, sum over states - on the two cells where it is feasible
    within the bench's time (cfg 1 and the one-cell Si-like mini2), perturbations/s with and without the one-off eigh."""
    import synth
    from oracle import chi0 as ochi0
    from oracle import gsphere as ogs
    from oracle import hamiltonian as oham
    out = {}
    for name in ("cfg1", "mini2"):
        cfg = synth.get_config(name)
        m = ogs.enumerate_sphere(cfg["n2max"])
        atoms = synth.atoms_for(cfg)
        vloc = synth.vloc_for(cfg, atoms)
        beta, dcoef = synth.kb_projectors(m, cfg["L"], atoms, 0.8, cfg["projectors"])
        dV = synth.perturbations(cfg)
        t0 = time.time()
        H = oham.dense_h(m, cfg["L"], cfg["N"], vloc, beta, dcoef)
        eps, U = oham.eigensystem(H, m, real_orbitals=cfg["mode"] == "gamma")
        t_eig = time.time() - t0
        t0 = time.time()
        ochi0.chi0_sum_over_states(eps, U, cfg["n_occ"], dV, [0.0], m, cfg["L"], cfg["N"])
        t_sos = time.time() - t0
        out[name] = {"n_g_full": int(len(m)), "n_occ": cfg["n_occ"], "n_pert": int(len(dV)), "eigh_s": t_eig, "sum_over_states_s": t_sos,
                     "perturbations_per_s_without_eigh": len(dV) / t_sos, "perturbations_per_s_with_eigh": len(dV) / (t_sos + t_eig)}
    return out


def cpu_pcg_leg(cfg, osd, dV0, alpha, aux, budget_s, iters_hint=None):
    """SURVEY 8(d) CPU leg (iii) and the cpu_baseline value: the oracle's own PCG route (oracle/iterative.py) on a bounded sample of
    (perturbation 0, state v) columns of THIS workload.  Returns the record and the solved columns {v: x} (for the parity sample)."""
    from oracle import iterative as oit
    cores = len(os.sched_getaffinity(0))
    n_occ = cfg["n_occ"]
    t0 = time.time()
    sols, iters = {}, 0
    # where one column alone exceeds the budget (cfg 5: ~3 s per H*psi on the host) the iteration cap bounds the sample instead
    probe_t = time.time()
    osd.apply_H(osd.U[:, 0])
    t_h = time.time() - probe_t
    cap = MAX_ITER if t_h * 30 < budget_s else max(2, int(budget_s / (1.3 * t_h)))
    for v in range(n_occ):
        b = osd.rhs(dV0, v)
        x, it, rel = oit.pcg_sternheimer(osd.apply_H, osd.U, osd.eps[v], v, b, osd.g2, alpha_of(alpha, aux, v), tol=TOL, max_iter=cap)
        iters += it
        if rel <= TOL:
            sols[v] = x
        if time.time() - t0 > budget_s or cap < MAX_ITER:
            break
    dt = time.time() - t0
    n_done = max(len(sols), 1)
    if sols:
        value = len(sols) / n_occ / dt
        sample = "oracle.iterative.pcg_sternheimer on %d of %d (i=0, v) columns of %s, tol %.0e, %d H*psi, %.1f s" % (len(sols), n_occ, cfg["name"], TOL, iters, dt)
    else:
        # truncated solve: seconds per PCG iteration x the iteration count of a converged column (the GPU run's mean, same algorithm)
        per_it = dt / max(iters, 1)
        n_it = iters_hint or 30
        value = 1.0 / (n_occ * per_it * n_it)
        sample = ("oracle.iterative.pcg_sternheimer, %d iterations of column (0, 0) of %s in %.1f s (one column does not fit the time budget); "
                  "value = 1 / (n_occ x s-per-iteration x %.1f iterations per column, the mean count of the GPU run)" % (iters, cfg["name"], dt, n_it))
    rec = {"value": value, "unit": "perturbations/s", "cores": cores, "kind": "oracle", "sample": sample, "h_apply_per_s": iters / dt}
    return rec, sols


# ------------------------------------------------------------------------------------------------ roofline
def aux_ncols(cfg):
    m = cfg["n_max"]
    return sum(1 for x in range(-m, m + 1) for y in range(-m, m + 1) if x * x + y * y <= cfg["n2max"])


def ncu_traffic_table():
    """profiles/ncu_dram_traffic.csv: dram__bytes_read.sum + dram__bytes_write.sum of one launch per kernel class, captured with
    `ncu --set full` at the launch sizes this bench uses (commands and dates in profiles/ncu_dram_traffic.md)."""
    p = os.path.join(ROOT, "profiles", "ncu_dram_traffic.csv")
    rows = {}
    if os.path.exists(p):
        for r in csv.DictReader(open(p)):
            try:
                rows[(r["kernel"], int(r["N"]), r["precision"])] = (float(r["dram_bytes"]) / float(r["units"]), r["unit_name"], r["capture"])
            except (KeyError, ValueError):
                pass
    return rows


_FP64_PEAK = {}


def measure_fp64_peak():
    """The box's own FP64 yardstick: cuBLAS DGEMM 8192^3 through torch, best of 5, TFLOP/s (measured once per run)."""
    if "v" in _FP64_PEAK:
        return _FP64_PEAK["v"]
    import torch
    n = 8192
    a = torch.randn((n, n), dtype=torch.float64, device="cuda")
    b = torch.randn((n, n), dtype=torch.float64, device="cuda")
    best = 1e9
    for _ in range(6):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        torch.matmul(a, b)
        e1.record()
        torch.cuda.synchronize()
        best = min(best, e0.elapsed_time(e1))
    del a, b
    torch.cuda.empty_cache()
    _FP64_PEAK["v"] = 2.0 * n ** 3 / (best * 1e-3) / 1e12
    return _FP64_PEAK["v"]


def roofline(cfg, top, prof, n_h, n_freq, solver, hbm_peak, peak_src, mixed, n_g, fp64_peak, shift_updates=0, hist_passes=0, i8=False):
    """Roofline entry for the kernel class that took the most time in the profiled step (DESIGN.md section 6 states the per-unit
    figures).  n_h = vectors pushed through H in that step."""
    N = cfg["N"]
    gamma = cfg["mode"] == "gamma"
    n_cols = aux_ncols(cfg)
    slots = n_h / (2 if gamma else 1)                       # FFT slots pushed through H*psi in the profiled step
    csz = 8 if mixed else 16
    t = prof[top]["ms"] * 1e-3
    spans = max(1, prof[top]["spans"])
    fp64_src = "measured in this run: cuBLAS DGEMM 8192^3 FP64 (DMMA and the FP64 FMA pipe have the same nominal rate on B200, 37.2 TFLOP/s)"
    out = {"kernel": top, "avg_launch_ms": prof[top]["ms"] / spans, "launches": spans, "traffic": None}
    table = ncu_traffic_table()
    tkey = ((("cg_vec_msh" if hist_passes > 0 else "cg_vec_ms") if (top == "cg_vec" and solver == 1) else top), N, "mixed" if mixed else ("i8" if (i8 and top.startswith("gemm")) else "fp64"))
    rows = cfg["n_proj"] + cfg["n_occ"]
    if not gamma:
        rows *= 2
    if top in ("k1_g2r_z", "k2_planes", "k3_r2g_z"):
        stick = N * n_cols * csz
        sphere = (2 if gamma else 1) * n_g * 16
        per_slot = {"k1_g2r_z": sphere + stick, "k2_planes": 2 * stick, "k3_r2g_z": stick + 2 * sphere}[top]
        gbs = per_slot * slots / t / 1e9
        units = slots
        if top == "k2_planes":
            # the plane kernel is bound on the SM (FP64 issue / shared memory), not by HBM: nominal 5 N log2 N flops
            # per 1D transform, 2 (nr + N) transforms per plane, plus the V_loc multiply
            nr = 2 * cfg["n_max"] + 1
            fl_slot = N * (2 * (nr + N) * 5.0 * N * np.log2(N) + 2 * N * N)
            ach = fl_slot * slots / t / 1e12
            peak = fp64_peak * (2.0 if mixed else 1.0)
            out.update({"bound": "alu", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
                        "peak_source": fp64_src + ("; x2 for the FP32 path" if mixed else ""),
                        "algorithmic_flops_per_slot": fl_slot, "algorithmic_bytes_per_slot": per_slot,
                        "hbm_view": {"achieved_gbs": gbs, "peak_gbs": hbm_peak, "frac": gbs / hbm_peak, "peak_source": peak_src}})
            smem_slot = N * (8 * nr * N + 4 * N * N) * csz
            smem_peak = 128.0 * 148 * sm_clock_mhz() * 1e6 / 1e9
            smem_gbs = smem_slot * slots / t / 1e9
            out["smem_view"] = {"achieved_gbs": smem_gbs, "peak_gbs": smem_peak, "frac": smem_gbs / smem_peak,
                                "algorithmic_smem_bytes_per_slot": smem_slot,
                                "peak_source": "128 B/clk/SM x 148 SMs x max SM clock (MEASURED_PEAKS.json sm_max_mhz, else 1965 MHz)"}
        else:
            out.update({"bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak,
                        "peak_source": peak_src, "algorithmic_bytes_per_slot": per_slot})
    elif top in ("gemm_tn", "gemm_update"):
        # each of the two GEMMs of a low-rank apply does 2 rows (2 n_g) flops per vector; the class time covers one of them
        flops = 2.0 * rows * (2 * n_g) * n_h
        ach = flops / t / 1e12
        peak = fp64_peak
        out.update({"bound": "tensor", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak, "peak_source": fp64_src,
                    "algorithmic_flops_per_vector": 2.0 * rows * 2 * n_g,
                    "algorithmic_bytes_per_vector": (1 if top == "gemm_tn" else 2) * 2 * n_g * 8,
                    "note": "FP64 DMMA (mma.sync m8n8k4; tcgen05 has no FP64 kind)" if not mixed else "3xTF32 products, FP64 operands in memory; peak shown is the FP64 one"})
        if i8:
            # WEST_FP64_I8: the contraction runs as 21 or 36 int8 slice-pair products per FP64 product (6 or 8 slices, pairs with i + j < S) on the INT8
            # tensor path; its roofline is the int8 tensor peak = the measured dense bf16 rate x the nominal ratio 2 (B200_PROFILING.md)
            p = os.path.join(ROOT, "MEASURED_PEAKS.json")
            bf16 = float(json.load(open(p)).get("bf16_tflops_sustained", 1370.0)) if os.path.exists(p) else 1370.0
            n_prod = 21.0 if TOL >= 1e-9 else 36.0     # west.h: 6 slices (21 pair products) when the CG tolerance is 1e-9 or looser, else 8 (36)
            ops = n_prod * flops
            out.update({"bound": "tensor", "achieved": ops / t / 1e12, "peak": 2.0 * bf16, "unit": "TFLOP/s", "frac": ops / t / 1e12 / (2.0 * bf16),
                        "peak_source": "int8 tensor: 2 x the sustained dense bf16 rate of MEASURED_PEAKS.json (else 2 x 1370)", "fp64_equivalent_tflops": ach,
                        "int8_products_per_fp64_product": n_prod,
                        "note": "tcgen05.mma kind::i8: exact int8 slice-pair products (6 slices = 21 products at this tolerance), int32 accumulation in TMEM, FP64 sums; the class time "
                                "includes the per-call slicing of the vector / coefficient block; `achieved` counts int8 operations"})
        units = n_h
    else:
        # CG vector kernel.  PCG/COCG column-resident or streaming: 4 reads + 3 writes of a column per iteration (p, Ap, x, r | x, r, p).
        # multi-shift: r, p, Ap (3 reads + 2 writes) plus, per live shift, p_s (2 real vectors read + written) and Re x_s (1 read + written)
        if solver == 1:
            # 8 passes for the seed recurrence (p, Ap | r, Ap -> r | r, p -> p) and 6 per live shift (p_s: two real vectors read and written, Re x_s
            # read and written); the library counts the (column, shift) updates it performed (west_stats.n_shift_updates)
            if hist_passes > 0:
                # Krylov-history variant: 8 passes for the seed recurrence (p, Ap | r_k, Ap -> r_k+1 | r_k+1, p -> p) and the history contractions,
                # whose column-vector passes the library counts (west_stats.n_hist_passes); both run in this kernel class
                per_col = (8 + float(hist_passes) / max(n_h, 1)) * 16 * n_g
                note = "multi-shift with Krylov history: 8 + %.2f (history contractions, counted by the library) vector passes of 16 n_g bytes per column and iteration" % (hist_passes / max(n_h, 1))
            else:
                per_col = (8 + 6.0 * shift_updates / max(n_h, 1)) * 16 * n_g
                note = "multi-shift: 8 + 6 x (live shifts per column, measured: %.2f of %d) vector passes of 16 n_g bytes per column and iteration" % (shift_updates / max(n_h, 1), n_freq)
        else:
            per_col = 7 * 16 * n_g
            note = "7 vector passes of 16 n_g bytes per column and iteration"
        ach = per_col * n_h / t / 1e9
        out.update({"bound": "hbm", "achieved": ach, "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak, "peak_source": peak_src,
                    "algorithmic_bytes_per_column": per_col, "note": note})
        units = n_h
    if tkey in table:
        per_unit, unit_name, cap = table[tkey]
        out["traffic"] = per_unit * units / spans
        out["traffic_note"] = "ncu dram__bytes_read.sum + dram__bytes_write.sum per %s (%s) x %s per launch here" % (unit_name, cap, unit_name)
    return out


# ------------------------------------------------------------------------------------------------ the hot path
def chi0_op(wb, solver, omegas):
    B = wb.binding
    if solver == 1:
        return B.WEST_OP_CHI0_MULTISHIFT
    if solver == 2 and max(omegas) == 0:
        return B.WEST_OP_CHI0_BLOCK
    return B.WEST_OP_CHI0_IW if max(omegas) > 0 else B.WEST_OP_CHI0


def make_workspace(w, wb, op, n_pert, n_freq, precision, reserve_bytes):
    """The caller-owned workspace of the timed calls (west.h): west_workspace_bytes for the whole block if the device has room for it,
    else for the largest number of perturbations that fits (the library then walks the block in sub-blocks)."""
    import torch
    free = torch.cuda.mem_get_info()[0] - reserve_bytes
    fit = n_pert
    if op == wb.binding.WEST_OP_CHI0_MULTISHIFT:
        # multi-shift solver: the library turns every byte beyond the minimum into ring slots of its Krylov history (west_set_ms_history),
        # so hand it the full-history size if the device has it, else what is free
        full = w.workspace_bytes(wb.binding.WEST_OP_CHI0_MULTISHIFT_HIST, n_pert, n_freq, precision)
        need = min(full, free // 256 * 256)
        if need >= w.workspace_bytes(op, 1, n_freq, precision):
            ws = torch.empty(need, dtype=torch.uint8, device="cuda")
            w.set_workspace(ws)
            return ws, n_pert
    for nb in range(1, n_pert + 1):
        fit = (n_pert + nb - 1) // nb
        need = w.workspace_bytes(op, fit, n_freq, precision)
        if need <= free or fit == 1:
            break
    ws = torch.empty(need, dtype=torch.uint8, device="cuda")
    w.set_workspace(ws)
    return ws, fit


def run_chi0(a, wb, cfg, w, dV_np, alpha, aux, omegas, solver, precision, steps, warmup, local, world, barrier, e2e_steps, want_cpu, label, profile_in_timed=False):
    """Times `steps` calls of west_chi0_apply on the block dV_np (after `warmup` untimed ones) and returns the record of that workload.
    want_cpu: 0 nothing from the oracle, 1 parity_sample only, 2 parity_sample + cpu_baseline with its legs.
    profile_in_timed: take the per-kernel-class times from the timed steps themselves (one CUDA-event pair around every launch) instead of
    an extra step - only for the long sub-record, where a step takes a hundred seconds and the events cost nothing next to it."""
    import torch
    import torch.distributed as dist
    dev = torch.device("cuda")
    n_pert, N, n_freq = dV_np.shape[0], cfg["N"], len(omegas)
    dV = torch.from_numpy(dV_np).to(dev)
    dn = torch.empty((n_freq, n_pert, N, N, N), dtype=torch.float64, device=dev)
    mixed = precision == wb.WEST_MIXED
    kw = dict(solver=solver, tol=TOL, max_iter=MAX_ITER if solver != 1 else 2000, alpha_pv=alpha, precond=a.precond, check_every=a.check_every,
              precision=precision, dn=dn)
    ws = None
    if a.workspace:
        # room left for the parity sample's dpsi block (parity_and_cpu: the whole block if it is below 40 GB, else one perturbation)
        dpsi_bytes = 16 * w.n_g * n_pert * cfg["n_occ"] * (2 if cfg["mode"] == "gamma" else 1) * n_freq
        if dpsi_bytes >= (40 << 30):
            dpsi_bytes //= n_pert
        ws, fit = make_workspace(w, wb, chi0_op(wb, solver, omegas), n_pert, n_freq, precision, reserve_bytes=(4 << 30) + min(dpsi_bytes, 40 << 30))
    stats = None
    for _ in range(warmup):
        _, _, stats = w.chi0_apply(dV, omegas, **kw)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    launches0 = w.launch_count()
    if profile_in_timed:
        w.set_profile(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.cudart().cudaProfilerStart()        # no-op outside a profiler; `ncu --profile-from-start off` then lists the timed steps only
    e0.record()
    n_h = 0
    for _ in range(steps):
        _, _, stats = w.chi0_apply(dV, omegas, **kw)
        n_h += stats["n_h_apply"]
    e1.record()
    barrier()
    torch.cuda.cudart().cudaProfilerStop()
    ms = e0.elapsed_time(e1)
    launches = w.launch_count() - launches0
    clocks = sampler.finish()
    if profile_in_timed:
        prof = w.get_profile()
        w.set_profile(False)
        for v in prof.values():
            v["ms"] /= steps
            v["spans"] = max(v["spans"] // steps, 1) if v["spans"] else 0
        n_h_prof, pst = n_h / steps, stats
    else:
        # ---- per-kernel-class times: one extra, untimed step with the event profiler on
        w.set_profile(True)
        _, _, pst = w.chi0_apply(dV, omegas, **kw)
        prof = w.get_profile()
        w.set_profile(False)
        n_h_prof = pst["n_h_apply"]
    # ---- end to end: pinned host dV -> device, chi0_apply, dn -> pinned host, all inside the timed region
    e2e_ms = None
    if e2e_steps > 0:
        h_dV = torch.from_numpy(dV_np).pin_memory()
        h_dn = torch.empty(dn.shape, dtype=torch.float64).pin_memory()
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            dV.copy_(h_dV, non_blocking=True)
            w.chi0_apply(dV, omegas, **kw)
            h_dn.copy_(dn, non_blocking=True)
            torch.cuda.synchronize()
        e2e_ms = (time.perf_counter() - t0) * 1e3 / e2e_steps
        del h_dV, h_dn
    t = torch.tensor([ms, e2e_ms or 0.0], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms, e2e_ms = float(t[0]), (float(t[1]) if e2e_ms is not None else None)

    units = n_pert * n_freq * world
    hbm_peak, peak_src = peaks()
    fp64_peak = measure_fp64_peak()
    top = max(prof, key=lambda k: prof[k]["ms"])
    rows = (cfg["n_proj"] + cfg["n_occ"]) * (1 if cfg["mode"] == "gamma" else 2)
    t_gemm = (prof["gemm_tn"]["ms"] + prof["gemm_update"]["ms"]) * 1e-3
    gemm_tf = 2 * 2.0 * rows * (2 * w.n_g) * n_h_prof / t_gemm / 1e12 if t_gemm > 0 else None
    rec = {
        "value": units * steps / (ms * 1e-3), "unit": "perturbations/s", "steps": steps, "warmup": warmup, "ms_per_step": ms / steps,
        "dtype": ("f64" if precision != wb.WEST_FP64_I8 else "f64 (projector GEMMs inside H*psi: exact int8-slice products on tcgen05 kind::i8 - 6 slices of 7 bits per operand row at this tolerance - FP64 sums)") if not mixed else "f32 FFT + 3xTF32 GEMMs inside H*psi / f64 vectors, dots, dn",
        "config": {"workload": label, "N": N, "n_g": w.n_g, "n_occ": cfg["n_occ"], "n_pert_per_gpu": n_pert, "n_freq": n_freq, "omega_ry": [round(x, 6) for x in omegas],
                   "n_proj": cfg["n_proj"], "n_deflated": a.deflate, "alpha_pv": "per-orbital (eps_v - eps_1) + W/2" if alpha <= 0 else alpha, "tol": TOL,
                   "solver": {0: "PCG/COCG per frequency", 1: "multi-shift CG", 2: "block CG"}[solver], "ms_history_slots": stats.get("ms_history_slots", 0), "cg_iters": stats["iters"], "cg_iters_min": stats["iters_min"],
                   "unconverged": stats["n_unconverged"], "sub_blocks": stats["n_sub_blocks"], "gap_ry": aux["gap"],
                   "workspace": "caller-owned, %.1f GB (west_set_workspace): no allocation in the timed calls" % (ws.numel() / 1e9) if ws is not None else "context-owned (lazy)",
                   "l2": "inputs per step (vector sets, %.1f GB) exceed the 126 MB L2" % (4 * 16 * w.n_g * n_pert * cfg["n_occ"] / 1e9)},
        "h_apply_per_s": n_h * world / (ms * 1e-3), "h_apply_per_step": n_h / steps,
        "gpu_launches": int(launches), "clocks": clocks,
        "roofline": roofline(cfg, top, prof, n_h_prof, n_freq, solver, hbm_peak, peak_src, mixed, w.n_g, fp64_peak, pst.get("n_shift_updates", 0), pst.get("n_hist_passes", 0), precision == wb.WEST_FP64_I8),
        "gemm": {"achieved_tflops": gemm_tf, "peak_tflops": fp64_peak, "frac": (gemm_tf / fp64_peak) if gemm_tf else None,
                 "note": "KB + P_v GEMMs of the CG loop in the profiled step (RHS projection excluded from the flop count)" +
                         ("; FP64-EQUIVALENT rate of the int8-slice products against the FP64 peak (may exceed 1)" if precision == wb.WEST_FP64_I8 else "")},
        "kernel_ms_per_step": {k: round(v["ms"], 3) for k, v in prof.items() if v["spans"]},
        "kernel_ms_note": "CUDA events around every launch of the timed step(s)" if profile_in_timed else "one extra untimed step with CUDA events around every launch; the timed steps run without them",
        "phase_ms_last_step": {"rhs": stats["ms_rhs"], "cg": stats["ms_cg"], "dn": stats["ms_dn"]},
        "device_gb": (w.device_bytes() + (ws.numel() if ws is not None else 0)) / 1e9,
    }
    if e2e_ms is not None:
        rec["e2e"] = {"value": units / (e2e_ms * 1e-3), "unit": "perturbations/s", "steps": e2e_steps,
                      "h2d_bytes_per_step": int(dV.numel() * 8), "d2h_bytes_per_step": int(dn.numel() * 8)}
    if want_cpu:
        try:
            rec.update(parity_and_cpu(a, wb, cfg, w, dV, dV_np, alpha, aux, omegas, kw, n_h / steps, want_cpu))
        except Exception as e:          # the oracle legs never take the GPU numbers down with them
            rec["cpu_baseline_error"] = repr(e)[:300]
    w.set_workspace(None)
    del ws, dV, dn
    torch.cuda.empty_cache()
    return rec


def parity_and_cpu(a, wb, cfg, w, dV, dV_np, alpha, aux, omegas, kw, n_h_step, level):
    """parity_sample: the TIMED configuration (same options, same block) once more with dpsi requested, sampled columns against the
    oracle - its own PCG / COCG solutions where a column is affordable on the host, else the true residual with its H.
    cpu_baseline: the oracle's PCG on a bounded sample of the same workload, plus SURVEY 8(d)'s legs (i) and (ii)."""
    import torch
    from oracle import iterative as oit
    n_pert, n_occ, n_freq = dV_np.shape[0], cfg["n_occ"], len(omegas)
    gamma = cfg["mode"] == "gamma"
    dpsi_bytes = 16 * w.n_g * n_pert * n_occ * (2 if gamma else 1) * n_freq
    free = torch.cuda.mem_get_info()[0]
    npar = n_pert if dpsi_bytes < min(40 << 30, free - (2 << 30)) else 1
    kw = dict(kw)
    kw.pop("dn")
    _, dpsi, st = w.chi0_apply(dV[:npar].contiguous(), omegas, want_dpsi=True, **kw)
    osd = OracleSide(cfg, aux)
    big = cfg["N"] >= 144
    out = {}
    if kw["solver"] == 1:
        mean_iters = n_h_step / (n_pert * n_occ)                      # one Krylov sequence serves every frequency
    else:
        mean_iters = n_h_step / (n_pert * n_occ * sum(2 if om > 0 else 1 for om in omegas)) * 1.0
    sols = {}
    if level >= 2:
        base, sols = cpu_pcg_leg(cfg, osd, dV_np[0], alpha, aux, budget_s=12.0 if big else 15.0, iters_hint=mean_iters)
        base["h_apply_leg"] = cpu_h_apply_leg(cfg, osd, 4 if big else 64)
        base["sum_over_states_leg"] = cpu_sum_over_states_leg()
        out["cpu_baseline"] = base
    elif not big and omegas[0] == 0.0:
        _, sols = cpu_pcg_leg(cfg, osd, dV_np[0], alpha, aux, budget_s=3.0)

    def col(wi, i, v):
        if gamma:
            return osd.full(dpsi[wi, i, v, 0].cpu().numpy()) + 1j * osd.full(dpsi[wi, i, v, 1].cpu().numpy())
        return dpsi[wi, i, v].cpu().numpy()

    worst, n, kind = 0.0, 0, None
    if sols and omegas[0] == 0.0:
        kind = "dpsi of the timed configuration vs oracle.iterative.pcg_sternheimer (both to tol %.0e; relative max-norm)" % TOL
        for v, x in sols.items():
            got = col(0, 0, v)
            worst = max(worst, float(np.max(np.abs(got - x)) / np.max(np.abs(x))))
            n += 1
    resid, nres = 0.0, 0
    samples = [(0, 0, 0), (n_freq - 1, npar - 1, n_occ - 1)]
    for wi, i, v in samples[:2 if not big else 2]:
        resid = max(resid, osd.true_residual(dV_np[i], v, col(wi, i, v), omegas[wi], alpha_of(alpha, aux, v)))
        nres += 1
    if not big and max(omegas) > 0:
        wi = n_freq - 1
        x, it, rel = oit.cocg_sternheimer(osd.apply_H, osd.U, osd.eps[3], 3, osd.rhs(dV_np[0], 3), osd.g2, osd.minus, alpha_of(alpha, aux, 3), omegas[wi], tol=TOL, max_iter=MAX_ITER)
        got = col(wi, 0, 3)
        worst = max(worst, float(np.max(np.abs(got - x)) / np.max(np.abs(x))))
        n += 1
        kind = (kind + "; " if kind else "") + "one column at omega = %.3g Ry vs oracle.iterative.cocg_sternheimer" % omegas[wi]
    out["parity_sample"] = {"relmax": worst if n else None, "n_columns": n, "kind": kind,
                            "true_residual_max": resid, "n_residual_columns": nres,
                            "residual_kind": "|| (H - eps_v - i omega + alpha_v P_v) dpsi + P_c dV psi_v || / || rhs || with the oracle's matrix-free H, columns (first, first) and (last, last)",
                            "block": "%d of %d perturbations, all %d frequencies, options of the timed calls" % (npar, n_pert, n_freq), "unconverged": st["n_unconverged"]}
    del dpsi
    torch.cuda.empty_cache()
    return out


def main():
    a = parse()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    import synth
    if a.op == "fft":
        return bench_fft(a, rank, world, local)
    cfg = synth.get_config(a.workload)
    n_pert = a.n_pert or cfg.get("pert_batch", cfg["n_pert"])
    omegas = omegas_for(a, cfg, a.workload)

    if a.impl == "reference":
        if rank != 0:
            return
        run_reference(a, cfg, n_pert, omegas)
        return

    import torch
    import torch.distributed as dist
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    import paper_2203_05623_b200 as wb
    precision = wb.WEST_MIXED if cfg["precision"] == "mixed" else wb.WEST_FP64
    if a.precision == "i8" and precision == wb.WEST_FP64:
        precision = wb.WEST_FP64_I8

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if a.op == "pipes":
        # yardstick: DMMA and DFMA warps alone and together (west_probe_fp64_pipes)
        c1 = synth.get_config("cfg1")
        wp = wb.West(c1["L"], c1["n2max"], c1["N"], wb.WEST_FULL)
        rows = []
        for nd in (0, 4, 8, 12, 16):
            for mode in (1, 2, 3):
                if (nd == 0 and mode & 1) or (nd == 16 and mode & 2):
                    continue
                ms, fd, ff = wp.probe_fp64_pipes(mode, nd)
                rows.append({"dmma_warps": nd, "dfma_warps": 16 - nd, "mode": {1: "DMMA only", 2: "DFMA only", 3: "both"}[mode], "ms": round(ms, 3),
                             "dmma_tflops": round(fd / ms / 1e9, 2), "dfma_tflops": round(ff / ms / 1e9, 2), "sum_tflops": round((fd + ff) / ms / 1e9, 2)})
        wp.close()
        if rank == 0:
            print(json.dumps({"metric": "FP64 pipe yardstick: DMMA / DFMA warps alone and together", "unit": "TFLOP/s", "n_gpus": 1, "rows": rows}))
        return
    if a.op in ("happly", "gemm"):
        return bench_kernels(a, wb, cfg, rank, world, barrier)
    # every rank: same cell and orbitals, its own block of perturbations (seeded stream offset by rank)
    w, dV_np, alpha, aux = setup_gpu(cfg, n_pert, a.chunk, verbose=(rank == 0), n_defl=a.deflate, alpha_factor=a.alpha_factor)
    w.set_cg_kernel(a.cg_kernel)
    w.set_ms_history(a.ms_history)
    if world > 1:
        dV_np = synth.perturbations(cfg, n_pert=n_pert, first=rank * n_pert)
    dev = torch.device("cuda")
    if a.op == "lanczos":
        return bench_lanczos(a, cfg, w, torch.from_numpy(dV_np).to(dev), n_pert, rank, world, barrier)
    if a.op == "pdep":
        return bench_pdep(a, cfg, w, alpha, n_pert, rank, world, barrier)
    if a.op == "spin":
        w.close()
        N = cfg["N"]
        dn = torch.empty((1, n_pert, N, N, N), dtype=torch.float64, device=dev)
        kw = dict(solver=0, tol=TOL, max_iter=MAX_ITER, alpha_pv=alpha, precond=a.precond, check_every=a.check_every, precision=precision, dn=dn)
        return bench_spin(a, cfg, torch.from_numpy(dV_np).to(dev), n_pert, rank, world, barrier, kw)

    solver = a.solver if a.solver >= 0 else (1 if len(omegas) > 1 else 0)
    big = cfg["N"] >= 144
    e2e_steps = min(a.steps, 2) if big else a.steps
    rec = run_chi0(a, wb, cfg, w, dV_np, alpha, aux, omegas, solver, precision, a.steps, a.warmup, local, world, barrier, e2e_steps,
                   want_cpu=(2 if (world == 1 and rank == 0 and not a.no_cpu_baseline) else 0), label=a.workload)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    line = {"metric": "chi0*dV perturbations/s (batched Sternheimer PCG to tol %.0e)" % TOL, "value": rec.pop("value"), "unit": rec.pop("unit"),
            "n_gpus": world, "steps": a.steps, "warmup": a.warmup, "ms_per_step": rec.pop("ms_per_step"), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": rec.pop("dtype"), "data": "synthetic (seeded Si-like cell, GPU-computed orbitals)"}
    rec.pop("steps"); rec.pop("warmup")
    line.update(rec)
    if "e2e" in line and line["e2e"]["steps"] != a.steps:
        line["e2e"]["note"] = "end-to-end loop cut to %d steps (a step of this workload takes %.0f s)" % (line["e2e"]["steps"], line["ms_per_step"] / 1e3)

    # ---- sub-records: the other configs of BASELINE.json on the same driver clock (default workload, one GPU only)
    if a.workload == "cfg5" and a.omegas == "default" and world == 1 and not a.no_sub:
        subs = {}
        late = lambda: time.time() - T_START > SUB_DEADLINE_S
        skipped = {"skipped": "time budget of the run (%d s) reached before this sub-record" % SUB_DEADLINE_S}
        if precision == wb.WEST_FP64:
            # the headline workload once more with WEST_FP64_I8: the projector GEMMs as exact int8-slice products on tcgen05 kind::i8
            # (DESIGN.md section 6j).  Same inputs, same tolerance, same parity sample; a separate record because its dtype statement differs.
            try:
                if late():
                    raise TimeoutError(skipped["skipped"])
                subs["cfg5_i8"] = run_chi0(a, wb, cfg, w, dV_np, alpha, aux, omegas, solver, wb.WEST_FP64_I8, SUB_STEPS, SUB_WARMUP, local, world, barrier, 0,
                                           want_cpu=0 if a.no_cpu_baseline else 1, label="cfg5, projector GEMMs from int8 slices (WEST_FP64_I8)")
            except Exception as e:
                subs["cfg5_i8"] = {"error": repr(e)[:300]}
        try:
            if late():
                raise TimeoutError(skipped["skipped"])
            om_iw = [x for x in cfg["omegas"] if x > 0]
            r = run_chi0(a, wb, cfg, w, dV_np, alpha, aux, om_iw, 1 if a.solver < 0 else a.solver, precision, 1, 0, local, world, barrier, 0,
                         want_cpu=0 if a.no_cpu_baseline else 1, label="cfg5 imaginary frequencies", profile_in_timed=True)
            r["note"] = "ONE timed step, no warm-up of its own (the kernels are warm from the headline steps; a step takes about 100 s)"
            subs["cfg5_iw"] = r
        except Exception as e:
            subs["cfg5_iw"] = {"error": repr(e)[:300]}
        if precision == wb.WEST_FP64:
            # the same four frequencies with the int8-slice GEMMs - only while the run is early enough to leave the named configs their time
            try:
                if time.time() - T_START > 1150.0:
                    raise TimeoutError("skipped: the run had taken more than 1150 s before this optional sub-record")
                r = run_chi0(a, wb, cfg, w, dV_np, alpha, aux, om_iw, 1 if a.solver < 0 else a.solver, wb.WEST_FP64_I8, 1, 0, local, world, barrier, 0,
                             want_cpu=0 if a.no_cpu_baseline else 1, label="cfg5 imaginary frequencies, projector GEMMs from int8 slices (WEST_FP64_I8)", profile_in_timed=True)
                r["note"] = "ONE timed step, no warm-up of its own"
                subs["cfg5_iw_i8"] = r
            except Exception as e:
                subs["cfg5_iw_i8"] = {"error": repr(e)[:300]}
        w.close()
        del w, aux
        torch.cuda.empty_cache()
        try:
            c4 = synth.get_config("cfg4")
            w2, dV2, alpha2, aux2 = setup_gpu(c4, c4["n_pert"], a.chunk, verbose=True, alpha_factor=a.alpha_factor)
            w2.set_ms_history(a.ms_history)
            for name in ("cfg2", "cfg3", "cfg4"):
                if late():
                    subs[name] = dict(skipped)
                    continue
                try:
                    c = synth.get_config(name)
                    om = omegas_for(a, c, name)
                    prec = wb.WEST_MIXED if c["precision"] == "mixed" else wb.WEST_FP64
                    subs[name] = run_chi0(a, wb, c, w2, dV2[:c["n_pert"]], alpha2, aux2, om, 1 if len(om) > 1 else 0, prec, SUB_STEPS, SUB_WARMUP, local, world,
                                          barrier, SUB_STEPS if name == "cfg2" else 0, want_cpu=0 if a.no_cpu_baseline else (2 if name == "cfg2" else 1), label=name)
                except Exception as e:
                    subs[name] = {"error": repr(e)[:300]}
            w2.close()
            del w2, aux2
            torch.cuda.empty_cache()
            # cfg3 once more with west_set_deflation: 128 conduction eigenstates (an eigensolver's guard states) handed over as extra inputs.
            # Exact (DESIGN 6e); it lifts the lower end of the UNPRECONDITIONED multi-shift operator's spectrum, which is what sets its
            # iteration count.  A separate record: BASELINE's cfg3 is the plain one above.
            try:
                if late():
                    raise TimeoutError(skipped["skipped"])
                c3 = synth.get_config("cfg3")
                w3, dV3, alpha3, aux3 = setup_gpu(c3, c3["n_pert"], a.chunk, verbose=True, n_defl=128, alpha_factor=a.alpha_factor)
                w3.set_ms_history(a.ms_history)
                keep = a.deflate
                a.deflate = 128
                subs["cfg3_deflated"] = run_chi0(a, wb, c3, w3, dV3, alpha3, aux3, omegas_for(a, c3, "cfg3"), 1, wb.WEST_FP64, SUB_STEPS, SUB_WARMUP, local, world,
                                                 barrier, 0, want_cpu=0 if a.no_cpu_baseline else 1, label="cfg3 + 128 deflated conduction states")
                a.deflate = keep
                w3.close()
            except Exception as e:
                subs["cfg3_deflated"] = {"error": repr(e)[:300]}
        except Exception as e:
            subs["cfg2-4"] = {"error": repr(e)[:300]}
        line["workloads"] = subs
    else:
        w.close()
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def bench_kernels(a, wb, cfg, rank, world, barrier):
    """--op happly: metric (1) of BASELINE.json, H*psi applications/s of west_h_apply (KB projectors included) on random vectors of the
    workload's cell, with the per-kernel-class times; the small fixed launch set the ncu captures of profiles/ use.
    --op gemm: the KB + P_v contraction shapes of the CG loop (rows = n_proj + n_occ, n_vec columns, K = 2 n_g) on west_gemm_tn /
    west_gemm_update next to cuBLAS DGEMM (through torch) on the same operands."""
    import torch
    import synth
    mode = wb.WEST_GAMMA if cfg["mode"] == "gamma" else wb.WEST_FULL
    w = wb.West(cfg["L"], cfg["n2max"], cfg["N"], mode)
    g = torch.Generator(device="cuda").manual_seed(1)
    n_vec = a.n_vec or cfg.get("pert_batch", cfg["n_pert"]) * cfg["n_occ"]
    rows = (cfg["n_proj"] + cfg["n_occ"]) * (1 if mode == wb.WEST_GAMMA else 2)
    K = 2 * w.n_g
    prec = wb.WEST_MIXED if a.precision == "mixed" else (wb.WEST_FP64_I8 if a.precision == "i8" else wb.WEST_FP64)
    hbm_peak, peak_src = peaks()
    if a.op == "gemm":
        A = torch.randn(rows, K, dtype=torch.float64, device="cuda", generator=g)
        B = torch.randn(n_vec, K, dtype=torch.float64, device="cuda", generator=g)
        Cm = torch.randn(rows, n_vec, dtype=torch.float64, device="cuda", generator=g)
        out = torch.empty(rows, n_vec, dtype=torch.float64, device="cuda")

        def tm(fn):
            for _ in range(max(1, a.warmup)):
                fn()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(a.steps):
                fn()
            e1.record()
            torch.cuda.synchronize()
            return e0.elapsed_time(e1) / a.steps
        fl = 2.0 * rows * n_vec * K
        t_tn, t_up = tm(lambda: w.gemm_tn(A, B, out)), tm(lambda: w.gemm_update(Cm, A, B))
        t_ctn, t_cup = tm(lambda: torch.matmul(A, B.T, out=out)), tm(lambda: B.addmm_(Cm.T, A))
        peak = measure_fp64_peak()
        print(json.dumps({"metric": "projector GEMM TFLOP/s (FP64 DMMA)", "value": fl / t_tn / 1e9, "unit": "TFLOP/s", "n_gpus": 1, "steps": a.steps, "warmup": a.warmup,
                          "ms_per_step": t_tn + t_up, "higher_is_better": True, "dtype": "f64", "data": "synthetic (normal random operands)",
                          "config": {"workload": a.workload, "op": "gemm", "rows": rows, "n_vec": n_vec, "k": K},
                          "west_gemm_tn": {"ms": t_tn, "tflops": fl / t_tn / 1e9}, "west_gemm_update": {"ms": t_up, "tflops": fl / t_up / 1e9},
                          "cublas_tn": {"ms": t_ctn, "tflops": fl / t_ctn / 1e9}, "cublas_update": {"ms": t_cup, "tflops": fl / t_cup / 1e9},
                          "fp64_peak_tflops": peak, "gpu_launches": int(w.launch_count())}))
        w.close()
        return
    atoms, vloc = build_inputs(cfg)
    miller, _, _, _ = w.gsphere()
    beta, dcoef = synth.kb_projectors(miller, cfg["L"], atoms, 0.8, cfg["projectors"])
    w.set_vloc(torch.from_numpy(vloc).cuda())
    w.set_kb(torch.from_numpy(np.ascontiguousarray(beta)).cuda(), dcoef)
    x = torch.randn((n_vec, w.n_g), dtype=torch.float64, device="cuda", generator=g) + 0j
    y = torch.empty_like(x)
    ws = torch.empty(w.workspace_bytes(wb.binding.WEST_OP_H_APPLY, n_vec, 1, prec), dtype=torch.uint8, device="cuda")
    w.set_workspace(ws)
    for _ in range(max(1, a.warmup)):
        w.h_apply(x, y, precision=prec)
    barrier()
    l0 = w.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(a.steps):
        w.h_apply(x, y, precision=prec)
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1) / a.steps
    launches = w.launch_count() - l0
    w.set_profile(True)
    w.h_apply(x, y, precision=prec)
    prof = w.get_profile()
    w.set_profile(False)
    fp64_peak = measure_fp64_peak()
    top = max(("k1_g2r_z", "k2_planes", "k3_r2g_z"), key=lambda k: prof[k]["ms"])
    t_fft = sum(prof[k]["ms"] for k in ("k1_g2r_z", "k2_planes", "k3_r2g_z")) * 1e-3
    n_cols = aux_ncols(cfg)
    csz = 8 if prec == wb.WEST_MIXED else 16
    slots = n_vec / (2 if mode == wb.WEST_GAMMA else 1)
    fft_bytes = (4 * cfg["N"] * n_cols * csz + 3 * (2 if mode == wb.WEST_GAMMA else 1) * w.n_g * 16) * slots
    print(json.dumps({"metric": "H*psi applications/s (west_h_apply, KB projectors included)", "value": n_vec * world / (ms * 1e-3), "unit": "vectors/s", "n_gpus": world,
                      "steps": a.steps, "warmup": a.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                      "dtype": {wb.WEST_FP64: "f64", wb.WEST_MIXED: "f32 FFT + 3xTF32 GEMMs", wb.WEST_FP64_I8: "f64 (projector GEMMs: exact int8-slice products on tcgen05 kind::i8, FP64 sums)"}[prec], "data": "synthetic (normal random vectors)",
                      "config": {"workload": a.workload, "op": "happly", "n_vec": n_vec, "N": cfg["N"], "n_g": w.n_g, "n_proj": cfg["n_proj"]},
                      "gpu_launches": int(launches), "kernel_ms_per_step": {k: round(v["ms"], 3) for k, v in prof.items() if v["spans"]},
                      "fft_path": {"ms": t_fft * 1e3, "algorithmic_gbs": fft_bytes / t_fft / 1e9, "frac_of_hbm": fft_bytes / t_fft / 1e9 / hbm_peak, "peak_source": peak_src,
                                   "note": "K1 + K2 + K3 against their algorithmic bytes (DESIGN.md section 6)"},
                      "roofline": roofline(cfg, top, prof, n_vec, 1, 0, hbm_peak, peak_src, prec == wb.WEST_MIXED, w.n_g, fp64_peak)}))
    w.set_workspace(None)
    w.close()


def bench_lanczos(a, cfg, w, phi, n_pert, rank, world, barrier, n_steps=30):
    """Widening row SURVEY 8(f)-2: N_Lanczos = 30 chains for every (perturbation, orbital), brakets included."""
    import torch
    for _ in range(a.warmup):
        al, be, _, _ = w.lanczos(phi, n_steps, cfg["n_occ"], want_brakets=True)
        w.lanczos_diag(al, be)
    barrier()
    w.set_profile(True)
    l0 = w.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(a.steps):
        al, be, _, _ = w.lanczos(phi, n_steps, cfg["n_occ"], want_brakets=True)
        w.lanczos_diag(al, be)                      # d, U of Eq. 19 for every chain
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    prof = w.get_profile()
    w.set_profile(False)
    if rank != 0:
        return
    chains = n_pert * cfg["n_occ"] * world
    print(json.dumps({"metric": "Lanczos chains/s (N_Lanczos = %d, brakets and tridiagonal eigensolves included)" % n_steps, "value": chains * a.steps / (ms * 1e-3),
                      "unit": "chains/s", "n_gpus": world, "steps": a.steps, "warmup": a.warmup, "ms_per_step": ms / a.steps,
                      "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                      "config": {"workload": a.workload, "op": "lanczos", "n_pert_per_gpu": n_pert, "n_occ": cfg["n_occ"], "n_steps": n_steps},
                      "h_apply_per_s": chains * n_steps * a.steps / (ms * 1e-3), "gpu_launches": int(w.launch_count() - l0),
                      "kernel_ms_per_step": {k: round(v["ms"] / a.steps, 3) for k, v in prof.items() if v["spans"]}}))


def bench_pdep(a, cfg, w, alpha, n_pdep, rank, world, barrier):
    """Widening row SURVEY 8(f)-3: wstat-like run, N_PDEP leading eigenpotentials of chi0bar by Davidson (residual 1e-4, CG tol 1e-8)."""
    import torch
    from paper_2203_05623_b200 import pdep as gp
    out = None
    for _ in range(a.warmup):
        out = gp.pdep(w, n_pdep, cfg["n_occ"], alpha, tol=1e-4, tol_cg=TOL)
    barrier()
    t0 = time.perf_counter()
    for _ in range(a.steps):
        out = gp.pdep(w, n_pdep, cfg["n_occ"], alpha, tol=1e-4, tol_cg=TOL)
    torch.cuda.synchronize()
    dt = (time.perf_counter() - t0) / a.steps
    if rank != 0:
        return
    lam, _, res, n_app = out
    print(json.dumps({"metric": "PDEP Davidson time (N_PDEP = %d, residual 1e-4)" % n_pdep, "value": dt, "unit": "s", "n_gpus": world,
                      "steps": a.steps, "warmup": a.warmup, "ms_per_step": dt * 1e3, "higher_is_better": False, "scaling": "weak",
                      "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                      "config": {"workload": a.workload, "op": "pdep", "n_pdep": n_pdep, "chi0_applications": int(n_app),
                                 "lambda_min": float(lam[0]), "lambda_max_kept": float(lam[-1]), "max_residual": float(res.max())},
                      "chi0_applications_per_s": n_app / dt}))


def bench_spin(a, cfg, dV, n_pert, rank, world, barrier, kw):
    """Widening row SURVEY 8(f)-4, second half: the same cell with N_spin = 2.  h^sigma = T + V_loc +- B + V_NL (synth.spin_splitting_field),
    n_occ orbitals per channel with one electron each; a step = chi0*dV summed over both channels (two Sternheimer batches)."""
    import torch
    import synth
    import paper_2203_05623_b200 as wb
    B = synth.spin_splitting_field(cfg)
    ws, alphas, gaps = [], [], []
    for sgn in (+1, -1):
        w, _, alpha, aux = setup_gpu(cfg, 1, a.chunk, verbose=(rank == 0), vloc_add=sgn * B)
        ws.append(w); alphas.append(alpha); gaps.append(aux["gap"])
    kw = dict(kw, alpha_pv=alphas)
    kw.pop("dn")
    stats = None
    for _ in range(a.warmup):
        _, stats = wb.West.chi0_apply_spin(ws, dV, [0.0], **kw)
    barrier()
    l0 = sum(w.launch_count() for w in ws)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(a.steps):
        _, stats = wb.West.chi0_apply_spin(ws, dV, [0.0], **kw)
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    if rank != 0:
        return
    print(json.dumps({"metric": "spin-polarised chi0*dV perturbations/s (N_spin = 2, PCG to tol %.0e)" % TOL, "value": n_pert * world * a.steps / (ms * 1e-3),
                      "unit": "perturbations/s", "n_gpus": world, "steps": a.steps, "warmup": a.warmup, "ms_per_step": ms / a.steps,
                      "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                      "config": {"workload": a.workload, "op": "spin", "n_spin": 2, "n_pert_per_gpu": n_pert, "n_occ_per_channel": cfg["n_occ"],
                                 "gaps_ry": gaps, "cg_iters": [st["iters"] for st in stats], "unconverged": [st["n_unconverged"] for st in stats]},
                      "h_apply_per_s": sum(st["n_h_apply"] for st in stats) * world / (ms / a.steps * 1e-3),
                      "gpu_launches": int(sum(w.launch_count() for w in ws) - l0), "device_gb": sum(w.device_bytes() for w in ws) / 1e9}))


def bench_fft(a, rank, world, local):
    """Widening row SURVEY 8(f)-4, first half: Fig. 3 of the paper - ONE dense C2C FFT of a 128^3 or 256^3 grid, FP64 or
    FP32, data resident on the device, mean over the timed steps (the paper averages 100: run with --steps 100).  Each step is timed
    with its own CUDA-event pair and a 256 MB L2 flush in between, because the 128^3 grid fits the 126 MB L2.  N > 1: replicas."""
    import torch
    import torch.distributed as dist
    import synth
    import paper_2203_05623_b200 as wb
    n = {"fft128": 128, "fft256": 256, "fft64": 64}.get(a.workload)
    if n is None:
        raise SystemExit("--op fft needs --workload fft64 | fft128 | fft256")
    if a.impl == "reference":
        if rank == 0:
            from oracle import fft_dense as ofd
            ts = []
            ns = min(n, 128)
            xs = synth.dense_grid(ns, 1)[0]
            for _ in range(a.warmup + a.steps):
                t0 = time.time()
                ofd.dft3(xs, -1)
                ts.append((time.time() - t0) * (n / ns) ** 4)
            v = float(np.mean(ts[a.warmup:])) * 1e3
            print(json.dumps({"impl": "reference", "metric": "time of one dense C2C 3D FFT (Fig. 3)", "value": v, "unit": "ms", "n_gpus": a.gpus,
                              "steps": a.steps, "warmup": a.warmup, "ms_per_step": v, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
                              "dtype": "f64", "data": "synthetic", "config": {"workload": a.workload, "op": "fft", "n": n},
                              "cpu_baseline": {"value": v, "unit": "ms", "cores": len(os.sched_getaffinity(0)), "kind": "oracle",
                                               "sample": "oracle.fft_dense.dft3 on the whole grid" if n <= 128 else "dft3 on a 128^3 grid, time scaled by 16 (its cost is 3 n^4)"},
                              "e2e": {"value": v, "unit": "ms", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))
        return
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    cdt, esz = (torch.complex128, 16) if a.precision == "fp64" else (torch.complex64, 8)
    x_np = synth.dense_grid(n, 1)
    x = torch.from_numpy(x_np).to("cuda", dtype=cdt)
    y = torch.empty_like(x)
    w = wb.West(10.0, 25, 24, wb.WEST_FULL)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    def timed(fn, k):
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(k)]
        for e0, e1 in ev:
            flush.zero_()
            e0.record(); fn(); e1.record()
        torch.cuda.synchronize()
        return [e0.elapsed_time(e1) for e0, e1 in ev]

    for _ in range(max(a.warmup, 3)):
        w.fft3d_dense(x, -1, out=y)
        torch.fft.fftn(x, dim=(1, 2, 3), out=y)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local)
    sampler.start()
    l0 = w.launch_count()
    t = timed(lambda: w.fft3d_dense(x, -1, out=y), a.steps)
    launches = w.launch_count() - l0
    sampler.stop_flag.set(); sampler.join()
    t_lib = timed(lambda: torch.fft.fftn(x, dim=(1, 2, 3), out=y), a.steps)
    # back-to-back variant: one event pair around KB transforms of KB DIFFERENT grids (together larger than the L2, so
    # every transform still reads cold data) - the host's enqueue time of a single call no longer sits inside the bracket
    KB = max(8, min(20, (1 << 30) // (x.numel() * esz)))
    xs = [x.clone() for _ in range(KB)]

    def batched(fn):
        for xi in xs:
            fn(xi)
        best = []
        for _ in range(5):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for xi in xs:
                fn(xi)
            e1.record()
            torch.cuda.synchronize()
            best.append(e0.elapsed_time(e1) / KB)
        return float(np.median(best))
    tb_own = batched(lambda xi: w.fft3d_dense(xi, -1, out=y))
    tb_lib = batched(lambda xi: torch.fft.fftn(xi, dim=(1, 2, 3), out=y))
    del xs
    # end to end: pinned host grid -> device, transform, result -> pinned host
    hx = torch.from_numpy(x_np[...]).to(cdt).pin_memory()
    hy = torch.empty_like(hx).pin_memory()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(a.steps):
        x.copy_(hx, non_blocking=True)
        w.fft3d_dense(x, -1, out=y)
        hy.copy_(y, non_blocking=True)
        torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3 / a.steps
    ms = float(np.mean(t))
    tt = torch.tensor([ms, e2e_ms], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        dist.destroy_process_group()
    ms, e2e_ms = float(tt[0]), float(tt[1])
    if rank != 0:
        return
    hbm_peak, peak_src = peaks()
    alg = 2.0 * n ** 3 * esz
    line = {"metric": "time of one dense C2C 3D FFT (Fig. 3)", "value": ms, "unit": "ms", "n_gpus": world, "steps": a.steps, "warmup": max(a.warmup, 3),
            "ms_per_step": ms, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64" if esz == 16 else "f32", "data": "synthetic (seeded complex normal grid)",
            "config": {"workload": a.workload, "op": "fft", "n": n, "precision": a.precision, "l2": "256 MB flush between timed steps", "replicas": world},
            "ffts_per_s": world * 1e3 / ms, "ms_median": float(np.median(t)),
            "library": {"what": "cuFFT through torch.fft.fftn, same buffers, same timing loop", "ms_mean": float(np.mean(t_lib)), "ratio": float(np.mean(t_lib)) / ms},
            "back_to_back": {"what": "%d transforms of %d different grids per event pair (GPU time per transform, host enqueue outside); value / ms_mean above are single calls, host-inclusive" % (KB, KB),
                             "ms": tb_own, "library_ms": tb_lib, "ratio": tb_lib / tb_own},
            "e2e": {"value": e2e_ms, "unit": "ms", "h2d_bytes_per_step": int(x.numel() * esz), "d2h_bytes_per_step": int(y.numel() * esz)},
            "gpu_launches": int(launches), "clocks": sampler.summary(),
            "roofline": {"kernel": "dense_axis_pass (3 launches per FFT)", "bound": "hbm", "achieved": alg / (ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                         "frac": alg / (ms * 1e-3) / 1e9 / hbm_peak, "peak_source": peak_src, "traffic": None,
                         "algorithmic_bytes": alg, "note": "algorithmic = read the grid once + write it once; the three axis passes move 3x that "
                                                         "(through HBM at 256^3, mostly through L2 at 128^3): three_pass_frac = %.3f" % (3 * alg / (ms * 1e-3) / 1e9 / hbm_peak)}}
    if world == 1 and not a.no_cpu_baseline:
        from oracle import fft_dense as ofd
        # the DFT-matrix definition costs 3 n^4 complex multiply-adds: 256^3 takes ~50 s, so it is sampled on the 128^3 grid and scaled by 16
        ns = min(n, 128)
        xs = x_np[0] if ns == n else synth.dense_grid(ns, 1)[0]
        t0 = time.time()
        ofd.dft3(xs, -1)
        dt = (time.time() - t0) * (n / ns) ** 4
        sample = "oracle.fft_dense.dft3 (DFT matrices) on the whole %d^3 grid" % n if ns == n else \
                 "oracle.fft_dense.dft3 on a 128^3 grid, time scaled by (256/128)^4 = 16 (its cost is 3 n^4)"
        line["cpu_baseline"] = {"value": dt * 1e3, "unit": "ms", "cores": len(os.sched_getaffinity(0)), "kind": "oracle", "sample": sample}
    print(json.dumps(line))




def oracle_states(cfg):
    """Occupied orbitals from the ORACLE's own eigensolver (oracle.iterative.lowest_states), cached under .cache/ (git-ignored)."""
    from oracle import gsphere as ogs
    from oracle import iterative as oit
    import synth
    m = ogs.enumerate_sphere(cfg["n2max"])
    atoms = synth.atoms_for(cfg)
    vloc = synth.vloc_for(cfg, atoms)
    beta, dcoef = synth.kb_projectors(m, cfg["L"], atoms, 0.8, cfg["projectors"])
    path = os.path.join(ROOT, ".cache", "oracle_states_cfg%d_%d.npz" % (cfg["cfg"], cfg["n_occ"]))
    if os.path.exists(path):
        d = np.load(path)
        eps, U = d["eps"], d["U"]
    else:
        if cfg["mode"] == "gamma":
            eps, U, _ = oit.lowest_states(cfg["n_occ"], m, cfg["L"], cfg["N"], vloc, beta, dcoef, tol=1e-9)
        else:
            from oracle import hamiltonian as oham
            eps, Uall = oham.eigensystem(oham.dense_h(m, cfg["L"], cfg["N"], vloc, beta, dcoef), m, real_orbitals=False)
            eps, U = eps[:cfg["n_occ"]], Uall[:, :cfg["n_occ"]]
        try:
            os.makedirs(os.path.dirname(path), exist_ok=True)
            np.savez(path, eps=eps, U=U)
        except OSError:
            pass
    return m, vloc, beta, dcoef, eps, U


def run_reference(a, cfg, n_pert, omegas):
    """--impl reference: the oracle (oracle/) as it stands on the host cores, on its own inputs - nothing of the CUDA library is loaded.
    Each step is a bounded sample of the workload: (perturbation 0, state v) columns solved by the oracle's PCG / COCG for about
    8 s.  cfg 5: a 1024-state eigensolve at 145 405 plane waves is infeasible on the host, so a step times PCG ITERATIONS at that size
    (the oracle's H*psi plus the P_v products, random vectors in place of the orbitals) and the iteration count per column is the
    oracle's own mean on the one-cell Si-like mini2 (same material, cutoff, preconditioner and alpha rule)."""
    import synth
    from oracle import chi0 as ochi0
    from oracle import gsphere as ogs
    from oracle import hamiltonian as oham
    from oracle import iterative as oit
    cores = len(os.sched_getaffinity(0))
    n_occ, L, N = cfg["n_occ"], cfg["L"], cfg["N"]
    big = N >= 144
    n_freq = len(omegas)
    vals, sample = [], ""
    if not big:
        m, vloc, beta, dcoef, eps, U = oracle_states(cfg)
        idx, g2, minus = ogs.fft_index(m, N), ogs.g2_of(m, L), ogs.index_of_minus(m)
        apply_H = lambda y: oham.apply_h(y, m, L, N, vloc, beta, dcoef)
        width = float(eps[n_occ - 1] - eps[0])
        dV0 = synth.perturbations(cfg, n_pert=1)[0]
        v_next = 0
        for _ in range(a.warmup + a.steps):
            t0 = time.time()
            done = 0
            while time.time() - t0 < 8.0:
                v = v_next % n_occ
                v_next += 1
                b = ochi0.rhs_vectors(U[:, v:v + 1], dV0[None], idx, N)[0, 0]
                al = max(float(eps[v] - eps[0]) + 0.5 * width, 0.01)
                for om in omegas:
                    if om > 0:
                        oit.cocg_sternheimer(apply_H, U, eps[v], v, b, g2, minus, al, om, tol=TOL, max_iter=MAX_ITER)
                    else:
                        oit.pcg_sternheimer(apply_H, U, eps[v], v, b, g2, al, tol=TOL, max_iter=MAX_ITER)
                done += 1
            # `done` columns x n_freq solves in dt seconds; a perturbation is n_occ columns
            vals.append(done * n_freq / n_occ / (time.time() - t0))
        sample = "per step: oracle PCG/COCG on (i=0, v) columns for 8 s (%d frequencies each), orbitals from oracle.iterative.lowest_states" % n_freq
    else:
        mini = synth.get_config("mini2")
        mm = ogs.enumerate_sphere(mini["n2max"])
        at = synth.atoms_for(mini)
        vl = synth.vloc_for(mini, at)
        be, dc = synth.kb_projectors(mm, mini["L"], at, 0.8, mini["projectors"])
        e_m, U_m = oham.eigensystem(oham.dense_h(mm, mini["L"], mini["N"], vl, be, dc), mm, real_orbitals=True)
        idx_m, g2_m = ogs.fft_index(mm, mini["N"]), ogs.g2_of(mm, mini["L"])
        Uo = U_m[:, :mini["n_occ"]]
        wd = float(e_m[mini["n_occ"] - 1] - e_m[0])
        dVm = synth.perturbations(mini, n_pert=1)[0]
        its = []
        for v in range(mini["n_occ"]):
            b = ochi0.rhs_vectors(Uo[:, v:v + 1], dVm[None], idx_m, mini["N"])[0, 0]
            _, it, _ = oit.pcg_sternheimer(lambda y: oham.apply_h(y, mm, mini["L"], mini["N"], vl, be, dc), Uo, e_m[v], v, b, g2_m,
                                           max(float(e_m[v] - e_m[0]) + 0.5 * wd, 0.01), tol=TOL, max_iter=MAX_ITER)
            its.append(it)
        iters_col = float(np.mean(its))
        m = ogs.enumerate_sphere(cfg["n2max"])
        atoms = synth.atoms_for(cfg)
        vloc = synth.vloc_for(cfg, atoms)
        beta, dcoef = synth.kb_projectors(m, L, atoms, 0.8, cfg["projectors"])
        rng = np.random.Generator(np.random.PCG64(5))
        n = len(m)
        Ur = (rng.standard_normal((n, n_occ)) + 1j * rng.standard_normal((n, n_occ))) / np.sqrt(2.0 * n)
        x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
        for _ in range(a.warmup + a.steps):
            t0 = time.time()
            y = oham.apply_h(x, m, L, N, vloc, beta, dcoef)
            y = y - 0.3 * x + 1.0 * (Ur @ (Ur.conj().T @ x))          # the shift and alpha P_v of one operator application
            x2 = x + 0.1 * y                                           # the vector updates and dots of one PCG iteration
            _ = np.vdot(x2, y), np.vdot(y, y)
            dt = time.time() - t0
            # omega > 0 (COCG): the same iteration on complex vectors, same cost per frequency in this CPU code
            vals.append(1.0 / (n_occ * dt * iters_col))
        sample = ("per step: ONE PCG iteration of the oracle at cfg5 size (oracle.hamiltonian.apply_h + P_v products on %d coefficients, random vectors in place of "
                  "orbitals: a 1024-state eigensolve is infeasible on the host); value = 1 / (n_occ x s-per-iteration x %.1f iterations per column, "
                  "the oracle PCG's mean on mini2)" % (n, iters_col))
    vals = vals[a.warmup:]
    v = float(np.mean(vals))
    line = {"impl": "reference", "metric": "chi0*dV perturbations/s (batched Sternheimer PCG to tol %.0e)" % TOL, "value": v,
            "unit": "perturbations/s", "n_gpus": a.gpus, "steps": a.steps, "warmup": a.warmup, "ms_per_step": 1e3 * n_pert * n_freq / v if v else None,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic (seeded Si-like cell, oracle-side inputs)",
            "config": {"workload": a.workload, "N": N, "n_occ": n_occ, "n_pert_per_gpu": n_pert, "n_freq": n_freq, "omega_ry": [round(x, 6) for x in omegas],
                       "n_proj": cfg["n_proj"], "tol": TOL, "solver": "PCG/COCG per column (oracle/iterative.py)", "alpha_pv": "per-orbital (eps_v - eps_1) + W/2"},
            "cpu_baseline": {"value": v, "unit": "perturbations/s", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": "perturbations/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


if __name__ == "__main__":
    main()
