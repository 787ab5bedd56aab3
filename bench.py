#!/usr/bin/env python
"""bench.py - throughput of the chi0*dV hot path (Eq. 10-11 of arXiv 2203.05623) on B200, one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2] [--impl reference]

A step = one west_chi0_apply over the workload's perturbation block: RHS (a1), batched PCG to the stated tolerance with
the dual-space H*psi, KB / P_v GEMMs and fused vector updates (a2-a9), and the dn accumulation (a10).
metric  = chi0*dV perturbations/s (whole job, all ranks); the line also carries H*psi applications/s.
N > 1   = weak scaling: every rank holds the full orbitals and its own block of perturbations, no collective on the
          data path ("images"); value = all ranks' perturbations / max-over-ranks time.
--impl reference = the CPU oracle (oracle/) timed on a bounded sample of the same workload.
Inputs are seeded and synthetic (synth/), the occupied orbitals come from the library's own GPU eigensolver (set-up,
untimed).  Nothing here reads /root/reference.
"""
import argparse
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


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg2")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--chunk", type=int, default=0, help="FFT slots per chunk (0 = library default)")
    ap.add_argument("--check-every", type=int, default=1, help="CG convergence poll / compaction period")
    ap.add_argument("--precond", type=int, default=1, help="0 none, 1 R4 default, 2 Teter-Payne-Allan")
    ap.add_argument("--solver", type=int, default=-1, help="0 per-frequency PCG/COCG, 1 multi-shift CG; -1 = 1 for cfg3, else 0")
    ap.add_argument("--op", default="chi0", choices=["chi0", "lanczos", "pdep", "fft", "spin"],
                    help="chi0 = the hot path (default); lanczos = Eq. 15-19 chains; pdep = Davidson shell for chi0bar; fft = the dense "
                         "C2C FFT of Fig. 3 (--workload fft128 | fft256, --precision); spin = N_spin = 2 chi0 (widening rows)")
    ap.add_argument("--precision", default="fp64", choices=["fp64", "fp32"], help="--op fft only")
    ap.add_argument("--deflate", type=int, default=0, help="number of conduction eigenstates handed to west_set_deflation (0 = off)")
    ap.add_argument("--n-pert", type=int, default=0, help="override the perturbation count (0 = the config's)")
    ap.add_argument("--alpha-factor", type=float, default=1.5, help="alpha_pv = factor x (eps_Nv - eps_1), reading R3 (the result does not depend on it; "
                                                                         "must exceed 1; measured at cfg 2: 1.25 fastest, 1.5 keeps half a band width of margin, DESIGN.md R3)")
    ap.add_argument("--cg-kernel", type=int, default=0, help="west_set_cg_kernel: 0 automatic (column-resident where it fits), 1 streaming, 2 column split over a 2-CTA cluster")
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

    def summary(self):
        sm = [float(r[0]) for r in self.rows if r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) > 2 + i and r[2 + i].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons,
                "samples": len(self.rows)}


def build_inputs(cfg):
    """Seeded synthetic cell (synth/): potentials, projectors on the library's own sphere, perturbations."""
    import synth
    atoms = synth.atoms_for(cfg)
    vloc = synth.vloc_for(cfg, atoms)
    return atoms, vloc


def setup_gpu(cfg, n_pert, chunk, verbose, n_defl=0, vloc_add=None, alpha_factor=1.5):
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
        print("# eigensolver: %.1f s, residual %.2e, gap %.4f Ry" % (time.time() - t0, res, gap), file=sys.stderr)
    w.set_states(psi, eps[:cfg["n_occ"]])
    alpha = max(alpha_factor * float(eps[cfg["n_occ"] - 1] - eps[0]), 0.01)
    dV = synth.perturbations(cfg, n_pert=n_pert)
    return w, dV, alpha, dict(eps=eps, psi=psi, gap=gap, res=res, miller=miller, vloc=vloc, beta=beta, dcoef=dcoef)


def cpu_baseline(cfg, aux, dV0, alpha, budget_s=20.0):
    """The oracle's own PCG route (oracle/iterative.py) on a bounded sample of (perturbation 0, state v) columns.

    The orbitals handed to it are the bench's GPU-computed ones; the oracle first re-checks them as eigenvectors with its
    own matrix-free H (no parity claim rests on this leg - it is a timing baseline)."""
    from oracle import gsphere as ogs
    from oracle import hamiltonian as oham
    from oracle import iterative as oit
    from oracle import chi0 as ochi0
    L, N = cfg["L"], cfg["N"]
    m = ogs.enumerate_sphere(cfg["n2max"])
    idx = ogs.fft_index(m, N)
    g2 = ogs.g2_of(m, L)
    gamma = cfg["mode"] == "gamma"
    sel = np.nonzero(ogs.half_sphere_mask(m))[0] if gamma else np.arange(len(m))
    psi = aux["psi"].cpu().numpy()
    U = (ogs.expand_half_to_full(psi, m) if gamma else psi).T.copy()          # [n_g_full, n_occ]
    beta = ogs.expand_half_to_full(aux["beta"], m) if gamma else aux["beta"]
    eps = aux["eps"]
    apply_H = lambda y: oham.apply_h(y, m, L, N, aux["vloc"], beta, aux["dcoef"])
    r = apply_H(U[:, 0]) - eps[0] * U[:, 0]
    assert np.linalg.norm(r) < 1e-6, "orbitals are not eigenvectors of the oracle's H"
    b = ochi0.rhs_vectors(U, dV0[None], idx, N)[0]                             # [n_occ, n_g]
    cores = len(os.sched_getaffinity(0))
    t0 = time.time()
    n_done, iters = 0, 0
    for v in range(cfg["n_occ"]):
        x, it, rel = oit.pcg_sternheimer(apply_H, U, eps[v], v, b[v], g2, alpha, tol=TOL, max_iter=MAX_ITER)
        n_done += 1
        iters += it
        if time.time() - t0 > budget_s:
            break
    dt = time.time() - t0
    return {"value": n_done / cfg["n_occ"] / dt, "unit": "perturbations/s", "cores": cores, "kind": "oracle",
            "sample": "oracle.iterative.pcg_sternheimer on %d of %d (i=0, v) columns of %s, tol %.0e, %d H*psi, %.1f s"
                      % (n_done, cfg["n_occ"], cfg["name"], TOL, iters, dt),
            "h_apply_per_s": iters / dt}


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
    omegas = [0.0] if a.workload != "cfg3" else list(cfg["omegas"])

    if a.impl == "reference":
        if rank != 0:
            return
        run_reference(a, cfg, n_pert)
        return

    import torch
    import torch.distributed as dist
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    import paper_2203_05623_b200 as wb
    precision = wb.WEST_MIXED if cfg["precision"] == "mixed" else wb.WEST_FP64
    # every rank: same cell and orbitals, its own block of perturbations (seeded stream offset by rank)
    w, dV_np, alpha, aux = setup_gpu(cfg, n_pert, a.chunk, verbose=(rank == 0), n_defl=a.deflate, alpha_factor=a.alpha_factor)
    w.set_cg_kernel(a.cg_kernel)
    if world > 1:
        dV_np = synth.perturbations(cfg, n_pert=n_pert, first=rank * n_pert)
    dev = torch.device("cuda")
    dV = torch.from_numpy(dV_np).to(dev)
    N = cfg["N"]
    dn = torch.empty((len(omegas), n_pert, N, N, N), dtype=torch.float64, device=dev)
    solver = a.solver if a.solver >= 0 else (1 if a.workload == "cfg3" else 0)
    kw = dict(solver=solver, tol=TOL, max_iter=MAX_ITER if solver == 0 else 2000, alpha_pv=alpha, precond=a.precond, check_every=a.check_every, precision=precision, dn=dn)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if a.op == "lanczos":
        return bench_lanczos(a, cfg, w, dV, n_pert, rank, world, barrier)
    if a.op == "pdep":
        return bench_pdep(a, cfg, w, alpha, n_pert, rank, world, barrier)
    if a.op == "spin":
        w.close()
        return bench_spin(a, cfg, dV, n_pert, rank, world, barrier, kw)
    stats = None
    for _ in range(a.warmup):
        _, _, stats = w.chi0_apply(dV, omegas, **kw)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    w.set_profile(True)
    launches0 = w.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    n_h = 0
    for _ in range(a.steps):
        _, _, stats = w.chi0_apply(dV, omegas, **kw)
        n_h += stats["n_h_apply"]
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    prof = w.get_profile()
    w.set_profile(False)
    launches = w.launch_count() - launches0
    sampler.stop_flag.set()
    sampler.join()

    # ---- end to end: pinned host dV -> device, chi0_apply, dn -> pinned host, all inside the timed region
    h_dV = torch.from_numpy(dV_np).pin_memory()
    h_dn = torch.empty(dn.shape, dtype=torch.float64).pin_memory()
    barrier()
    t0 = time.perf_counter()
    for _ in range(a.steps):
        dV.copy_(h_dV, non_blocking=True)
        w.chi0_apply(dV, omegas, **kw)
        h_dn.copy_(dn, non_blocking=True)
        torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0

    t = torch.tensor([ms, e2e_s * 1e3], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms, e2e_ms = float(t[0]), float(t[1])
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    units = n_pert * len(omegas) * world
    value = units * a.steps / (ms * 1e-3)
    hbm_peak, peak_src = peaks()
    # ---- roofline of the dominant kernel class
    top = max(prof, key=lambda k: prof[k]["ms"])
    n_cols = aux_ncols(cfg)
    fp64_peak = measure_fp64_peak()
    roof = roofline(cfg, top, prof, n_h, stats, hbm_peak, peak_src, n_cols, precision == wb.WEST_MIXED, w, fp64_peak)
    rows = (cfg["n_proj"] + cfg["n_occ"]) * (1 if cfg["mode"] == "gamma" else 2)
    t_gemm = (prof["gemm_tn"]["ms"] + prof["gemm_update"]["ms"]) * 1e-3
    gemm_tf = 2 * 2.0 * rows * (2 * w.n_g) * n_h / t_gemm / 1e12 if t_gemm > 0 else None
    line = {
        "metric": "chi0*dV perturbations/s (batched Sternheimer PCG to tol %.0e)" % TOL,
        "value": value, "unit": "perturbations/s", "n_gpus": world, "steps": a.steps, "warmup": a.warmup,
        "ms_per_step": ms / a.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64" if precision == wb.WEST_FP64 else "f32 FFT / f64 vectors",
        "data": "synthetic (seeded Si-like cell, GPU-computed orbitals)",
        "config": {"workload": a.workload, "N": N, "n_g": w.n_g, "n_occ": cfg["n_occ"], "n_pert_per_gpu": n_pert, "n_freq": len(omegas),
                   "n_proj": cfg["n_proj"], "n_deflated": a.deflate, "alpha_pv_factor": a.alpha_factor, "tol": TOL, "solver": "multi-shift CG" if solver == 1 else "PCG/COCG per frequency", "cg_iters": stats["iters"], "unconverged": stats["n_unconverged"],
                   "gap_ry": aux["gap"], "l2": "inputs per step (4 vector sets, %.1f GB) exceed the 126 MB L2" % (4 * 16 * w.n_g * n_pert * cfg["n_occ"] / 1e9)},
        "h_apply_per_s": n_h * world / (ms * 1e-3),
        "e2e": {"value": units * a.steps / (e2e_ms * 1e-3), "unit": "perturbations/s",
                "h2d_bytes_per_step": int(dV.numel() * 8), "d2h_bytes_per_step": int(dn.numel() * 8)},
        "gpu_launches": int(launches),
        "clocks": sampler.summary(),
        "roofline": roof,
        "gemm": {"achieved_tflops": gemm_tf, "peak_tflops": fp64_peak, "frac": (gemm_tf / fp64_peak) if gemm_tf else None,
                 "note": "KB + P_v DMMA GEMMs of the CG loop (RHS projection excluded from the flop count)"},
        "kernel_ms_per_step": {k: round(v["ms"] / a.steps, 3) for k, v in prof.items() if v["spans"]},
        "phase_ms_last_step": {"rhs": stats["ms_rhs"], "cg": stats["ms_cg"], "dn": stats["ms_dn"]},
        "device_gb": w.device_bytes() / 1e9,
    }
    if world == 1 and not a.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(cfg, aux, dV_np[0], alpha)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


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


def aux_ncols(cfg):
    m = cfg["n_max"]
    return sum(1 for x in range(-m, m + 1) for y in range(-m, m + 1) if x * x + y * y <= cfg["n2max"])


# dram__bytes_read.sum + dram__bytes_write.sum of one k2_planes<double,8,9,K2_H> launch of 51 slots under
# `ncu --set full` (profiles/r01_k2_planes_full_details_v6.txt): 52.66 MB + 0.84 MB -> bytes per slot
NCU_K2_DRAM_BYTES_PER_SLOT_CFG2 = (52.657920e6 + 0.844032e6) / 51.0


def measure_fp64_peak():
    """The box's own FP64 yardstick: cuBLAS DGEMM 8192^3 through torch, best of 5, TFLOP/s."""
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
    return 2.0 * n ** 3 / (best * 1e-3) / 1e12


def roofline(cfg, top, prof, n_h, stats, hbm_peak, peak_src, n_cols, mixed, w, fp64_peak):
    """Roofline entry for the kernel class that took the most time (DESIGN.md section 6 states the per-unit figures)."""
    N = cfg["N"]
    gamma = cfg["mode"] == "gamma"
    slots = n_h / (2 if gamma else 1)                       # FFT slots pushed through H*psi in the timed region
    csz = 8 if mixed else 16
    t = prof[top]["ms"] * 1e-3
    spans = max(1, prof[top]["spans"])
    fp64_src = "measured in this run: cuBLAS DGEMM 8192^3 FP64 (DMMA and the FP64 FMA pipe have the same nominal rate on B200, 37.2 TFLOP/s)"
    out = {"kernel": top, "avg_launch_ms": prof[top]["ms"] / spans, "traffic": None}
    if top in ("k1_g2r_z", "k2_planes", "k3_r2g_z"):
        stick = N * n_cols * csz
        sphere = (2 if gamma else 1) * w.n_g * 16
        per_slot = {"k1_g2r_z": sphere + stick, "k2_planes": 2 * stick, "k3_r2g_z": stick + 2 * sphere}[top]
        gbs = per_slot * slots / t / 1e9
        if top == "k2_planes":
            # the plane kernel is bound by FP64 issue / shared memory, not by HBM: nominal 5 N log2 N flops
            # per 1D transform, 2 (nr + N) transforms per plane, plus the V_loc multiply
            nr = 2 * cfg["n_max"] + 1
            fl_slot = N * (2 * (nr + N) * 5.0 * N * np.log2(N) + 2 * N * N)
            ach = fl_slot * slots / t / 1e12
            peak = fp64_peak * (2.0 if mixed else 1.0)
            out.update({"bound": "alu", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
                        "peak_source": fp64_src + ("; x2 for the FP32 path" if mixed else ""),
                        "algorithmic_flops_per_slot": fl_slot, "algorithmic_bytes_per_slot": per_slot,
                        "hbm_view": {"achieved_gbs": gbs, "peak_gbs": hbm_peak, "frac": gbs / hbm_peak, "peak_source": peak_src}})
            # shared-memory view: the four two-stage 1D passes move 8 nr N + 4 N^2 elements per plane through shared
            # memory; peak = 128 B/clk/SM x 148 SMs x the SM clock.  Removing FP64 work from this kernel does not shorten it; this is the
            # more loaded of its two pipes (profiles/r01_k2_pipe_experiments.md)
            smem_slot = N * (8 * nr * N + 4 * N * N) * csz
            smem_peak = 128.0 * 148 * sm_clock_mhz() * 1e6 / 1e9
            smem_gbs = smem_slot * slots / t / 1e9
            out["smem_view"] = {"achieved_gbs": smem_gbs, "peak_gbs": smem_peak, "frac": smem_gbs / smem_peak,
                                "algorithmic_smem_bytes_per_slot": smem_slot,
                                "peak_source": "128 B/clk/SM x 148 SMs x max SM clock (MEASURED_PEAKS.json sm_max_mhz, else 1965 MHz)"}
            if N == 72 and not mixed:
                out["traffic"] = NCU_K2_DRAM_BYTES_PER_SLOT_CFG2 * slots / spans
                out["traffic_note"] = "ncu dram bytes per slot (51-slot capture, cold L2) x slots per launch; algorithmic = %.3e B/slot" % per_slot
        else:
            out.update({"bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak,
                        "peak_source": peak_src, "algorithmic_bytes_per_slot": per_slot})
    elif top in ("gemm_tn", "gemm_update"):
        rows = cfg["n_proj"] + cfg["n_occ"]
        if not gamma:
            rows *= 2
        flops = 2.0 * rows * (2 * w.n_g) * n_h
        ach = flops / t / 1e12
        out.update({"bound": "tensor", "achieved": ach, "peak": fp64_peak, "unit": "TFLOP/s", "frac": ach / fp64_peak,
                    "peak_source": fp64_src})
    else:
        per_col = 10 * 16 * w.n_g
        ach = per_col * n_h / t / 1e9
        out.update({"bound": "hbm", "achieved": ach, "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak, "peak_source": peak_src})
    return out


def run_reference(a, cfg, n_pert):
    """--impl reference: the oracle on the host cores, same metric/unit; needs the GPU only to produce the orbitals."""
    import torch
    w, dV_np, alpha, aux = setup_gpu(cfg, 1, 0, verbose=True)
    res = []
    for _ in range(a.warmup + a.steps):
        res.append(cpu_baseline(cfg, aux, dV_np[0], alpha, budget_s=10.0))
    res = res[a.warmup:]
    v = float(np.mean([r["value"] for r in res]))
    line = {"impl": "reference", "metric": "chi0*dV perturbations/s (batched Sternheimer PCG to tol %.0e)" % TOL, "value": v,
            "unit": "perturbations/s", "n_gpus": a.gpus, "steps": a.steps, "warmup": a.warmup, "ms_per_step": 1e3 / v if v else None,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": a.workload}, "cpu_baseline": dict(res[-1], value=v),
            "e2e": {"value": v, "unit": "perturbations/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


if __name__ == "__main__":
    main()
