"""Times the cfg-2 chi0*dV step split over n contexts, each on its own CUDA stream and host thread with 64 / n perturbations:
`python -m paper_2203_05623_b200.time_streams [n]`.  An experiment (profiles/r01_k2_pipe_experiments.md): do HBM-bound vector kernels
of one block overlap SM-bound FFT / GEMM kernels of another?  (They do not: every kernel fills all SMs.)"""
import sys
import threading
import time

import torch

import bench
import synth

from . import WEST_FP64


def main(n_ctx=2, n_pert=64, reps=3):
    cfg = synth.get_config("cfg2")
    n_each = n_pert // n_ctx
    streams = [torch.cuda.Stream() for _ in range(n_ctx)]
    ctxs = []
    for k, s in enumerate(streams):
        with torch.cuda.stream(s):
            w, dV_np, alpha, _ = bench.setup_gpu(cfg, n_pert, 0, verbose=False)
            dV = torch.from_numpy(dV_np[k * n_each:(k + 1) * n_each].copy()).cuda()
            dn = torch.empty((1, n_each) + (cfg["N"],) * 3, dtype=torch.float64, device="cuda")
            ctxs.append((w, dV, dn, alpha))
        s.synchronize()

    def work(k, n):
        w, dV, dn, alpha = ctxs[k]
        with torch.cuda.stream(streams[k]):
            for _ in range(n):
                w.chi0_apply(dV, [0.0], solver=0, tol=bench.TOL, max_iter=bench.MAX_ITER, alpha_pv=alpha, precond=1, check_every=1,
                             precision=WEST_FP64, dn=dn)
            streams[k].synchronize()

    def run(n):
        ts = [threading.Thread(target=work, args=(k, n)) for k in range(n_ctx)]
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for t in ts:
            t.start()
        for t in ts:
            t.join()
        torch.cuda.synchronize()
        return (time.perf_counter() - t0) / n

    run(2)
    print("contexts %d: %.1f ms per %d perturbations" % (n_ctx, run(reps) * 1e3, n_pert))
    for w, _, _, _ in ctxs:
        w.close()


if __name__ == "__main__":
    main(int(sys.argv[1]) if len(sys.argv) > 1 else 2)
