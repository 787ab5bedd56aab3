"""Times the kernel classes of west_h_apply on the cfg-2 cell with random vectors (no KB): `python -m paper_2203_05623_b200.time_h_apply`.
A small fixed workload for ncu captures of the FFT kernels (8192 real vectors = 4096 transform slots, chunks of 2048 slots)."""
import torch

import synth

from . import WEST_GAMMA, West


def main(n_vec=8192, reps=5, workload="cfg2", precision=0):
    cfg = synth.get_config(workload)
    w = West(cfg["L"], cfg["n2max"], cfg["N"], WEST_GAMMA)
    g = torch.Generator(device="cuda").manual_seed(1)
    w.set_vloc(torch.randn((cfg["N"],) * 3, dtype=torch.float64, device="cuda", generator=g))
    x = torch.randn((n_vec, w.n_g), dtype=torch.float64, device="cuda", generator=g) + 0j
    y = torch.empty_like(x)
    for _ in range(2):
        w.h_apply(x, y, precision=precision)
    w.set_profile(True)
    for _ in range(reps):
        w.h_apply(x, y, precision=precision)
    p = w.get_profile()
    print({k: round(v["ms"] / reps, 3) for k, v in p.items() if v["spans"]})
    w.close()


if __name__ == "__main__":
    import sys
    if len(sys.argv) > 1 and sys.argv[1] == "cfg5":
        main(n_vec=1024, reps=3, workload="cfg5")
    elif len(sys.argv) > 1 and sys.argv[1] == "mixed":
        main(precision=1)
    else:
        main()
