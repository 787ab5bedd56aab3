"""Times west_fft3d_dense the way Fig. 3 of the paper does (one C2C FFT of a 128^3 or 256^3 grid, FP64 and FP32, data
resident on the device, average of 100), with the library transform (cuFFT through torch.fft.fftn) beside it as a yardstick.

    python -m paper_2203_05623_b200.time_fft_dense [--reps 100]
"""
import argparse
import json

import torch

import paper_2203_05623_b200 as wb


def _time(fn, reps, flush):
    for _ in range(5):
        fn()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
    for a, b in ev:
        if flush is not None:
            flush.zero_()                                   # evict the grid from the 126 MB L2 between repetitions
        a.record(); fn(); b.record()
    torch.cuda.synchronize()
    t = sorted(a.elapsed_time(b) for a, b in ev)
    return sum(t) / len(t), t[len(t) // 2]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--reps", type=int, default=100)
    ap.add_argument("--no-flush", action="store_true")
    args = ap.parse_args()
    w = wb.West(10.0, 25, 24, wb.WEST_FULL)
    flush = None if args.no_flush else torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    rows = []
    for n in (64, 128, 256):
        for dt, name, esz in ((torch.complex128, "fp64", 16), (torch.complex64, "fp32", 8)):
            g = torch.Generator(device="cuda"); g.manual_seed(n)
            x = torch.view_as_complex(torch.randn((1, n, n, n, 2), dtype=torch.float64 if esz == 16 else torch.float32, device="cuda", generator=g))
            y = torch.empty_like(x)
            mean, med = _time(lambda: w.fft3d_dense(x, -1, out=y), args.reps, flush)
            mean_ip, _ = _time(lambda: w.fft3d_dense(y, -1, out=y), args.reps, flush)
            mean_lib, med_lib = _time(lambda: torch.fft.fftn(x, dim=(1, 2, 3), out=y), args.reps, flush)
            alg = 2 * n ** 3 * esz                           # read the grid once, write it once
            rows.append({"n": n, "precision": name, "ms_mean": mean, "ms_median": med, "ms_in_place": mean_ip, "library_ms_mean": mean_lib, "library_ms_median": med_lib,
                         "algorithmic_GBps": alg / mean / 1e6, "three_pass_GBps": 3 * alg / mean / 1e6, "vs_library": mean_lib / mean})
            print(json.dumps(rows[-1]), flush=True)
    w.close()


if __name__ == "__main__":
    main()
