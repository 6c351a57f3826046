"""Stand-alone 3-D FFT timing, two measurements:

    python -m paper_1111_0716_b200.fft3d_crossover                 # both
    python -m paper_1111_0716_b200.fft3d_crossover --mode batched  # GPU vs GPU, large batches (~1 GiB, nothing stays in L2)
    python -m paper_1111_0716_b200.fft3d_crossover --mode crossover

batched:   the library's fused two-pass transform (exx_fft3d_fused), its generic per-axis transform (exx_fft3d) and, for
           orientation, cuFFT through torch.fft.fftn, per grid size.
crossover: the paper's third intercept offloads an FFT3D call only above a size threshold found by benchmarking once per system
           ("optimal size ... 28^3" on their Fermi box).  This is that measurement here: ONE box per call, host
           transform (numpy's pocketfft on one core, and scipy.fft with every host core) against the library's transform
           INCLUDING the copy of the box from pinned host memory to the device and back, and with the box already resident.
           Prints the smallest N from which the GPU route wins.

One JSON line per size.  numpy/scipy/cuFFT are yardsticks only: nothing on the product path calls them.
"""
import argparse
import json
import os
import time

import numpy as np

FUSED = (16, 32, 40, 48, 64, 72, 80, 96, 128)


def main():
    import torch
    from . import binding as B
    from . import workloads as W
    ap = argparse.ArgumentParser()
    ap.add_argument("--mode", default="both", choices=["both", "batched", "crossover"])
    ap.add_argument("--sizes", type=int, nargs="*", default=[48, 64, 72, 96, 128])
    ap.add_argument("--crossover-sizes", type=int, nargs="*", default=[8, 10, 12, 16, 20, 24, 30, 32, 36, 40, 48, 64, 72, 96, 128])
    ap.add_argument("--reps", type=int, default=5)
    args = ap.parse_args()

    def timed(f, reps=args.reps):
        f()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            f()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    def host_timed(f, reps):
        f()
        best = float("inf")
        for _ in range(reps):
            t0 = time.perf_counter()
            f()
            best = min(best, time.perf_counter() - t0)
        return best * 1e3

    if args.mode in ("both", "batched"):
        for n in args.sizes:
            g = B.Exx((n, n, n), W.cubic(10.0), np.zeros((1, 3)), [1.0], 2.0, nbands=1)
            nb = max(8, min(256, (1 << 31) // (n ** 3 * 16 * 2)))   # ~1 GiB per buffer: larger than L2
            x = torch.randn(nb * n ** 3, dtype=torch.complex128, device="cuda")
            y = torch.empty_like(x)
            tf = timed(lambda: g.fft3d_fused(x, nb, -1, y))
            tg = timed(lambda: g.fft3d(y, nb, -1))
            tc = timed(lambda: torch.fft.fftn(x.view(nb, n, n, n), dim=(1, 2, 3)))
            box = n ** 3 * 16
            print(json.dumps({"mode": "batched", "n": n, "batch": nb, "fused_us_per_box": 1e3 * tf / nb, "generic_us_per_box": 1e3 * tg / nb,
                              "cufft_us_per_box": 1e3 * tc / nb, "fused_GBs_at_64B_per_point": 4 * box * nb / tf / 1e6,
                              "generic_GBs_at_96B_per_point": 6 * box * nb / tg / 1e6}), flush=True)
            g.close()

    if args.mode in ("both", "crossover"):
        import scipy.fft
        cores = os.cpu_count() or 1
        rows = []
        for n in args.crossover_sizes:
            g = B.Exx((n, n, n), W.cubic(10.0), np.zeros((1, 3)), [1.0], 1.0, nbands=1)
            rng = np.random.default_rng(n)
            xh = rng.standard_normal((n, n, n)) + 1j * rng.standard_normal((n, n, n))
            reps = 50 if n <= 48 else 10
            t_np = host_timed(lambda: np.fft.fftn(xh), reps)
            t_sp = host_timed(lambda: scipy.fft.fftn(xh, workers=cores), reps)
            pin_in = torch.from_numpy(xh.reshape(-1).copy()).pin_memory()
            pin_out = torch.empty_like(pin_in).pin_memory()
            xd = torch.empty(n ** 3, dtype=torch.complex128, device="cuda")
            yd = torch.empty_like(xd)
            fused = n in FUSED

            def dev_only():
                if fused:
                    g.fft3d_fused(xd, 1, -1, yd)
                else:
                    g.fft3d(xd, 1, -1)

            def with_copies():
                xd.copy_(pin_in, non_blocking=True)
                dev_only()
                pin_out.copy_(yd if fused else xd, non_blocking=True)

            t_dev = timed(dev_only, reps)
            # the caller waits for the result: synchronise inside the timed call, time on the host clock
            def call_and_wait():
                with_copies()
                torch.cuda.synchronize()
            t_e2e = host_timed(call_and_wait, reps)
            rows.append((n, t_np, t_sp, t_e2e, t_dev))
            print(json.dumps({"mode": "crossover", "n": n, "kernels": "fused two-pass" if fused else "generic per-axis",
                              "host_numpy_1core_ms": t_np, "host_scipy_%dcores_ms" % cores: t_sp, "gpu_with_h2d_d2h_ms": t_e2e,
                              "gpu_resident_ms": t_dev, "box_MB": n ** 3 * 16 / 1e6}), flush=True)
            g.close()

        def first_win(col):
            wins = [r[0] for r in rows if r[3] < r[col]]
            # the crossover is the size from which the GPU route wins for good
            for n in sorted(wins):
                if all(r[3] < r[col] for r in rows if r[0] >= n):
                    return n
            return None
        print(json.dumps({"mode": "crossover", "summary": True, "paper_crossover_n": 28,
                          "crossover_n_vs_numpy_1core": first_win(1), "crossover_n_vs_scipy_%dcores" % cores: first_win(2),
                          "note": "smallest tested N from which one transform incl. H2D + D2H of the box beats the host transform"}), flush=True)


if __name__ == "__main__":
    main()
