"""Stand-alone batched 3-D FFT timing (S8(f)-3): the library's fused two-pass transform (exx_fft3d_fused), its generic per-axis
transform (exx_fft3d) and, for orientation, cuFFT through torch.fft.fftn, per grid size.

    python -m paper_1111_0716_b200.fft3d_crossover [--sizes 48 64 72 96 128]

The paper benchmarks FFT3D once per system to choose where transforms run (crossover 28^3 on their box);
this is that measurement for this library.  One JSON line per size.  cuFFT is only a yardstick here: nothing on the product path
calls it.
"""
import argparse
import json

import numpy as np


def main():
    import torch
    from . import binding as B
    from . import workloads as W
    ap = argparse.ArgumentParser()
    ap.add_argument("--sizes", type=int, nargs="*", default=[48, 64, 72, 96, 128])
    ap.add_argument("--reps", type=int, default=5)
    args = ap.parse_args()

    def timed(f):
        f()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.reps):
            f()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / args.reps

    for n in args.sizes:
        g = B.Exx((n, n, n), W.cubic(10.0), np.zeros((1, 3)), [1.0], 2.0, nbands=1)
        nb = max(8, min(256, (1 << 31) // (n ** 3 * 16 * 2)))   # ~1 GiB per buffer: larger than L2
        x = torch.randn(nb * n ** 3, dtype=torch.complex128, device="cuda")
        y = torch.empty_like(x)
        tf = timed(lambda: g.fft3d_fused(x, nb, -1, y))
        tg = timed(lambda: g.fft3d(y, nb, -1))
        tc = timed(lambda: torch.fft.fftn(x.view(nb, n, n, n), dim=(1, 2, 3)))
        box = n ** 3 * 16
        print(json.dumps({"n": n, "batch": nb, "fused_us_per_box": 1e3 * tf / nb, "generic_us_per_box": 1e3 * tg / nb,
                          "cufft_us_per_box": 1e3 * tc / nb, "fused_GBs_at_64B_per_point": 4 * box * nb / tf / 1e6,
                          "generic_GBs_at_96B_per_point": 6 * box * nb / tg / 1e6}))
        g.close()


if __name__ == "__main__":
    main()
