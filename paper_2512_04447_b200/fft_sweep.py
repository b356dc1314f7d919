"""Second workload: the paper's batched 3-D FFT study (Fig. 4):
time per wave function of the FFT Laplacian as a function of grid size, for a single orbital and for a
batch of 512, on the kernels of rsdft_apply_h (plan without atoms, V_loc = 0: forward FFT, |G|^2/2, inverse
FFT, i.e. two 3-D transforms per orbital).

    python -m paper_2512_04447_b200.fft_sweep [--grids 32,48,...] [--batches 1,512] [--reps 20]

Prints one JSON line per (grid, batch).  Supported lengths: 16*M, M in {1..8, 10, 12, 16} (the paper's sweep
reaches 256^3: use e.g. --grids 160,192,256 --batches 1,64 there, 512 orbitals of 256^3 do not fit)."""
import argparse
import json

import numpy as np


def main():
    import torch
    from . import rsdft, workloads as wl
    ap = argparse.ArgumentParser()
    ap.add_argument("--grids", default="32,48,64,80,96,112,128")
    ap.add_argument("--batches", default="1,512")
    ap.add_argument("--reps", type=int, default=20)
    args = ap.parse_args()
    if not torch.cuda.is_available():
        raise RuntimeError("fft_sweep needs a CUDA device (there is no CPU fallback)")
    rsdft.load()
    for N in [int(x) for x in args.grids.split(",")]:
        ng = N ** 3
        plan = rsdft.rsdft_plan_create((N, N, N), (0.2 * N,) * 3)
        for b in [int(x) for x in args.batches.split(",")]:
            X = wl.orbital_block(ng, range(min(b, 8)), 7, 0, device="cuda")
            if b > X.shape[0]:
                X = X.repeat((b + X.shape[0] - 1) // X.shape[0], 1)[:b].contiguous()
            HX = torch.empty_like(X)
            for _ in range(3):
                rsdft.rsdft_apply_h(plan, X, HX)
            torch.cuda.synchronize()
            e0 = torch.cuda.Event(enable_timing=True)
            e1 = torch.cuda.Event(enable_timing=True)
            reps = args.reps if b == 1 else max(3, args.reps // 4)
            e0.record()
            for _ in range(reps):
                rsdft.rsdft_apply_h(plan, X, HX)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / reps
            flops = 2 * 5.0 * ng * np.log2(ng) * b                   # two transforms, 5 N log2 N each
            print(json.dumps(dict(grid=N, batch=b, ms_per_call=ms, us_per_wavefunction=1e3 * ms / b,
                                  pts_per_s=b * ng / ms * 1e3, nominal_fft_tflops=flops / ms / 1e9,
                                  model_gbs=80.0 * b * ng / ms / 1e6)), flush=True)
            del X, HX
        plan.close()


if __name__ == "__main__":
    main()
