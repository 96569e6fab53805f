"""x-sweep variants timed side by side (north star: "for N >= 1024 a parallel-cyclic-reduction variant is chosen if it
measures faster").

    python -m paper_1911_03386_b200.sweepstudy            # markdown table on stdout

For every (shape, gamma dt) the same device field is swept along x by ch_sweep (include/ch.h) with option sweep = 0 (chunked
periodic LU, the production sweep) and sweep = 3 (parallel cyclic reduction); CUDA events around `reps` launches on the
context's stream; the x-sweep alone moves 16 B per point.  Argument marshalling only: both sweeps are libch kernels.
"""
from __future__ import annotations

import sys


def time_sweep(B, torch, M, N, sigma, option, reps=20):
    e = B.Ensemble(M, N, 2, sigma / 0.5, 0.5, options={"sweep": option})
    w = torch.randn((M, N, N), dtype=torch.float64, device="cuda")
    for _ in range(3):
        B.ch_sweep(e.ctx, w, 0)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        B.ch_sweep(e.ctx, w, 0)
    e1.record()
    torch.cuda.synchronize()
    e.close()
    return e0.elapsed_time(e1) / reps


def main():
    import torch
    from . import binding as B, build
    build.build()
    assert torch.cuda.is_available(), "sweepstudy needs a CUDA device (no CPU fallback)"
    rows = [(32, 1024, 0.01), (8, 2048, 0.01), (2, 4096, 0.01), (8, 2048, 529.0), (128, 512, 529.0), (128, 512, 0.01)]
    print("| shape | gamma dt | chunked LU ms (GB/s) | PCR ms (GB/s) | PCR / LU |")
    print("|---|---|---|---|---|")
    for M, N, sigma in rows:
        gb = M * N * N * 16 / 1e9
        lu, pcr = time_sweep(B, torch, M, N, sigma, 0), time_sweep(B, torch, M, N, sigma, 3)
        print(f"| {M} x {N}^2 | {sigma:g} | {lu:.4f} ({gb / lu * 1e3:.0f}) | {pcr:.4f} ({gb / pcr * 1e3:.0f}) | {pcr / lu:.2f} |")
    return 0


if __name__ == "__main__":
    sys.exit(main())
