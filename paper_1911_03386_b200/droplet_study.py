"""Model 1 ensemble study of the paper's section 3.3 (SURVEY.md section 8(f) NEXT-4 + NEXT-1): M realisations of N
droplets, radii uniform on (0, 1) (eq. (38)), integrated to t = 40; beta_j(t) sampled every `dt_sample`; then the
ensemble moments mu_1, mu_2 (eq. (41)), beta_0 = average of mu_1 over [20, 40] (eq. (42)) and the slope k of mu_2 = k t over
[0, 40] -- the two columns of the paper's Table 2.

    python -m paper_1911_03386_b200.droplet_study [N ...]      # markdown table on stdout

Argument marshalling only: the integration runs in libch's ch_droplet_* kernels, the statistics in ch_stats_*.
"""
from __future__ import annotations

import sys

import numpy as np

from . import binding as B


def initial_radii(M, N, seed=0):
    """eq. (38): one seeded stream per realisation."""
    return np.stack([np.random.default_rng(seed + m).uniform(0.0, 1.0, N) for m in range(M)])


def study(N, M=100, t_end=40.0, dt_sample=0.1, eps=1e-3, rtol=1e-6, atol=1e-9, seed=0):
    """(beta_0, k, series) with series a CUDA tensor [S][M][4] = {F, dF/dt, beta, V} at t = s dt_sample."""
    import torch
    S = int(round(t_end / dt_sample)) + 1
    ctx = B.ch_droplet_create(M, N, eps)
    B.ch_droplet_set_state(ctx, initial_radii(M, N, seed))
    series = torch.zeros((S, M, 4), dtype=torch.float64, device="cuda")
    B.ch_droplet_energy(ctx, series[0])
    for s in range(1, S):
        B.ch_droplet_integrate(ctx, s * dt_sample, rtol, atol)
        B.ch_droplet_energy(ctx, series[s])
    B.ch_droplet_destroy(ctx)
    moments = torch.empty((S, 4), dtype=torch.float64, device="cuda")
    B.ch_stats_moments(series, moments)
    out = torch.empty(3, dtype=torch.float64, device="cuda")
    B.ch_stats_fit(moments, 0.0, dt_sample, 0.5 * t_end, t_end, out)
    beta0 = float(out[0].item())
    B.ch_stats_fit(moments, 0.0, dt_sample, 0.0, t_end, out)
    k = float(out[1].item())
    return beta0, k, series


def main():
    import time
    import torch
    from . import build
    build.build()
    assert torch.cuda.is_available(), "droplet_study needs a CUDA device (no CPU fallback)"
    Ns = [int(a) for a in sys.argv[1:]] or [512, 1024, 2048]
    print("| N | beta_0 = (1/20) int_20^40 mu_1 dt | k (mu_2 = k t over [0, 40]) | seconds |")
    print("|---|---|---|---|")
    for N in Ns:
        t = time.time()
        b0, k, _ = study(N)
        print(f"| {N} | {b0:.4f} | {k:.3e} | {time.time() - t:.1f} |", flush=True)
    return 0


if __name__ == "__main__":
    sys.exit(main())
