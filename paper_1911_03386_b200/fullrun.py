"""A BASELINE.json config run to its full length (the step counts the configs state: 5000 ... 20000 steps), from and to host
memory, with the invariants that hold at any size checked on the result.

    python -m paper_1911_03386_b200.fullrun cfg3 [cfg1 cfg2 ...]      # one markdown table row per config on stdout

Per config: the synthetic initial ensemble of inputs.CONFIGS -> ch_set_state, per-member series
{F, dF/dt, beta, mass} every `stride` steps -> ch_step(nsteps) -> ch_get_state.  Checked: mass of every member conserved to
round-off over the whole run, F strictly decreasing from sample to sample, everything finite, -1 <= C <= 1 to
within the overshoot of the explicit nonlinear term.  Reported: wall time of the stepping (CUDA events), updates/s, the
ensemble mean of beta over the second half of the run (the paper's quantity; context, not a pin: the paper's
runs are 2pi-periodic boxes at gamma = 0.01, these are h = 1 boxes at gamma = 1).  Argument marshalling only.
"""
from __future__ import annotations

import sys

import numpy as np


def run(name: str) -> dict:
    import torch
    from . import binding as B, inputs
    c = inputs.CONFIGS[name]
    M, N, D, nsteps, stride = c["ensemble"], c["N"], c["D"], c["nsteps"], c["stride"]
    C0 = inputs.config_state(name)
    e = B.Ensemble(M, N, D, c["gamma"], c["dt"])
    mode = B.ch_get_option(e.ctx, "fuse_mode") if D == 2 else -1
    e.set_state(C0)
    e.set_series(stride, nsteps // stride + 1)
    e.step(min(nsteps, 20))                               # warm-up (kept: part of the run)
    torch.cuda.synchronize()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record()
    e.step(nsteps - min(nsteps, 20))
    t1.record()
    torch.cuda.synchronize()
    ms = t0.elapsed_time(t1)
    C, s = e.get_state(), e.series()
    launches = B.ch_launch_count(e.ctx)
    e.close()
    F, mass, beta = s[:, :, 0], s[:, :, 3], s[:, :, 2]
    scale = np.abs(C0).reshape(M, -1).sum(axis=1)
    drift = float((np.abs(mass - mass[0]) / scale).max())
    assert s.shape[0] == nsteps // stride + 1 and np.isfinite(s).all() and np.isfinite(C).all(), name
    assert drift <= 1e-12, (name, drift)
    assert (np.diff(F, axis=0) < 0).all(), name
    assert np.abs(C).max() <= 1.2, (name, np.abs(C).max())
    half = s.shape[0] // 2
    return {"config": name, "fuse_mode": mode, "steps": nsteps, "samples": s.shape[0], "launches": launches,
            "seconds": ms * 1e-3 * nsteps / max(1, nsteps - 20), "updates_per_s": M * N ** D * (nsteps - 20) / (ms * 1e-3),
            "mass_drift": drift, "F0": float(F[0].mean()), "F_end": float(F[-1].mean()),
            "beta_mean_second_half": float(beta[half:].mean()), "beta_std_over_members_at_end": float(beta[-1].std()),
            "max_abs_C": float(np.abs(C).max())}


def main(argv):
    import torch
    from . import build
    build.build()
    assert torch.cuda.is_available(), "fullrun needs a CUDA device (no CPU fallback)"
    names = argv or ["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"]
    print("| config | 2D step (`fuse_mode`) | steps | samples per member | kernel launches | stepping time s | updates/s | max mass drift / sum abs C0 | "
          "mean F: start -> end | mean beta, second half | std of beta over members at the end | max abs C |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|")
    for n in names:
        r = run(n)
        print(f"| {r['config']} | {r['fuse_mode']} | {r['steps']} | {r['samples']} | {r['launches']} | {r['seconds']:.2f} | {r['updates_per_s']:.3e} | "
              f"{r['mass_drift']:.1e} | {r['F0']:.5g} -> {r['F_end']:.5g} | {r['beta_mean_second_half']:.3f} | {r['beta_std_over_members_at_end']:.3f} | "
              f"{r['max_abs_C']:.3f} |", flush=True)


if __name__ == "__main__":
    main(sys.argv[1:])
