"""Grid-doubling self-convergence study of the paper's Appendix A.

For n in `ns` (each twice the one before) the single-droplet initial condition is advanced to time T on the
n x n grid of [0, L]^2 with dt = dt_factor * dx, through the library's h = 1 units (include/ch.h):
gamma' = gamma / dx^2, dt' = dt / dx^2, so gamma' dt' = gamma dt / dx^4 grows from ~1 (n = 64) to ~10^5
(n = 4096) -- the robustness regime of the sweeps.  E_n (eq. A.1) is reduced on the device by
ch_grid_doubling_error.  With dt proportional to dx the error is O(dx^2) + O(dt): log2(E_n / E_2n) falls from 2
towards 1 as n grows (first order in time; measured 1.59, 1.46 at n = 512, 1024).
Argument marshalling only: every step and the reduction run in libch's kernels.
"""
from __future__ import annotations

import math

import numpy as np

from . import binding as B
from . import inputs


BASE_N, BASE_FACTOR = 64, 0.4     # time quantum tau = BASE_FACTOR * L / BASE_N; every run ends at the same multiple of tau


def scaled_parameters(n, L, gamma, T, dt_factor):
    """(gamma', dt', nsteps) in h = 1 units.  dt = dt_factor dx, so the step count must scale exactly with n and with
    1 / dt_factor: the end time is fixed once as round(T / tau) tau, tau = BASE_FACTOR L / BASE_N, and
    nsteps = round(T / tau) * (BASE_FACTOR / dt_factor) * (n / BASE_N).  (Rounding T / dt per grid would leave the coarse
    and the fine field of eq. (A.1) one fine time step apart -- an O(dt) offset of the size of the error being measured.)"""
    dx = L / n
    dt = dt_factor * dx
    mult = (BASE_FACTOR / dt_factor) * (n / BASE_N)
    if abs(mult - round(mult)) < 1e-9 and mult >= 1:
        nsteps = int(round(T / (BASE_FACTOR * L / BASE_N))) * int(round(mult))
    else:
        nsteps = int(round(T / dt))
    return gamma / dx ** 2, dt / dx ** 2, nsteps


def final_state(n, L=2 * math.pi, gamma=0.01, T=10.0, dt_factor=0.1, axes=(1.8, 0.9)):
    """Device tensor [1][n][n]: the relaxing elliptical droplet at time ~T on the n x n grid."""
    import torch
    g, d, nsteps = scaled_parameters(n, L, gamma, T, dt_factor)
    C0 = inputs.droplet_state(n, L, gamma, axes[0], axes[1])
    e = B.Ensemble(1, n, 2, g, d)
    e.set_state(C0)
    e.step(nsteps)
    out = torch.empty((1, n, n), dtype=torch.float64, device="cuda")
    B.ch_get_state(e.ctx, out)
    torch.cuda.synchronize()
    e.close()
    return out


def study(ns, **kw):
    """[(n, E_n, log2(E_{n/2} / E_n) or None)] for n = ns[1:], E_n comparing grid n with grid n/2 (eq. A.1)."""
    import torch
    assert all(b == 2 * a for a, b in zip(ns, ns[1:]))
    states = [final_state(n, **kw) for n in ns]
    E = []
    for coarse, fine in zip(states, states[1:]):
        out = torch.empty(1, dtype=torch.float64, device="cuda")
        B.ch_grid_doubling_error(fine, coarse, out)
        E.append(float(out.item()))
    rows = []
    for k, n in enumerate(ns[1:]):
        rows.append((n, E[k], None if k == 0 else float(np.log2(E[k - 1] / E[k]))))
    return rows
