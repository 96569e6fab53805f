"""CPU oracle of Model 1, the discrete droplet-population (mean-field Mullins-Sekerka / LSW) model of the paper
(SURVEY.md section 8(f) NEXT-4).  TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline leg, never by the product path (paper_1911_03386_b200/), and it shares no code with csrc/ch_droplet.cu.

Plain numpy, fp64, one realisation at a time, in the paper's order and notation (P:nnn = PAPER.md line nnn):

    dR_i/dt = H(R_i + eps) (-1/R_i^2 + ubar/R_i)                     eq. (39), P:368-376 (eq. (13), regularised)
    ubar    = sum_i H(R_i) / sum_i H(R_i) R_i                        eq. (14)
    F       = sum_i H(R_i) R_i^2 / 2                                 eq. (31), on the constraint surface
    dF/dt   = - sum_i H(R_i) (1 - ubar R_i)^2 / R_i                  eq. (33)
    beta    = - (t / F) dF/dt                                        eq. (36)
    V       = sum_i H(R_i) R_i^3 / 3                                 the conserved volume

H(s) = 1 for s > 0, else 0.  Time integration: the paper uses Matlab's ODE45, i.e. the explicit
Dormand-Prince 5(4) pair with adaptive steps; the tableau below is the published Dormand-Prince (1980) one.

Readings:
  G21  ODE45's tolerances and step controller are not stated.  Controller used here (the textbook one of Hairer,
       Norsett & Wanner II.4): err = max_i |e_i| / (atol + rtol max(|R_i|, |R_i^new|)); accept iff err <= 1;
       h_new = h min(5, max(0.2, 0.9 err^(-1/5))); defaults rtol = 1e-6, atol = 1e-9.
  G22  F and dF/dt sum over living droplets only (H(R_i)): a dead droplet sits at R_i in [-eps, 0] and has no surface.
  G24  The mobility of eq. (34) is printed as m = H(R) R^3; eq. (13) and eq. (33) require m = H(R) R^-3
       (dR/dt = -m dF/dR with dF/dR = R - ubar R^2).  Nothing here uses m: eq. (33) is implemented as printed.
  G23  Between -eps < R_i <= 0 the regularised right-hand side keeps its sign (both terms negative) and carries the droplet
       to R_i <= -eps, where it stops; R_i = 0 exactly (measure zero) is treated as dead (right-hand side 0).
"""
from __future__ import annotations

import numpy as np

# Dormand-Prince 5(4): nodes c, matrix a, 5th-order weights b (= last row of a: FSAL), embedded 4th-order weights bh
C = np.array([0.0, 1 / 5, 3 / 10, 4 / 5, 8 / 9, 1.0, 1.0])
A = [
    [],
    [1 / 5],
    [3 / 40, 9 / 40],
    [44 / 45, -56 / 15, 32 / 9],
    [19372 / 6561, -25360 / 2187, 64448 / 6561, -212 / 729],
    [9017 / 3168, -355 / 33, 46732 / 5247, 49 / 176, -5103 / 18656],
    [35 / 384, 0.0, 500 / 1113, 125 / 192, -2187 / 6784, 11 / 84],
]
B5 = np.array([35 / 384, 0.0, 500 / 1113, 125 / 192, -2187 / 6784, 11 / 84, 0.0])
B4 = np.array([5179 / 57600, 0.0, 7571 / 16695, 393 / 640, -92097 / 339200, 187 / 2100, 1 / 40])


def ubar(R):
    """eq. (14)."""
    alive = R > 0
    den = R[alive].sum()
    return alive.sum() / den if den > 0 else 0.0


def rhs(R, eps):
    """eq. (39)."""
    u = ubar(R)
    out = np.zeros_like(R)
    on = (R + eps > 0) & (R != 0)
    r = R[on]
    out[on] = -1.0 / (r * r) + u / r
    return out


def energy(R, t):
    """(F, dF/dt, beta, V) of eq. (31), (33), (36) and the conserved volume."""
    alive = R > 0
    r = R[alive]
    u = ubar(R)
    F = 0.5 * np.sum(r * r)
    Fd = -np.sum((1.0 - u * r) ** 2 / r)
    beta = -t * Fd / F if F > 0 else 0.0
    return np.array([F, Fd, beta, np.sum(r ** 3) / 3.0])


def dopri5_step(f, y, h, k1=None):
    """One Dormand-Prince step: returns (y5, e, k7) -- the 5th-order solution, the difference to the embedded 4th-order
    one, and the last stage (the first stage of the next step, FSAL)."""
    k = [f(y) if k1 is None else k1]
    for s in range(1, 7):
        ys = y.copy()
        for j, a in enumerate(A[s]):
            if a != 0.0:
                ys = ys + h * a * k[j]
        k.append(f(ys))
    y5 = y.copy()
    e = np.zeros_like(y)
    for j in range(7):
        if B5[j] != 0.0:
            y5 = y5 + h * B5[j] * k[j]
        if B5[j] - B4[j] != 0.0:
            e = e + h * (B5[j] - B4[j]) * k[j]
    return y5, e, k[6]


def integrate(R0, t_end, eps=1e-3, rtol=1e-6, atol=1e-9, h0=1e-4, t0=0.0, max_steps=10_000_000, record=False):
    """Adaptive integration of eq. (39) from t0 to t_end (controller: reading G21).  Returns (R, steps) with steps the
    list of ACCEPTED step sizes (the fixed sequence the CUDA path replays in the parity test); with record=True also
    the list of (t, F, dF/dt, beta, V) after every accepted step."""
    f = lambda y: rhs(y, eps)
    R, t, h = np.array(R0, dtype=np.float64), float(t0), float(h0)
    steps, rec = [], []
    k1 = f(R)
    n = 0
    while t < t_end and n < max_steps:
        n += 1
        h = min(h, t_end - t)
        Rn, e, k7 = dopri5_step(f, R, h, k1)
        err = np.max(np.abs(e) / (atol + rtol * np.maximum(np.abs(R), np.abs(Rn))))
        if err <= 1.0:
            t += h
            R, k1 = Rn, k7
            steps.append(h)
            if record:
                rec.append(np.concatenate(([t], energy(R, t))))
        h *= min(5.0, max(0.2, 0.9 * err ** -0.2)) if err > 0 else 5.0
    return (R, np.array(steps), np.array(rec)) if record else (R, np.array(steps))


def replay(R0, steps, eps=1e-3):
    """Advance by a given sequence of step sizes (no error control): what the fixed-sequence parity test compares."""
    f = lambda y: rhs(y, eps)
    R = np.array(R0, dtype=np.float64)
    k1 = f(R)
    for h in steps:
        R, _, k1 = dopri5_step(f, R, float(h), k1)
    return R


def run_series(R0, sample_dt, nsamples, eps=1e-3, rtol=1e-6, atol=1e-9, h0=1e-4):
    """[nsamples][5] = (t, F, dF/dt, beta, V) at t = k sample_dt, k = 0 .. nsamples - 1: one integrate() call per sample
    interval, each restarted with the step size h0 (the last step of an interval is clipped to land on the sample time)."""
    R = np.array(R0, dtype=np.float64)
    out = [np.concatenate(([0.0], energy(R, 0.0)))]
    for k in range(1, nsamples):
        R, _ = integrate(R, k * sample_dt, eps, rtol, atol, h0, t0=(k - 1) * sample_dt)
        out.append(np.concatenate(([k * sample_dt], energy(R, k * sample_dt))))
    return R, np.array(out)
