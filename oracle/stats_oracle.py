"""TEST INFRASTRUCTURE ONLY -- plain numpy fp64 restatement of the paper's ensemble statistics of the
coarsening rate.  Shares no code with the CUDA path; only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline leg may import it.

    moments   eq. (41a,b), P:452-456   mu_1 = (1/M) sum_j beta_j,  mu_p = (1/M) sum_j (beta_j - mu_1)^p, p = 2, 3, 4
    beta0     eq. (42), P:460          (1 / (t2 - t1)) int_{t1}^{t2} mu_1 dt
    slope_k   P:548                    least-squares fit of mu_2(t) to the trend line mu_2 = k t
    hist      Figs 9, 14, 18           histogram of beta over the members at each sample time
    grid_doubling_error  eq. (A.1), P:672-674   (1/|Omega|) sum |mean of the 4 fine values in a coarse cell - coarse value| dx_c^2

Readings (G18-G20): the integral of eq. (42) is the trapezoid rule over the stored
samples inside the window, divided by the time span those samples cover; the trend line goes through the
origin, so k = sum t mu_2 / sum t^2; bins are [lo + b w, lo + (b + 1) w), values outside are dropped.
Pins: tests/test_stats_pins.py.  Parity status: pinned.
"""
import numpy as np


def moments(series):
    """series[S][M][4] -> [S][4] = mu_1 .. mu_4 of column 2 (beta) over the members."""
    beta = np.asarray(series, dtype=np.float64)[:, :, 2]
    M = beta.shape[1]
    out = np.empty((beta.shape[0], 4))
    for s in range(beta.shape[0]):
        mu1 = beta[s].sum() / M
        d = beta[s] - mu1
        out[s] = mu1, (d ** 2).sum() / M, (d ** 3).sum() / M, (d ** 4).sum() / M
    return out


def window(nsamples, t0, dt_sample, t1, t2):
    t = t0 + np.arange(nsamples) * dt_sample
    return t, (t >= t1) & (t <= t2)


def beta0(mom, t0, dt_sample, t1, t2):
    t, sel = window(len(mom), t0, dt_sample, t1, t2)
    ts, m1 = t[sel], mom[sel, 0]
    if len(ts) == 0:
        return 0.0
    if len(ts) == 1:
        return float(m1[0])
    integral = 0.0
    for i in range(1, len(ts)):
        integral += 0.5 * (m1[i] + m1[i - 1]) * (ts[i] - ts[i - 1])
    return integral / (ts[-1] - ts[0])


def slope_k(mom, t0, dt_sample, t1, t2):
    t, sel = window(len(mom), t0, dt_sample, t1, t2)
    ts, m2 = t[sel], mom[sel, 1]
    stt = float((ts * ts).sum())
    return float((ts * m2).sum()) / stt if stt > 0 else 0.0


def hist(series, lo, width, nbins):
    beta = np.asarray(series, dtype=np.float64)[:, :, 2]
    out = np.zeros((beta.shape[0], nbins), dtype=np.int32)
    for s in range(beta.shape[0]):
        for b in beta[s]:
            q = np.floor((b - lo) / width)
            if 0 <= q < nbins:
                out[s, int(q)] += 1
    return out


def grid_doubling_error(fine, coarse):
    """eq. (A.1): fine[M][2n][2n], coarse[M][n][n] -> E[M]; |Omega| = n^2 dx_c^2, so E = sum|.| / n^2."""
    fine, coarse = np.asarray(fine, dtype=np.float64), np.asarray(coarse, dtype=np.float64)
    M, n = coarse.shape[0], coarse.shape[1]
    E = np.zeros(M)
    for m in range(M):
        total = 0.0
        for i in range(n):
            for j in range(n):
                avg = 0.25 * (fine[m, 2 * i, 2 * j] + fine[m, 2 * i, 2 * j + 1] + fine[m, 2 * i + 1, 2 * j] + fine[m, 2 * i + 1, 2 * j + 1])
                total += abs(avg - coarse[m, i, j])
        E[m] = total / (n * n)
    return E
