"""Pins of oracle/stats_oracle.py (ensemble statistics of beta, eq. (41), (42)) against
closed forms and library routines it does not call."""
import numpy as np
import scipy.stats

from oracle import stats_oracle as so


def series_from_beta(beta):
    s = np.zeros(beta.shape + (4,))
    s[..., 2] = beta
    s[..., 0] = 7.0          # other columns must be ignored
    s[..., 1] = -3.0
    s[..., 3] = 11.0
    return s


def test_moments_of_an_arithmetic_progression_closed_form():
    # beta_j = a + h j, j = 1..M: mu_1 = a + h (M+1)/2, mu_2 = h^2 (M^2-1)/12, mu_3 = 0, mu_4 = h^4 (M^2-1)(3M^2-7)/240
    for M, a, h in [(5, 0.0, 1.0), (128, 0.28, 0.01), (1024, -1.0, 0.5)]:
        beta = (a + h * np.arange(1, M + 1))[None, :]
        m = so.moments(series_from_beta(beta))[0]
        assert abs(m[0] - (a + h * (M + 1) / 2)) <= 1e-12 * max(1, abs(m[0]))
        assert abs(m[1] - h ** 2 * (M * M - 1) / 12) <= 1e-11 * m[1]
        assert abs(m[2]) <= 1e-9 * m[1] ** 1.5
        assert abs(m[3] - h ** 4 * (M * M - 1) * (3 * M * M - 7) / 240) <= 1e-11 * m[3]


def test_moments_against_scipy_and_two_point_distribution():
    rng = np.random.default_rng(3)
    beta = rng.normal(0.3, 0.05, size=(7, 300)) + np.linspace(0, 1, 7)[:, None]
    m = so.moments(series_from_beta(beta))
    assert np.allclose(m[:, 0], beta.mean(axis=1), rtol=1e-13)
    for p in (2, 3, 4):
        assert np.allclose(m[:, p - 1], scipy.stats.moment(beta, p, axis=1), rtol=1e-10, atol=1e-18)
    # M/2 members at +d, M/2 at -d around c: mu_1 = c, mu_2 = d^2, mu_3 = 0, mu_4 = d^4; a dropped "- mu_1" fails
    two = np.array([[0.5 + 0.1] * 10 + [0.5 - 0.1] * 10])
    assert np.allclose(so.moments(series_from_beta(two))[0], [0.5, 0.01, 0.0, 1e-4], atol=1e-15)


def test_beta0_is_exact_for_linear_mu1_and_respects_the_window():
    S, t0, dts = 101, 0.0, 0.5                       # samples at t = 0, 0.5, ..., 50
    t = t0 + dts * np.arange(S)
    mom = np.zeros((S, 4))
    mom[:, 0] = 0.28 + 0.002 * t                     # trapezoid is exact: average = value at the window centre
    assert abs(so.beta0(mom, t0, dts, 20.0, 40.0) - (0.28 + 0.002 * 30.0)) <= 1e-14
    mom[t < 20, 0] = 99.0                            # outside the window: must not matter
    mom[t > 40, 0] = -99.0
    assert abs(so.beta0(mom, t0, dts, 20.0, 40.0) - 0.34) <= 1e-14
    # quadratic mu_1: trapezoid error h^2/12 * f'' exactly
    mom[:, 0] = t * t
    exact = (40.0 ** 3 - 20.0 ** 3) / 3 / 20.0
    assert abs(so.beta0(mom, t0, dts, 20.0, 40.0) - (exact + dts ** 2 / 12 * 2)) <= 1e-10
    # window endpoints between samples: only samples inside count, average over the span they cover
    mom[:, 0] = 1.0 + t
    assert abs(so.beta0(mom, t0, dts, 20.2, 39.9) - (1.0 + 0.5 * (20.5 + 39.5))) <= 1e-13


def test_slope_k_recovers_a_line_through_the_origin_and_matches_lstsq():
    S, t0, dts = 81, 10.0, 1.25
    t = t0 + dts * np.arange(S)
    mom = np.zeros((S, 4))
    mom[:, 1] = 0.0056 * t
    assert abs(so.slope_k(mom, t0, dts, 20.0, 100.0) - 0.0056) <= 1e-16
    rng = np.random.default_rng(5)
    mom[:, 1] = 0.0013 * t + 1e-3 * rng.standard_normal(S)
    sel = (t >= 20) & (t <= 100)
    ref = np.linalg.lstsq(t[sel, None], mom[sel, 1], rcond=None)[0][0]
    assert abs(so.slope_k(mom, t0, dts, 20.0, 100.0) - ref) <= 1e-13


def test_hist_against_numpy_histogram_and_edges():
    rng = np.random.default_rng(9)
    beta = rng.normal(0.3, 0.2, size=(4, 500))
    lo, width, nbins = -0.2, 0.05, 20
    h = so.hist(series_from_beta(beta), lo, width, nbins)
    edges = lo + width * np.arange(nbins + 1)
    for s in range(4):
        inside = beta[s][(beta[s] >= edges[0]) & (beta[s] < edges[-1])]
        assert np.array_equal(h[s], np.histogram(inside, bins=edges)[0])
        assert h[s].sum() == len(inside)
    # left edge belongs to the bin, right end is open, outside values are dropped
    b = np.array([[0.0, 0.25, 0.5, 0.999999, 1.0, -1e-9]])
    assert so.hist(series_from_beta(b), 0.0, 0.25, 4)[0].tolist() == [1, 1, 1, 1]


def test_grid_doubling_error_closed_forms():
    """eq. (A.1), P:672-674 on cell-centred grids: a linear field has E = 0 (the mean of the four fine
    samples IS the coarse sample); f = x^2 + y^2 has E = h_f^2 / 2 exactly; a constant offset d gives |d|."""
    n, L = 8, 2.0
    hf, hc = L / (2 * n), L / n
    xf, xc = (np.arange(2 * n) + 0.5) * hf, (np.arange(n) + 0.5) * hc
    lin_f = (3.0 * xf[None, :] - 2.0 * xf[:, None] + 0.7)[None]
    lin_c = (3.0 * xc[None, :] - 2.0 * xc[:, None] + 0.7)[None]
    assert so.grid_doubling_error(lin_f, lin_c)[0] <= 1e-15
    q_f = (xf[None, :] ** 2 + xf[:, None] ** 2)[None]
    q_c = (xc[None, :] ** 2 + xc[:, None] ** 2)[None]
    assert abs(so.grid_doubling_error(q_f, q_c)[0] - hf ** 2 / 2) <= 1e-14
    assert abs(so.grid_doubling_error(lin_f, lin_c - 0.25)[0] - 0.25) <= 1e-15
    # transposed operands / wrong 2x2 block fail: an x-only field against its y-only twin
    fx = np.tile(xf[None, :], (2 * n, 1))[None]
    assert so.grid_doubling_error(fx, np.tile(xc[None, :], (n, 1))[None])[0] <= 1e-15
    assert so.grid_doubling_error(fx, np.tile(xc[:, None], (1, n))[None])[0] > 0.1
    # members are independent
    two = so.grid_doubling_error(np.concatenate([lin_f, q_f]), np.concatenate([lin_c, q_c]))
    assert two[0] <= 1e-15 and abs(two[1] - hf ** 2 / 2) <= 1e-14
