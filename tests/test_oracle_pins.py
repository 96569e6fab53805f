"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these re-type the oracle's own formulas: each compares it with an
independent object -- a dense numpy solve, a closed form, an invariant, a
finite-difference of an independently defined quantity, or a worked limit.
Citations: P:nnn = /root/reference/PAPER.md line nnn; Gk = DESIGN.md reading k.
"""
import numpy as np
import pytest

from paper_1911_03386_b200 import inputs

ROW = lambda s: (s, -4 * s, 1 + 6 * s, -4 * s, s)   # rows of A = I + s (delta^2)^2


def circulant(N, s):
    A = np.zeros((N, N))
    for i in range(N):
        for o, v in zip(range(-2, 3), ROW(s)):
            A[i, (i + o) % N] += v
    return A


# ---------------------------------------------------------------- line solve
@pytest.mark.parametrize("N", [8, 16])
@pytest.mark.parametrize("sigma", [0.01, 1.0, 33.0, 529.0])
def test_line_solve_vs_dense_bruteforce(oracle, N, sigma):
    """north_star pin: brute-force dense solve of the cyclic system on 8/16-point lines."""
    rng = np.random.default_rng(N)
    b = rng.standard_normal((5, N))
    ref = np.linalg.solve(circulant(N, sigma), b.T).T
    for dense in (False, True):
        x = oracle.solve_lines(b, sigma, dense=dense)
        assert np.abs(x - ref).max() <= 1e-14 * (1 + 16 * sigma) * np.abs(ref).max()


@pytest.mark.parametrize("N", [8, 13, 64, 100])
@pytest.mark.parametrize("sigma", [0.01, 1.0, 529.0])
def test_line_solve_vs_dft_closed_form(oracle, N, sigma):
    """Textbook circulant: eigenvalues 1 + s (2 - 2cos(2 pi k/N))^2; naive O(N^2) DFT."""
    rng = np.random.default_rng(7)
    b = rng.standard_normal((3, N))
    k = np.arange(N)
    Fm = np.exp(-2j * np.pi * np.outer(k, k) / N)          # naive DFT matrix
    lam = 1 + sigma * (2 - 2 * np.cos(2 * np.pi * k / N)) ** 2
    ref = ((Fm.conj() @ ((Fm @ b.T) / lam[:, None])) / N).real.T
    x = oracle.solve_lines(b, sigma)
    assert np.abs(x - ref).max() <= 1e-14 * (1 + 16 * sigma) * np.abs(ref).max()


@pytest.mark.parametrize("N,sigma", [(16, 0.01), (64, 529.0), (512, 0.01), (512, 2.77e5)])
def test_line_solve_residual_and_constants(oracle, N, sigma):
    """A x = b on the cyclic stencil; constants are preserved (rows of A sum to 1)."""
    rng = np.random.default_rng(3)
    b = rng.standard_normal((4, N))
    x = oracle.solve_lines(b, sigma)
    Ax = sum(v * np.roll(x, -o, axis=1) for o, v in zip(range(-2, 3), ROW(sigma)))
    assert np.abs(Ax - b).max() <= 1e-13 * (1 + 16 * sigma)
    ones = oracle.solve_lines(np.full((1, N), 2.5), sigma)
    assert np.abs(ones - 2.5).max() <= 1e-13 * (1 + 16 * sigma) ** 0.5


# ------------------------------------------------------- linear growth factor
def growth_factor(theta, cbar, gamma, dt):
    """g = 1 - dt S [(3 cbar^2 - 1) + gamma S] / prod_d (1 + gamma dt s_d^2), s_d = 2-2cos(theta_d)."""
    s = 2 - 2 * np.cos(np.asarray(theta, dtype=np.float64))
    S = s.sum()
    return 1 - dt * S * ((3 * cbar ** 2 - 1) + gamma * S) / np.prod(1 + gamma * dt * s ** 2)


@pytest.mark.parametrize("N,modes,cbar,gamma,dt", [
    (16, (3, 1), 0.0, 1.0, 0.01),
    (16, (1, 2), -0.4, 1.0, 0.01),
    (32, (5, 3), 0.3, 0.5, 0.05),
    (16, (2, 7), 0.0, 66.4, 7.97),          # paper regime sigma = 529
    (8, (1, 2, 3), 0.0, 1.0, 0.01),
    (8, (3, 1, 2), -0.4, 2.0, 0.02),
])
def test_linear_growth_factor(oracle, N, modes, cbar, gamma, dt):
    """north_star pin: closed-form discrete growth rate of one small Fourier mode around cbar
    (mixed modes, so the RHS cross terms and every ADI factor are exercised)."""
    D = len(modes)
    eps, nsteps = 1e-7, 10
    theta = 2 * np.pi * np.array(modes) / N
    idx = np.indices((N,) * D)                    # idx[0] is the slowest axis (z or y)
    phase = sum(theta[d] * idx[D - 1 - d] for d in range(D))   # theta[0] <-> x (fastest)
    C0 = (cbar + eps * np.cos(phase))[None]
    C = oracle.step(C0, gamma, dt, nsteps)
    amp = 2 * np.mean((C[0] - cbar) * np.cos(phase))
    g = growth_factor(theta, cbar, gamma, dt)
    # O(eps^2) nonlinear correction bounds the tolerance
    assert abs(amp / eps - g ** nsteps) <= 2e-9 * max(1.0, abs(g) ** nsteps)
    # the mean is untouched and no other mode appears beyond O(eps^2)
    assert abs(C[0].mean() - cbar) <= 1e-14
    assert np.abs(C[0] - cbar - amp * np.cos(phase)).max() <= 50 * eps ** 2 + 1e-15


def test_finite_amplitude_single_mode_step(oracle):
    """One step from C = A cos(theta x) has a closed form at any amplitude:
    C^3 = A^3 (3 cos + cos 3.)/4, and each mode k is an eigenvector of Lap_h (-s_k) and of A_x, A_y."""
    N, m, A, gamma, dt = 32, 3, 0.7, 0.8, 0.02
    th = 2 * np.pi * m / N
    x = np.arange(N)
    C0 = np.tile(A * np.cos(th * x), (N, 1))[None]                  # uniform in y
    s1, s3 = 2 - 2 * np.cos(th), 2 - 2 * np.cos(3 * th)
    d1 = -dt * s1 * ((0.75 * A ** 3 - A) + gamma * s1 * A) / (1 + gamma * dt * s1 ** 2)
    d3 = -dt * s3 * (0.25 * A ** 3) / (1 + gamma * dt * s3 ** 2)
    ref = C0[0] + d1 * np.cos(th * x)[None, :] + d3 * np.cos(3 * th * x)[None, :]
    C1 = oracle.step(C0, gamma, dt, 1)[0]
    assert np.abs(C1 - ref).max() <= 1e-14
    # same mode along y: pins the y-sweep and the y part of the stencil separately
    C1t = oracle.step(np.ascontiguousarray(C0.transpose(0, 2, 1)), gamma, dt, 1)[0]
    assert np.abs(C1t - ref.T).max() <= 1e-14


# ------------------------------------------------ whole step vs dense algebra
def shift_ops(N, D):
    """Dense second-difference operators per axis in the library's index order (x fastest)."""
    I = np.eye(N)
    d2 = np.roll(I, 1, axis=1) - 2 * I + np.roll(I, -1, axis=1)
    ops = []
    for axis in range(D):                          # axis 0 = x = last kron factor
        mats = [I] * D
        mats[D - 1 - axis] = d2
        K = mats[0]
        for Mx in mats[1:]:
            K = np.kron(K, Mx)
        ops.append(K)
    return ops


@pytest.mark.parametrize("N,D,gamma,dt", [(8, 2, 1.0, 0.01), (16, 2, 66.4, 7.97), (8, 3, 1.0, 0.01), (8, 3, 5.0, 0.3)])
def test_step_vs_dense_kronecker(oracle, N, D, gamma, dt):
    """Brute force: assemble P = prod_d (I + gamma dt (d2_d)^2) as one dense N^D x N^D matrix and
    solve P dC = dt Lap mu with numpy; compare with the oracle's per-axis line solves."""
    rng = np.random.default_rng(11)
    C0 = rng.uniform(-1, 1, size=(1,) + (N,) * D)
    ops = shift_ops(N, D)
    lap = sum(ops)
    c = C0.reshape(-1)
    mu = c ** 3 - c - gamma * (lap @ c)
    P = np.eye(N ** D)
    for K in ops:
        P = P @ (np.eye(N ** D) + gamma * dt * (K @ K))
    ref = c + np.linalg.solve(P, dt * (lap @ mu))
    C1 = oracle.step(C0, gamma, dt, 1).reshape(-1)
    scale = np.abs(ref - c).max()
    cond = 1 + 16 * gamma * dt                    # condition number of one factor A_d
    assert np.abs(C1 - ref).max() <= 1e-14 * cond * max(1.0, scale)
    r = oracle.rhs(C0, gamma, dt).reshape(-1)
    assert np.abs(r - dt * (lap @ mu)).max() <= 1e-12 * np.abs(r).max()
    for axis in range(D):
        w = oracle.sweep(r.reshape(C0.shape), gamma * dt, axis).reshape(-1)
        K = ops[axis]
        ref_w = np.linalg.solve(np.eye(N ** D) + gamma * dt * (K @ K), r)
        assert np.abs(w - ref_w).max() <= 1e-14 * cond * np.abs(ref_w).max()


@pytest.mark.parametrize("D,N", [(2, 64), (3, 16)])
def test_literal_north_star_form_equals_delta_form(oracle, D, N):
    """G1/G2: (I+a dxx^2)(I+a dyy^2) C' = C + dt Lap(C^3-C) - 2a dxx dyy C + a^2 dxx^2 dyy^2 C
    (and its three-factor analogue) is the same scheme as P (C'-C) = dt Lap mu."""
    C0 = inputs.initial_state([5], N, D, 0.0, 0.1)
    a = oracle.step(C0, 1.0, 0.01, 200)
    b = oracle.step_literal(C0, 1.0, 0.01, 200)
    assert np.abs(a - b).max() <= 1e-13


# ---------------------------------------------------------------- invariants
def test_mass_conservation_and_monotone_energy(oracle):
    """P:36, P:507 (mass conserved), P:34 (F decreases)."""
    C0 = inputs.initial_state([0, 1], 64, 2, [0.0, -0.4], 0.1)
    C, series = oracle.run(C0, 1.0, 0.01, 3000, 1)
    mass = series[:, :, 3]
    assert np.abs(mass - mass[0]).max() <= 1e-11
    assert np.abs(C.reshape(2, -1).sum(1) - C0.reshape(2, -1).sum(1)).max() <= 1e-11
    F = series[:, :, 0]
    assert (np.diff(F, axis=0) < 0).all()
    assert (series[:, :, 1] < 0).all()
    assert (series[1:, :, 2] > 0).all() and (series[0, :, 2] == 0).all()


def test_dissipation_matches_centred_difference_of_energy(oracle):
    """Pins the 1/4 prefactor (G3) and the normalisation/sign of dF/dt (G4, G5):
    (F^{n+1} - F^{n-1}) / (2 dt) ~ Fdot^n; a 1/2 prefactor would be off by ~3x."""
    C0 = inputs.initial_state([2], 64, 2, 0.0, 0.1)
    _, s = oracle.run(C0, 1.0, 0.002, 400, 1)
    F, Fd = s[:, 0, 0], s[:, 0, 1]
    fd = (F[2:] - F[:-2]) / (2 * 0.002)
    rel = np.abs(fd - Fd[1:-1]) / np.abs(Fd[1:-1])
    assert np.median(rel) < 5e-3 and rel.max() < 5e-2


@pytest.mark.parametrize("N,dt,seed", [(16, 0.0005, 5), (24, 0.0005, 6)])
def test_dissipation_matches_centred_difference_of_energy_3d(oracle, N, dt, seed):
    """The same pin in D = 3 (eq. (4), eq. (6)): every axis term of sum_d (mu_{i+e_d} - mu_i)^2 enters
    (F^{n+1} - F^{n-1}) / (2 dt) ~ Fdot^n; dropping one axis is off by about a third."""
    C0 = inputs.initial_state([seed], N, 3, 0.0, 0.1)
    _, s = oracle.run(C0, 1.0, dt, 200, 1)
    F, Fd = s[:, 0, 0], s[:, 0, 1]
    fd = (F[2:] - F[:-2]) / (2 * dt)
    rel = np.abs(fd - Fd[1:-1]) / np.abs(Fd[1:-1])
    assert np.median(rel) < 5e-3 and rel.max() < 5e-2


def _golden_rows(name):
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", name)
    return [ln.split() for ln in open(path) if ln.strip() and not ln.startswith("#")]


@pytest.mark.parametrize("row", _golden_rows("mode_dissipation.txt"), ids=lambda r: "D%sN%s_%s%s%s" % (r[0], r[1], r[2], r[3], r[4]))
def test_single_mode_dissipation_closed_form(oracle, row):
    """Closed form (tests/golden/mode_dissipation.txt, written by make_golden.py with mpmath): for
    C = cbar + eps cos(theta . i), Fdot = -eps^2 K^2 (N^D / 2) sum_d s_d to leading order, each axis with its own s_d
    (distinct), so a dropped / duplicated / swapped axis term in the oracle's dissipation sum fails (beta = -t Fdot / F, eq. (6)
    P:64, is formed from this Fdot: test_run_series_convention)."""
    D, N = int(row[0]), int(row[1])
    m = [int(v) for v in row[2:5]][:D]
    cbar, gamma, eps, Fd_exp = (float(v) for v in row[5:9])
    idx = np.meshgrid(*[np.arange(N)] * D, indexing="ij")          # idx[0] is the slowest axis (z or y), idx[-1] is x
    phase = sum(2 * np.pi * m[d] / N * idx[D - 1 - d] for d in range(D))     # m = (m_x, m_y, m_z)
    C = (cbar + eps * np.cos(phase))[None]
    Fd = oracle.energy(C, gamma)[0, 1]
    # next order: mu has a 3 cbar eps^2 cos^2 term -> relative O(eps) corrections (O(eps^2) when cbar = 0)
    assert abs(Fd - Fd_exp) <= (20 * eps * (abs(cbar) + eps) + 1e-9) * abs(Fd_exp)
    # the oracle must tell the axes apart: permuting the mode numbers changes the closed form unless s_d are permuted too
    if D == 3:
        terms = [float(v) for v in row[9:12]]
        assert len({round(t / Fd_exp, 6) for t in terms}) == 3


def test_energy_of_random_initial_state_closed_form(oracle):
    """E[F(0)]/N^D = (cbar^4 + 2 cbar^2 A^2 + A^4/5 - 2 (cbar^2 + A^2/3) + 1)/4 + gamma D A^2/3
    for C0 = cbar + A U(-1,1) i.i.d. (pins both terms of F and the factor 1/2 gamma)."""
    for D, N, cbar, A, gamma in [(2, 256, 0.0, 0.1, 1.0), (2, 256, -0.4, 0.3, 2.5), (3, 48, 0.2, 0.5, 0.7)]:
        C0 = inputs.initial_state([9], N, D, cbar, A)
        F = oracle.energy(C0, gamma)[0, 0]
        exp = (cbar ** 4 + 2 * cbar ** 2 * A ** 2 + A ** 4 / 5 - 2 * (cbar ** 2 + A ** 2 / 3) + 1) / 4 \
            + gamma * D * A ** 2 / 3
        assert abs(F / N ** D - exp) <= 6 * max(A ** 2, A * abs(cbar)) * (1 + gamma) / np.sqrt(N ** D)
        assert abs(oracle.energy(C0, gamma)[0, 3] / N ** D - cbar) <= 4 * A / np.sqrt(N ** D)


def kink_pair(N, gamma_h):
    x = np.arange(N, dtype=np.float64)
    w = np.sqrt(2 * gamma_h)
    prof = np.where(x < N / 2, np.tanh((x - N / 4) / w), -np.tanh((x - 3 * N / 4) / w))
    return np.tile(prof, (N, 1))[None]


def test_tanh_kink_energy_and_near_stationarity(oracle):
    """north_star pin: the stationary interface of eq.(3) is tanh(x / sqrt(2 gamma)); its energy per
    unit length is (2 sqrt 2 / 3) sqrt(gamma).  h != 1 enters by gamma' = gamma/h^2, dt' = dt/h^2, F = h^D F'."""
    sigma_inf = 2 * np.sqrt(2) / 3
    errs, diss = [], []
    for h, N in [(1.0, 64), (0.5, 128), (0.25, 256)]:
        g = 1.0 / h ** 2
        C0 = kink_pair(N, g)
        e = oracle.energy(C0, g)[0]
        per_kink = e[0] * h ** 2 / (2 * N * h)           # F = h^2 F', two kinks of length N h
        errs.append(abs(per_kink - sigma_inf))
        diss.append(-e[1] / (N * h))                      # D = 2: dF/dt = h^(D-2) dF'/dt'
    assert errs[0] < 0.02 and errs[2] < errs[1] < errs[0] and errs[2] < 2e-3
    # dissipation of the sampled continuum kink vanishes as h -> 0 (it is O(h^4))
    assert 0 < diss[2] < diss[1] / 8 and diss[1] < diss[0] / 4 and diss[0] < 0.05
    C0 = kink_pair(64, 1.0)
    C = oracle.step(C0, 1.0, 0.01, 1000)
    assert np.abs(C - C0).max() < 0.05                      # relaxes only to the discrete kink
    assert abs(oracle.energy(C, 1.0)[0, 1]) < 1e-3          # ... which is stationary
    assert np.abs(C - C[:, :1, :]).max() <= 1e-13           # stays uniform in y (y-sweep = identity)
    Ct = oracle.step(np.ascontiguousarray(C0.transpose(0, 2, 1)), 1.0, 0.01, 1000)
    assert np.abs(Ct.transpose(0, 2, 1) - C).max() <= 1e-13


def test_discrete_steady_state_is_fixed_point(oracle):
    """If Lap_h mu = 0 the delta form returns C bit for bit, for any dt."""
    for D in (2, 3):
        C0 = np.full((1,) + (16,) * D, 0.37)
        for dt in (0.01, 10.0):
            assert np.array_equal(oracle.step(C0, 1.0, dt, 3), C0)
    C1 = np.ones((1, 16, 16))
    assert oracle.energy(C1, 1.0, 5.0)[0].tolist() == [0.0, 0.0, 0.0, 256.0]


# -------------------------------------------------------------- equivariances
def test_equivariances(oracle):
    C0 = inputs.initial_state([3, 4], 32, 2, [0.0, -0.3], 0.2)
    base = oracle.step(C0, 1.0, 0.01, 20)
    sh = oracle.step(np.roll(C0, (5, -9), axis=(1, 2)), 1.0, 0.01, 20)
    assert np.abs(np.roll(sh, (-5, 9), axis=(1, 2)) - base).max() <= 1e-13
    assert np.array_equal(oracle.step(-C0, 1.0, 0.01, 20), -base)
    tr = oracle.step(np.ascontiguousarray(C0.transpose(0, 2, 1)), 1.0, 0.01, 20)
    assert np.abs(tr.transpose(0, 2, 1) - base).max() <= 1e-13
    assert np.array_equal(oracle.step(C0[::-1], 1.0, 0.01, 20), base[::-1])
    assert np.array_equal(oracle.step(C0[1:], 1.0, 0.01, 20), base[1:])
    C3 = inputs.initial_state([8], 12, 3, 0.1, 0.2)
    b3 = oracle.step(C3, 1.0, 0.01, 5)
    p3 = oracle.step(np.ascontiguousarray(C3.transpose(0, 3, 1, 2)), 1.0, 0.01, 5)
    assert np.abs(p3.transpose(0, 2, 3, 1) - b3).max() <= 1e-13
    d3 = oracle.step(C3, 1.0, 0.01, 5, dense=True)
    assert np.abs(d3 - b3).max() <= 1e-13


def test_run_series_convention(oracle):
    """G6: sample k is the state after k*stride steps at t = k stride dt (+ t0); beta(0) = 0."""
    C0 = inputs.initial_state([6], 16, 2, 0.0, 0.1)
    Cend, s = oracle.run(C0, 1.0, 0.01, 40, 10)
    assert s.shape == (5, 1, 4)
    mid = oracle.step(C0, 1.0, 0.01, 20)
    e = oracle.energy(mid, 1.0, 20 * 0.01)
    assert np.array_equal(s[2], e)
    assert np.array_equal(Cend, oracle.step(mid, 1.0, 0.01, 20))
    assert s[0, 0, 2] == 0.0 and s[2, 0, 2] == -0.2 * s[2, 0, 1] / s[2, 0, 0]


def test_input_generator_is_order_independent_and_uniform():
    u = inputs.uniform_pm1(42, 200000)
    assert np.array_equal(u[:1000], inputs.uniform_pm1(42, 1000))
    assert -1 <= u.min() and u.max() < 1
    assert abs(u.mean()) < 0.01 and abs(u.var() - 1 / 3) < 0.01
    assert abs(np.corrcoef(u[:-1], u[1:])[0, 1]) < 0.01
    assert not np.array_equal(u[:10], inputs.uniform_pm1(43, 10))


# ------------------------------------------------------------------ golden fixtures (tests/golden/*.txt)
import os

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def golden_rows(name):
    rows = []
    for line in open(os.path.join(GOLDEN, name)):
        if line.strip() and not line.startswith("#"):
            rows.append(line.split())
    return rows


def test_golden_circulant_eigenvalues(oracle):
    """Fourier modes are eigenvectors of the cyclic pentadiagonal matrix: the oracle's solve (banded and dense path)
    must divide mode k by the stored lambda_k = 1 + sigma (2 - 2 cos(2 pi k/N))^2."""
    rows = golden_rows("circulant_eigenvalues.txt")
    assert len(rows) == 3 * 5 + 3 * 9
    for N, sigma, k, lam in rows:
        N, sigma, k, lam = int(N), float(sigma), int(k), float(lam)
        i = np.arange(N)
        b = np.stack([np.cos(2 * np.pi * k * i / N), np.sin(2 * np.pi * k * i / N) + (k == 0)])
        for dense in (False, True):
            v = oracle.solve_lines(b, sigma, dense=dense)
            assert np.abs(v * lam - b).max() <= 1e-13 * lam, (N, sigma, k, dense)


def test_golden_growth_factors(oracle):
    """One oracle step of a small single Fourier mode against the stored closed-form growth factor."""
    for D, N, mx, my, mz, cbar, gamma, dt, g in golden_rows("growth_factors.txt"):
        D, N, ms = int(D), int(N), (int(mx), int(my), int(mz))[: int(D)]
        cbar, gamma, dt, g = float(cbar), float(gamma), float(dt), float(g)
        idx = np.meshgrid(*[np.arange(N)] * D, indexing="ij")            # [z][y][x]: last axis is x
        phase = sum(2 * np.pi * m * ix / N for m, ix in zip(ms, idx[::-1]))
        mode = np.cos(phase)
        eps = 1e-7
        C1 = oracle.step((cbar + eps * mode)[None], gamma, dt, 1)[0]
        got = ((C1 - cbar) * mode).sum() / (eps * (mode * mode).sum())
        assert abs(got - g) <= 2e-7 * max(1.0, abs(g)), (D, N, ms, cbar, got, g)


def test_golden_kink_energy(oracle):
    """Energy per unit length of the sampled tanh interface tends to the stored (2 sqrt 2 / 3) sqrt(gamma) as h -> 0."""
    for gamma, sig in golden_rows("kink_energy.txt"):
        gamma, sig = float(gamma), float(sig)
        errs = []
        for h, N in [(np.sqrt(gamma), 64), (np.sqrt(gamma) / 4, 256)]:
            g = gamma / h ** 2                                          # h = 1 units: gamma' = gamma / h^2
            e = oracle.energy(kink_pair(N, g), g)[0]
            errs.append(abs(e[0] * h ** 2 / (2 * N * h) - sig) / sig)
        assert errs[0] < 0.03 and errs[1] < 2e-3, (gamma, errs)


def test_golden_table_a6_is_self_consistent():
    """The paper's printed Table A.6: the order column equals log2 of the ratio of the printed E_n to within
    their two printed digits, and tends to 1 (first order) -- the property the GPU study is compared with."""
    rows = [(int(n), float(e), float(o)) for n, e, o in golden_rows("table_A6.txt")]
    assert [r[0] for r in rows] == [128, 256, 512, 1024, 2048, 4096]
    for (n, e, o), (_, e2, _) in zip(rows, rows[1:]):
        assert abs(np.log2(e / e2) - o) < 0.06, n
    assert abs(rows[-1][2] - 1.0) < 0.01 and abs(rows[-2][2] - 1.0) < 0.01
