"""GPU-vs-oracle parity of Model 1, the droplet-population ensembles, through the C ABI.

Bar: with the oracle's own accepted step sequence replayed on the GPU every living radius agrees to
2e-8: only the summation order of ubar and FMA contraction differ (1e-16 per step), but the right-hand side is
DISCONTINUOUS at a droplet's death (H(R_i) switches ubar by O(1/N)) and a dying droplet moves at speed 1/R^2, so round-off
can register a death one step (h ~ 1e-7) earlier or later, which shifts every other radius by ~h/N ... 1e-9 (measured:
1e-11 when no death is near a step boundary, 1.1e-9 otherwise).  GPU-adaptive vs oracle-adaptive agree to the integration
tolerance; F, dF/dt, beta, V of the same state agree to 1e-12 relative.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_1911_03386_b200 import binding, build
    build.build()
    return binding


@pytest.fixture(scope="module")
def d():
    from oracle import droplet_oracle
    return droplet_oracle


def initial_radii(M, N, seed):
    """eq. (38): radii uniform on (0, 1); one seeded stream per realisation."""
    return np.stack([np.random.default_rng(seed + m).uniform(0, 1, N) for m in range(M)])


@pytest.mark.parametrize("M,N,t_end", [(3, 128, 0.3), (2, 300, 0.1), (1, 1024, 0.02), (4, 37, 1.0)])
def test_replay_of_the_oracle_step_sequence(B, d, M, N, t_end):
    import torch
    R0 = initial_radii(M, N, 10)
    runs = [d.integrate(R0[m], t_end) for m in range(M)]
    L = max(len(st) for _, st in runs)
    steps = np.zeros((M, L))
    for m, (_, st) in enumerate(runs):
        steps[m, :len(st)] = st                                  # rows padded with zeros: they end early
    ctx = B.ch_droplet_create(M, N, 1e-3)
    B.ch_droplet_set_state(ctx, R0)
    B.ch_droplet_replay(ctx, torch.from_numpy(steps).cuda())
    R, E = np.empty((M, N)), np.empty((M, 4))
    B.ch_droplet_get_state(ctx, R)
    B.ch_droplet_energy(ctx, E)
    B.ch_droplet_destroy(ctx)
    for m, (Ro, st) in enumerate(runs):
        alive = Ro > 0
        assert ((R[m] > 0) == alive).all()                       # the same droplets have died
        assert np.abs(R[m][alive] - Ro[alive]).max() <= 2e-8
        # a dying droplet crosses [-eps, 0] at speed ~1/eps^2: its resting place amplifies round-off, so only its death is compared
        Eo = d.energy(Ro, st.sum())
        assert np.abs(E[m][[0, 3]] - Eo[[0, 3]]).max() <= 1e-7 * np.abs(Eo[[0, 3]]).max()       # F, V
        # dF/dt (hence beta) is dominated by the smallest living droplet, (1 - ubar R)^2 / R: compare with the oracle's
        # formula evaluated on the GPU's own radii (the energy kernel), and loosely with the oracle's state
        Eg = d.energy(R[m], st.sum())
        assert np.abs(E[m] - Eg).max() <= 1e-12 * np.abs(Eg).max()


def test_energy_kernel(B, d):
    M, N = 5, 777
    R0 = initial_radii(M, N, 3)
    R0[:, ::7] = -1e-3                                            # dead droplets
    R0[0, 5] = 0.0
    ctx = B.ch_droplet_create(M, N, 1e-3)
    B.ch_droplet_set_state(ctx, R0)
    E = np.empty((M, 4))
    B.ch_droplet_energy(ctx, E)
    back = np.empty((M, N))
    B.ch_droplet_get_state(ctx, back)
    B.ch_droplet_destroy(ctx)
    assert np.array_equal(back, R0)
    for m in range(M):
        Eo = d.energy(R0[m], 0.0)
        assert np.abs(E[m] - Eo).max() <= 1e-12 * np.abs(Eo).max()


def test_adaptive_integration_against_the_oracle(B, d):
    """Both sides run their own controller (reading G21).  The accepted step sequences agree until round-off flips a
    decision; states agree to the integration tolerance either way."""
    import torch
    M, N, t_end = 3, 128, 0.5
    R0 = initial_radii(M, N, 77)
    ctx = B.ch_droplet_create(M, N, 1e-3)
    B.ch_droplet_set_state(ctx, R0)
    steps = torch.zeros((M, 200000), dtype=torch.float64, device="cuda")
    ns = torch.zeros(M, dtype=torch.int32, device="cuda")
    B.ch_droplet_integrate(ctx, t_end, steps=steps, nsteps=ns)
    R, E = np.empty((M, N)), np.empty((M, 4))
    B.ch_droplet_get_state(ctx, R)
    B.ch_droplet_energy(ctx, E)
    B.ch_droplet_destroy(ctx)
    ns, steps = ns.cpu().numpy(), steps.cpu().numpy()
    for m in range(M):
        Ro, st = d.integrate(R0[m], t_end)
        assert steps[m, :ns[m]].sum() == pytest.approx(t_end, rel=1e-12)
        assert abs(int(ns[m]) - len(st)) <= 0.02 * len(st)
        assert np.abs(steps[m, :50] - st[:50]).max() <= 1e-9 * st[:50].max()       # identical before round-off can matter
        alive = Ro > 1e-2
        assert np.abs(R[m][alive] - Ro[alive]).max() <= 2e-5
        Eo = d.energy(Ro, t_end)
        assert abs(E[m][0] - Eo[0]) <= 1e-5 * Eo[0] and abs(E[m][3] - Eo[3]) <= 1e-5 * Eo[3]


@pytest.mark.parametrize("N,t1", [(128, 0.01), (1024, 1e-4), (8192, 3e-7)])
def test_paper_ensembles_invariants(B, N, t1):
    """Table 1: M = 100 realisations of N droplets.  Volume conserved to the integration tolerance, energy
    decreasing, beta > 0, bitwise reproducible.  (Every death costs ~180 adaptive steps and deaths are sequential, so
    the horizon shrinks with N: ~100 deaths per realisation at each size.)"""
    import torch
    M = 100
    R0 = initial_radii(M, N, 1000)
    ctx = B.ch_droplet_create(M, N, 1e-3)
    out = []
    for rep in range(2):
        B.ch_droplet_set_state(ctx, R0)
        E = [np.empty((M, 4)) for _ in range(4)]
        B.ch_droplet_energy(ctx, E[0])
        for k, t in enumerate((t1, 2 * t1, 4 * t1)):
            B.ch_droplet_integrate(ctx, t)
            B.ch_droplet_energy(ctx, E[k + 1])
        out.append(np.stack(E))
    B.ch_droplet_destroy(ctx)
    assert np.array_equal(out[0], out[1])
    E = out[0]
    assert (np.diff(E[:, :, 0], axis=0) < 0).all() and (E[1:, :, 1] < 0).all() and (E[1:, :, 2] > 0).all()
    assert np.abs(E[:, :, 3] / E[0, :, 3] - 1).max() <= 1e-5


def test_droplet_errors(B):
    with pytest.raises(B.ChError):
        B.ch_droplet_create(0, 10, 1e-3)
    ctx = B.ch_droplet_create(2, 10, 1e-3)
    with pytest.raises(B.ChError):
        B.ch_droplet_integrate(ctx, 1.0)                           # no state yet
    B.ch_droplet_set_state(ctx, np.full((2, 10), 0.5))
    with pytest.raises(B.ChError):
        B.ch_droplet_integrate(ctx, 1.0, rtol=-1.0)
    B.ch_droplet_integrate(ctx, 1.0)
    R = np.empty((2, 10))
    B.ch_droplet_get_state(ctx, R)
    assert np.abs(R - 0.5).max() <= 1e-12                          # equal droplets are stationary
    B.ch_droplet_destroy(ctx)


def test_ensemble_study_against_the_papers_table_2(B):
    """Section 3.3 / Table 2 (tests/golden/table_2.txt): M = 100 realisations to t = 40, beta sampled every 0.1,
    beta_0 = mean of mu_1 over [20, 40], k = slope of mu_2 = k t -- Model 1 and the ensemble statistics (NEXT-4 + NEXT-1) end to
    end through the C ABI.  beta spikes whenever a droplet dies ((1 - ubar R)^2 / R), so mu_2 depends on how the series is
    sampled, which the paper does not say, and M = 100 leaves ~15 % noise on k: a sanity band, not a parity pin.  Measured
    here: N = 512: beta_0 = 0.299, k = 6.1e-3 (paper 0.24, 7.5e-3); N = 2048: 0.307, 3.9e-3 (paper 0.283, 1.7e-3)."""
    import os
    from paper_1911_03386_b200 import droplet_study
    paper = {int(l.split()[0]): (float(l.split()[1]), float(l.split()[2]))
             for l in open(os.path.join(os.path.dirname(__file__), "golden", "table_2.txt")) if l.strip() and not l.startswith("#")}
    got = {N: droplet_study.study(N)[:2] for N in (512, 2048)}
    for N, (b0, k) in got.items():
        assert 0.2 <= b0 <= 0.4, (N, b0)                           # approaching the LSW value 1/3 from below
        assert paper[N][1] / 3 <= k <= 3 * paper[N][1], (N, k)
    assert got[2048][1] < got[512][1]                              # the variance falls with N (k ~ 1/N)
