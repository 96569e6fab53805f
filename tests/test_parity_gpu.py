"""GPU-vs-oracle parity through the C ABI (the parity tests proper).

Tolerances (BASELINE.json north_star): max-abs field difference <= 1e-10 after 1000
steps; relative error <= 1e-9 on F(t) (and dF/dt, mass), beta compared with relative
1e-9 plus absolute 1e-12 (beta(0) = 0).  Same seeded inputs on both sides.
"""
import numpy as np
import pytest

from paper_1911_03386_b200 import inputs

pytestmark = pytest.mark.gpu

FIELD_TOL = 1e-10
SERIES_RTOL = 1e-9


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_1911_03386_b200 import binding, build
    build.build()
    return binding


def assert_series_close(s, so, rtol=SERIES_RTOL):
    assert s.shape == so.shape
    for q in (0, 1, 3):      # F, dF/dt, mass
        scale = np.maximum(np.abs(so[..., q]), 1e-300)
        # mass of a symmetric mixture is ~0: compare against sum|C| ~ its natural scale
        if q == 3:
            scale = np.maximum(scale, 1.0)
        assert (np.abs(s[..., q] - so[..., q]) / scale).max() <= rtol, f"series column {q}"
    assert (np.abs(s[..., 2] - so[..., 2]) <= rtol * np.abs(so[..., 2]) + 1e-12).all(), "beta"


def run_gpu(B, C0, gamma, dt, nsteps, stride, options=None, t0=0.0):
    M, N, D = C0.shape[0], C0.shape[1], C0.ndim - 1
    e = B.Ensemble(M, N, D, gamma, dt, options=options)
    e.set_state(C0)
    if t0:
        B.ch_set_time(e.ctx, t0)
    e.set_series(stride, nsteps // stride + 1)
    e.step(nsteps)
    C, s = e.get_state(), e.series()
    e.close()
    return C, s


# ------------------------------------------------------------------ per kernel
@pytest.mark.parametrize("N,D,M,gamma,dt", [
    (64, 2, 3, 1.0, 0.01), (512, 2, 2, 1.0, 0.01), (24, 2, 2, 1.0, 0.01), (8, 2, 1, 1.0, 0.01),
    (100, 2, 1, 0.5, 0.02), (32, 3, 2, 1.0, 0.01), (128, 3, 1, 1.0, 0.01), (64, 3, 3, 0.7, 0.02), (20, 3, 1, 1.0, 0.01), (8, 3, 1, 2.0, 0.01),
])
def test_rhs_kernel(B, oracle, N, D, M, gamma, dt):
    C0 = inputs.initial_state(range(50, 50 + M), N, D, -0.2, 0.5)
    e = B.Ensemble(M, N, D, gamma, dt)
    e.set_state(C0)
    r, ro = e.rhs(), oracle.rhs(C0, gamma, dt)
    e.close()
    assert np.abs(r - ro).max() <= 1e-13 * np.abs(ro).max()


@pytest.mark.parametrize("N,D,M", [(16, 2, 2), (64, 2, 3), (256, 2, 2), (512, 2, 2), (1024, 2, 1), (2048, 2, 1),
                                   (24, 2, 2), (8, 2, 1), (100, 2, 1), (32, 3, 2), (128, 3, 1), (20, 3, 1)])
@pytest.mark.parametrize("sigma", [0.01, 1.0, 529.0])
def test_sweep_kernels(B, oracle, N, D, M, sigma):
    """Each axis, chunked (N % 16 == 0) or generic path, against the oracle's banded solve.
    sigma = 529 is the paper's regime (gamma = 0.01, dx = 2 pi/512, dt = 0.0012)."""
    rng = np.random.default_rng(N * 10 + D)
    w = rng.standard_normal((M,) + (N,) * D)
    e = B.Ensemble(M, N, D, sigma / 0.5, 0.5)
    tol = 1e-14 * (1 + 16 * sigma)
    for axis in range(D):
        got, ref = e.sweep(w, axis), oracle.sweep(w, sigma, axis)
        assert np.abs(got - ref).max() <= tol * np.abs(ref).max(), f"axis {axis}"
    if B.ch_get_option(e.ctx, "chunked"):
        for scan in (1, 2):                            # K-term sum / warp-shuffle scan closure of the x-sweep
            B.ch_set_option(e.ctx, "scan", scan)
            got, ref = e.sweep(w, 0), oracle.sweep(w, sigma, 0)
            assert np.abs(got - ref).max() <= tol * np.abs(ref).max(), f"scan {scan}"
        B.ch_set_option(e.ctx, "scan", 0)
        B.ch_set_option(e.ctx, "sweep", 1)             # generic kernels on the same data
        for axis in range(D):
            got, ref = e.sweep(w, axis), oracle.sweep(w, sigma, axis)
            assert np.abs(got - ref).max() <= tol * np.abs(ref).max(), f"generic axis {axis}"
    e.close()


@pytest.mark.parametrize("N,D,M", [(8, 2, 2), (64, 2, 3), (1024, 2, 1), (2048, 2, 1), (4096, 2, 1), (32, 3, 1)])
@pytest.mark.parametrize("sigma", [0.01, 1.0, 529.0])
def test_pcr_x_sweep(B, oracle, N, D, M, sigma):
    """The parallel-cyclic-reduction x-sweep (option sweep = 3; the north star's measured alternative
    for N >= 1024) against the oracle's banded solve, truncated (sigma = 0.01) and full depth."""
    rng = np.random.default_rng(N + D)
    w = rng.standard_normal((M,) + (N,) * D)
    e = B.Ensemble(M, N, D, sigma / 0.5, 0.5, options={"sweep": 3})
    got, ref = e.sweep(w, 0), oracle.sweep(w, sigma, 0)
    e.close()
    assert np.abs(got - ref).max() <= 1e-14 * (1 + 16 * sigma) * np.abs(ref).max()


def test_energy_kernel(B, oracle):
    for N, D in [(64, 2), (512, 2), (24, 2), (32, 3), (20, 3), (64, 3), (128, 3)]:
        C0 = inputs.initial_state([1, 2], N, D, [0.0, -0.4], 0.3)
        e = B.Ensemble(2, N, D, 1.3, 0.01)
        e.set_state(C0)
        got, ref = e.energy(), oracle.energy(C0, 1.3, 0.0)
        e.close()
        assert_series_close(got[None], ref[None], 1e-12)


# ---------------------------------------------------------------- end to end
def test_cfg1_full_parity(B, oracle):
    """configs[0]: 1 member 64^2, every sample of the first 1000 steps and the final field."""
    c = inputs.CONFIGS["cfg1"]
    C0 = inputs.config_state("cfg1")
    C, s = run_gpu(B, C0, c["gamma"], c["dt"], 1000, c["stride"])
    Co, so = oracle.run(C0, c["gamma"], c["dt"], 1000, c["stride"])
    assert s.shape == (101, 1, 4)
    assert np.abs(C - Co).max() <= FIELD_TOL
    assert_series_close(s, so)


def test_cfg1_whole_run(B, oracle):
    """configs[0] in full: 5000 steps, 501 samples."""
    c = inputs.CONFIGS["cfg1"]
    C0 = inputs.config_state("cfg1")
    C, s = run_gpu(B, C0, c["gamma"], c["dt"], c["nsteps"], c["stride"])
    Co, so = oracle.run(C0, c["gamma"], c["dt"], c["nsteps"], c["stride"])
    assert s.shape == (501, 1, 4)
    assert np.abs(C - Co).max() <= FIELD_TOL
    assert_series_close(s, so)


def test_cfg2_all_members_short_and_subset_long(B, oracle):
    c = inputs.CONFIGS["cfg2"]
    C0 = inputs.config_state("cfg2")
    C, s = run_gpu(B, C0, c["gamma"], c["dt"], 1000, c["stride"])
    sub = [0, 31, 63]
    Co, so = oracle.run(C0[sub], c["gamma"], c["dt"], 1000, c["stride"])
    assert np.abs(C[sub] - Co).max() <= FIELD_TOL
    assert_series_close(s[:, sub], so)
    # all 64 members over 100 steps
    C, s = run_gpu(B, C0, c["gamma"], c["dt"], 100, c["stride"])
    Co, so = oracle.run(C0, c["gamma"], c["dt"], 100, c["stride"])
    assert np.abs(C - Co).max() <= FIELD_TOL
    assert_series_close(s, so)


def test_cfg3_headline_config_member_subset(B, oracle):
    """configs[2] at full size (128 x 512^2, the shape bench.py times), 1000 steps;
    members are independent, so the oracle checks the first, the last and one in the middle."""
    c = inputs.CONFIGS["cfg3"]
    C0 = inputs.config_state("cfg3")
    C, s = run_gpu(B, C0, c["gamma"], c["dt"], 1000, c["stride"])
    sub = [0, 77, 127]
    Co, so = oracle.run(C0[sub], c["gamma"], c["dt"], 1000, c["stride"])
    assert np.abs(C[sub] - Co).max() <= FIELD_TOL
    assert_series_close(s[:, sub], so)
    # properties at full size: mass conserved, F decreasing, for every member
    mass, F = s[:, :, 3], s[:, :, 0]
    assert np.abs(mass - mass[0]).max() <= 1e-9 * np.abs(mass[0]).max()
    assert (np.diff(F, axis=0) < 0).all()


def test_cfg4_3d_member_subset(B, oracle):
    """configs[3] at full size (16 x 128^3, the production 3D kernels: z-marching RHS, plane-pair x/y sweeps, fused
    z-sweep); north_star depth: the oracle follows one member of each mixture for 1000 steps (~90 s of host time)."""
    c = inputs.CONFIGS["cfg4"]
    C0 = inputs.config_state("cfg4")
    C, s = run_gpu(B, C0, c["gamma"], c["dt"], 1000, c["stride"])
    sub = [0, 15]
    Co, so = oracle.run(C0[sub], c["gamma"], c["dt"], 1000, c["stride"])
    assert np.abs(C[sub] - Co).max() <= FIELD_TOL
    assert_series_close(s[:, sub], so)


def test_3d_streaming_and_tile_rhs(B, oracle):
    """64^3 (the z-marching RHS kernel, several work units per CTA at M = 12) against the oracle and
    against the tile RHS kernel on the same data."""
    C0 = inputs.initial_state(range(3100, 3112), 64, 3, [0.0, -0.4] * 6, 0.05)
    e = B.Ensemble(12, 64, 3, 1.0, 0.01)
    assert B.ch_get_option(e.ctx, "rhs3_stream") > 0
    e.close()
    C, s = run_gpu(B, C0, 1.0, 0.01, 60, 20)
    Ct, st = run_gpu(B, C0, 1.0, 0.01, 60, 20, options={"rhs3": 1})
    assert np.abs(C - Ct).max() <= 1e-13
    assert_series_close(s, st, 1e-12)
    Cs, ss = run_gpu(B, C0, 1.0, 0.01, 60, 20, options={"sweep3": 1})      # separate x and y sweeps instead of the plane kernel
    assert np.abs(C - Cs).max() <= 1e-13
    assert_series_close(s, ss, 1e-12)
    sub = [0, 5, 11]
    Co, so = oracle.run(C0[sub], 1.0, 0.01, 60, 20)
    assert np.abs(C[sub] - Co).max() <= FIELD_TOL
    assert_series_close(s[:, sub], so)


def test_3d_streaming_rhs_at_96(B, oracle):
    """96^3: not a power of two -- the z-marching RHS kernel (wrap by modulo) with the separate chunked sweeps, several
    units per CTA, against the tile RHS kernel and the oracle (sampling every 10 steps: the DIAG variant too)."""
    C0 = inputs.initial_state(range(3500, 3505), 96, 3, [0.0, -0.4, 0.2, -0.1, 0.3], 0.05)
    e = B.Ensemble(5, 96, 3, 1.0, 0.01)
    assert B.ch_get_option(e.ctx, "rhs3_stream") > 0 and B.ch_get_option(e.ctx, "sweep_xy") == 0
    e.set_state(C0)
    r, ro = e.rhs(), oracle.rhs(C0, 1.0, 0.01)
    e.close()
    assert np.abs(r - ro).max() <= 1e-13 * np.abs(ro).max()
    C, s = run_gpu(B, C0, 1.0, 0.01, 40, 10)
    Ct, st = run_gpu(B, C0, 1.0, 0.01, 40, 10, options={"rhs3": 1})
    assert np.abs(C - Ct).max() <= 1e-13
    assert_series_close(s, st, 1e-12)
    Co, so = oracle.run(C0[[0, 4]], 1.0, 0.01, 40, 10)
    assert np.abs(C[[0, 4]] - Co).max() <= FIELD_TOL
    assert_series_close(s[:, [0, 4]], so)


def test_3d_plane_sweep_paper_regime(B, oracle):
    """x + y sweeps of a z-plane in one kernel at gamma dt = 529 (long closures: shuffle scan in x, K-term sum in y),
    64^3 and 128^3, against the oracle."""
    for N, M, nsteps in ((64, 2, 20), (128, 1, 6)):
        C0 = inputs.initial_state(range(3300, 3300 + M), N, 3, -0.3, 0.1)
        e = B.Ensemble(M, N, 3, 66.4, 7.97)
        assert B.ch_get_option(e.ctx, "sweep_xy") == 1
        e.close()
        Co, so = oracle.run(C0, 66.4, 7.97, nsteps, 2)
        for opts in (None, {"sweep3": 2}):               # N = 128: cluster pair / one CTA per plane
            C, s = run_gpu(B, C0, 66.4, 7.97, nsteps, 2, options=opts)
            assert np.abs(C - Co).max() <= FIELD_TOL, (N, opts)       # measured <= 1.5e-13
            assert_series_close(s, so)


def test_small_3d_1000_steps(B, oracle):
    C0 = inputs.initial_state([3000, 3008], 32, 3, [0.0, -0.4], 0.05)
    C, s = run_gpu(B, C0, 1.0, 0.01, 1000, 50)
    Co, so = oracle.run(C0, 1.0, 0.01, 1000, 50)
    assert np.abs(C - Co).max() <= FIELD_TOL
    assert_series_close(s, so)


def test_cfg5_long_lines_two_members(B, oracle):
    """configs[4] at full size (8 x 2048^2, cluster line kernel of 4 CTAs per line); north_star depth: the oracle
    follows two members for 1000 steps (~3 min of host time, side by side)."""
    c = inputs.CONFIGS["cfg5"]
    C0 = inputs.config_state("cfg5")
    C, s = run_gpu(B, C0, c["gamma"], c["dt"], 1000, c["stride"])
    sub = [2, 5]
    Co, so = oracle.run(C0[sub], c["gamma"], c["dt"], 1000, c["stride"])
    assert np.abs(C[sub] - Co).max() <= FIELD_TOL
    assert_series_close(s[:, sub], so)


def test_4096_lines_cluster_of_eight(B, oracle):
    """The paper's largest grid (n = 4096): cluster line kernel with 8 CTAs per line, sampling through
    the tile RHS kernel; one member, 100 steps sampled every 25, against the oracle (~70 s of host time)."""
    C0 = inputs.initial_state([4242], 4096, 2, -0.2, 0.05)
    e = B.Ensemble(1, 4096, 2, 1.0, 0.01)
    assert B.ch_get_option(e.ctx, "fuse_mode") == 4
    e.close()
    C, s = run_gpu(B, C0, 1.0, 0.01, 100, 25)
    Co, so = oracle.run(C0, 1.0, 0.01, 100, 25)
    assert np.abs(C - Co).max() <= FIELD_TOL
    assert_series_close(s, so)


@pytest.mark.parametrize("name,nsteps", [("cfg4", 300), ("cfg5", 300), ("cfg2", 2000)])
def test_full_size_invariants(B, name, nsteps):
    """Properties that hold at any size, on the full configs in the launch configuration bench.py times:
    mass conserved to round-off and F strictly decreasing for every member, beta finite."""
    c = inputs.CONFIGS[name]
    C0 = inputs.config_state(name)
    C, s = run_gpu(B, C0, c["gamma"], c["dt"], nsteps, c["stride"])
    mass, F = s[:, :, 3], s[:, :, 0]
    scale = np.abs(C0).reshape(C0.shape[0], -1).sum(axis=1)
    assert (np.abs(mass - mass[0]) <= 1e-12 * scale).all()
    assert (np.diff(F, axis=0) < 0).all()
    assert np.isfinite(s).all() and np.isfinite(C).all()
    assert np.abs(C.reshape(C.shape[0], -1).sum(axis=1) - mass[-1]).max() <= 1e-9 * scale.max()


def test_restart_parity_from_developed_state(B, oracle):
    """cbar = -0.4 is still linear at step 1000, so also compare from a coarsening state:
    GPU runs 10000 steps, the state is handed to both sides, compared after 1000 more."""
    C0 = inputs.initial_state([1000, 2000], 128, 2, [0.0, -0.4], 0.05)
    e = B.Ensemble(2, 128, 2, 1.0, 0.01)
    e.set_state(C0)
    e.step(10000)
    Cdev = e.get_state()
    assert np.abs(Cdev).max() > 0.9                       # phase separated
    e.set_state(Cdev)
    B.ch_set_time(e.ctx, 100.0)
    e.set_series(50, 21)
    e.step(1000)
    C, s = e.get_state(), e.series()
    e.close()
    Co, so = oracle.run(Cdev, 1.0, 0.01, 1000, 50, t0=100.0)
    assert np.abs(C - Co).max() <= FIELD_TOL
    assert_series_close(s, so)
    assert (s[:, :, 2] > 0.01).all()                      # beta is O(0.1) here, not ~0


def test_paper_regime_large_sigma(B, oracle):
    """sigma = gamma dt = 529 (the paper's gamma = 0.01, dx = 2 pi/512, dt = 0.0012 in h = 1 units):
    correction tables do not decay, cond(A) = 8.5e3 per factor."""
    C0 = inputs.initial_state([7, 8], 128, 2, [0.0, -0.4], 0.05)
    C, s = run_gpu(B, C0, 66.4, 7.97, 200, 10)
    Co, so = oracle.run(C0, 66.4, 7.97, 200, 10)
    # two oracle formulations (banded + Schur vs dense pivoted) differ by 5.6e-12 after these 200
    # steps at 64^2, the GPU differs from the oracle by 5.8e-12: the north star's bar holds at cond(A) = 8.5e3 too
    assert np.abs(C - Co).max() <= FIELD_TOL
    assert_series_close(s, so)


@pytest.mark.parametrize("N,M", [(512, 2), (1024, 1), (2048, 1), (4096, 1)])
def test_sweeps_at_the_convergence_study_extreme(B, oracle, N, M):
    """gamma dt / dx^4 = 2.77e5 (Appendix A at n = 4096; cond(A) = 4.4e6 per factor): every sweep variant the
    grid-doubling study runs (chunked LU with the two-level scan closure, K-term sum, generic) against the oracle's
    banded solve.  Measured 2.3e-11 relative = 0.05 cond(A) eps; bar = 0.5 cond(A) eps."""
    sigma = 2.77e5
    rng = np.random.default_rng(N)
    w = rng.standard_normal((M, N, N))
    tol = 0.5 * (1 + 16 * sigma) * 2.0 ** -53
    e = B.Ensemble(M, N, 2, sigma / 0.5, 0.5)
    ref = [oracle.sweep(w, sigma, axis) for axis in (0, 1)]
    for opts in ({}, {"scan": 1}, {"scan": 2}, {"sweep": 1}):
        for k, v in {"scan": 0, "sweep": 0, **opts}.items():
            B.ch_set_option(e.ctx, k, v)
        for axis in (0, 1):
            got = e.sweep(w, axis)
            assert np.abs(got - ref[axis]).max() <= tol * np.abs(ref[axis]).max(), (opts, axis)
    e.close()


def test_generic_paths_end_to_end(B, oracle):
    for N, D, opts in [(24, 2, None), (64, 2, {"sweep": 1}), (8, 2, None), (12, 3, None), (16, 3, {"sweep": 1})]:
        C0 = inputs.initial_state([11, 12], N, D, [0.0, -0.3], 0.1)
        C, s = run_gpu(B, C0, 1.0, 0.01, 300, 10, options=opts)
        Co, so = oracle.run(C0, 1.0, 0.01, 300, 10)
        assert np.abs(C - Co).max() <= FIELD_TOL, (N, D)
        assert_series_close(s, so)


@pytest.mark.parametrize("N", [16, 32, 48, 64, 80, 96, 128, 160, 176, 192, 224, 256, 320, 352, 384, 448, 512, 592, 1024])
@pytest.mark.parametrize("gamma,dt", [(1.0, 0.01), (66.4, 7.97)])
def test_fused_and_three_pass_2d_paths(B, oracle, N, gamma, dt):
    """Every 2D step variant against the oracle: the line-fused step (RHS + y-sweep with whole lines
    in one persistent CTA, N in {32, 64, 96, 128, 160, 192, 224, 256, 320, 384, 448, 512}; ragged last column strip, more tiles than
    resident CTAs at M = 40), the cluster-fused step (cluster sizes 1..8) and the three-pass step.
    N = 592 (37 chunks per line) has no legal split and must fall back to three passes by itself."""
    M = 2 if N <= 256 else 1
    nsteps = 100 if N <= 256 else 20
    C0 = inputs.initial_state([5, 6][:M], N, 2, [0.0, -0.4][:M], 0.1)
    Co, so = oracle.run(C0, gamma, dt, nsteps, 10)
    tol, rtol = FIELD_TOL, SERIES_RTOL                      # also at gamma dt = 529
    e = B.Ensemble(M, N, 2, gamma, dt)
    cs, line, mode = B.ch_get_option(e.ctx, "fused"), B.ch_get_option(e.ctx, "line"), B.ch_get_option(e.ctx, "fuse_mode")
    cline, local, res = B.ch_get_option(e.ctx, "cline"), B.ch_get_option(e.ctx, "local"), B.ch_get_option(e.ctx, "resident")
    e.close()
    assert (res != 0) == (N in (32, 64, 96, 128, 256))         # member-resident stepping: one CTA, or a cluster of 2 / 8
    assert (local != 0) == (gamma == 1.0 and N >= 64)          # one-pass local step: small gamma dt only
    assert (cs == 0) == (N == 592)
    assert (line != 0) == (N in (32, 64, 96, 128, 160, 192, 224, 256, 320, 384, 448, 512))
    assert (cline != 0) == (N == 1024)                         # flag kernel at K <= 2, scan kernel in the paper regime
    assert mode == (6 if res and N <= 128 else (3 if line else (4 if cline else (5 if local else (2 if cs else 0)))))
    variants = [{"fuse": 1}] + ([{"fuse": 6}] if res else []) + ([{"fuse": 5}] if local else []) + ([{"fuse": 2}] if cs else []) + ([{"fuse": 3}, {"fuse": 3, "linesync": 1}, {"fuse": 3, "linesync": 1, "scan": 2}, {"fuse": 3, "scan": 1}] if line else []) \
        + ([{"fuse": 4}] if cline else [])
    for opts in variants:
        C, s = run_gpu(B, C0, gamma, dt, nsteps, 10, options=opts)
        assert np.abs(C - Co).max() <= tol, (N, opts)
        assert_series_close(s, so, rtol)


@pytest.mark.parametrize("M,N", [(1, 512), (3, 512), (5, 256), (6, 256), (7, 256), (8, 256), (2, 96), (7, 64), (1, 32), (4, 32),
                                 (6, 32), (11, 32)])
def test_line_kernel_packed_leftover_strips(B, oracle, M, N):
    """Stepping kernels pack the NC % 28 leftover columns of two members (lanes 0-7 / 8-15 of the half-warps), or of
    four members when they are <= 4 columns (N = 256, 32: four lanes each), into one tile; ensembles that are not a
    multiple of the group leave part of the last packed tile idle.  Against the oracle."""
    C0 = inputs.initial_state(range(600, 600 + M), N, 2, -0.25, 0.1)
    nsteps = 30 if N >= 256 else 100
    C, s = run_gpu(B, C0, 1.0, 0.01, nsteps, 10, options={"fuse": 3})
    Co, so = oracle.run(C0, 1.0, 0.01, nsteps, 10)
    assert np.abs(C - Co).max() <= FIELD_TOL
    assert_series_close(s, so)


def test_line_kernel_persistent_tiles(B, oracle):
    """More tiles than resident CTAs (40 members x 10 strips at N = 256): every CTA of the line kernel
    loops over several tiles, prefetching the next one; members 0, 17 and 39 against the oracle and
    all members against the three-pass step."""
    C0 = inputs.initial_state(range(300, 340), 256, 2, -0.3, 0.1)
    C, s = run_gpu(B, C0, 1.0, 0.01, 60, 20, options={"fuse": 3})
    C3, s3 = run_gpu(B, C0, 1.0, 0.01, 60, 20, options={"fuse": 1})
    assert np.abs(C - C3).max() <= 1e-13
    assert_series_close(s, s3, 1e-12)
    sub = [0, 17, 39]
    Co, so = oracle.run(C0[sub], 1.0, 0.01, 60, 20)
    assert np.abs(C[sub] - Co).max() <= FIELD_TOL
    assert_series_close(s[:, sub], so)


# ---------------------------------------------------- invariants and edge cases
def test_determinism_and_member_independence(B):
    C0 = inputs.initial_state(range(2000, 2008), 256, 2, -0.4, 0.05)
    a, sa = run_gpu(B, C0, 1.0, 0.01, 200, 50)
    b, sb = run_gpu(B, C0, 1.0, 0.01, 200, 50)
    assert np.array_equal(a, b) and np.array_equal(sa, sb)            # run to run
    p, sp = run_gpu(B, C0[::-1].copy(), 1.0, 0.01, 200, 50)
    assert np.array_equal(p[::-1], a) and np.array_equal(sp[:, ::-1], sa)   # member position
    one, s1 = run_gpu(B, C0[3:4].copy(), 1.0, 0.01, 200, 50)
    assert np.array_equal(one[0], a[3]) and np.array_equal(s1[:, 0], sa[:, 3])   # ensemble size


@pytest.mark.parametrize("M,N,steps", [(40, 512, 30), (6, 1024, 20), (3, 2048, 10)])
def test_flag_synchronised_kernels_are_deterministic_and_match_three_pass(B, M, N, steps):
    """The line kernel (N = 512: more tiles than resident CTAs) and the cluster line kernel (N = 1024, 2048)
    synchronise warps and CTAs with release/acquire flags instead of barriers: repeated runs must agree
    bitwise, and agree with the barrier-synchronised variants and the three-pass step to round-off."""
    C0 = inputs.initial_state(range(500, 500 + M), N, 2, -0.3, 0.1)
    a, sa = run_gpu(B, C0, 1.0, 0.01, steps, 10)
    for _ in range(3):
        b, sb = run_gpu(B, C0, 1.0, 0.01, steps, 10)
        assert np.array_equal(a, b) and np.array_equal(sa, sb)
    ref, sr = run_gpu(B, C0, 1.0, 0.01, steps, 10, options={"fuse": 1})
    assert np.abs(a - ref).max() <= 1e-13
    assert_series_close(sa, sr, 1e-12)
    alt = {"fuse": 3, "linesync": 1} if N == 512 else {"fuse": 2}
    c, sc = run_gpu(B, C0, 1.0, 0.01, steps, 10, options=alt)
    assert np.abs(a - c).max() <= 1e-13
    assert_series_close(sa, sc, 1e-12)


# ------------------------------------- member-resident stepping (one CTA per member; fuse = 6)
@pytest.mark.parametrize("M,N,gamma,dt,nsteps,stride", [
    (3, 32, 1.0, 0.01, 1000, 7), (2, 64, 1.0, 0.01, 1000, 50), (2, 96, 0.5, 0.02, 1000, 100),
    (2, 64, 66.4, 7.97, 200, 10), (1, 96, 66.4, 7.97, 100, 1),         # gamma dt = 529: the full K-term closure
    (2, 128, 1.0, 0.01, 1000, 50), (3, 256, 1.0, 0.01, 1000, 100),     # clusters of 2 and 8 CTAs per member
    (2, 128, 66.4, 7.97, 200, 10), (1, 256, 66.4, 7.97, 100, 5),       # ... with chunk states pulled from every CTA of the cluster
])
def test_resident_stepping_parity(B, oracle, M, N, gamma, dt, nsteps, stride):
    """One launch per ch_step call, the member and its work array in shared memory for all its steps, the samples written
    from inside the kernel: field and series against the oracle at the north star's depth, and bitwise against the same
    job split into calls of 1, 0, n/2 - 1 and the remaining steps (samples at call boundaries are written once)."""
    C0 = inputs.initial_state(range(50, 50 + M), N, 2, -0.2, 0.1)
    e = B.Ensemble(M, N, 2, gamma, dt)
    assert B.ch_get_option(e.ctx, "fuse_mode") == (6 if N <= 128 else 3)      # auto-selected up to N = 128
    e.close()
    opts = {"fuse": 6}
    C, s = run_gpu(B, C0, gamma, dt, nsteps, stride, options=opts)
    Co, so = oracle.run(C0, gamma, dt, nsteps, stride)
    assert np.abs(C - Co).max() <= FIELD_TOL
    assert_series_close(s, so)
    e = B.Ensemble(M, N, 2, gamma, dt, options=opts)
    e.set_state(C0)
    e.set_series(stride, nsteps // stride + 1)
    for k in (1, 0, nsteps // 2 - 1, nsteps - nsteps // 2):
        e.step(k)
    assert B.ch_step_count(e.ctx) == nsteps and B.ch_series_count(e.ctx) == nsteps // stride + 1
    C2, s2 = e.get_state(), e.series()
    with pytest.raises(B.ChError):
        e.step(stride)                                         # the series is full: refused, nothing enqueued
    e.close()
    assert np.array_equal(C, C2) and np.array_equal(s, s2)


def test_resident_stepping_many_members_restart_and_determinism(B, oracle):
    """More members than CTAs fit the device at once (700 x 64^2: three per SM), against the line kernel's step; a member's
    result is bitwise independent of its position and of the ensemble around it; a restart with ch_set_time continues the
    series of one uninterrupted run."""
    C0 = inputs.initial_state(range(4000, 4700), 64, 2, -0.4, 0.05)
    a, sa = run_gpu(B, C0, 1.0, 0.01, 60, 20)
    b, sb = run_gpu(B, C0, 1.0, 0.01, 60, 20, options={"fuse": 3})
    assert np.abs(a - b).max() <= 1e-13
    assert_series_close(sa, sb, 1e-12)
    r, sr = run_gpu(B, C0[::-1].copy(), 1.0, 0.01, 60, 20)
    assert np.array_equal(r[::-1], a) and np.array_equal(sr[:, ::-1], sa)
    one, s1 = run_gpu(B, C0[333:334].copy(), 1.0, 0.01, 60, 20)
    assert np.array_equal(one[0], a[333]) and np.array_equal(s1[:, 0], sa[:, 333])
    sub = [0, 333, 699]
    Co, so = oracle.run(C0[sub], 1.0, 0.01, 60, 20)
    assert np.abs(a[sub] - Co).max() <= FIELD_TOL
    assert_series_close(sa[:, sub], so)
    # restart: 40 steps, then a new context from that state at t0 = 40 dt for the last 20
    h, _ = run_gpu(B, C0[:5].copy(), 1.0, 0.01, 40, 20)
    c, sc = run_gpu(B, h, 1.0, 0.01, 20, 20, t0=40 * 0.01)
    assert np.array_equal(c, a[:5])
    assert_series_close(sc[1:], sa[3:, :5], 1e-14)


@pytest.mark.parametrize("M,N", [(3, 32), (5, 64), (2, 96)])
def test_resident_stepping_one_and_two_lines_per_thread_agree_bitwise(B, M, N):
    """The two one-CTA kernels (one line per thread; two lines per thread, half the shared-memory traffic -- picked when CTAs share
    an SM) do the same arithmetic per point and combine the diagnostics in the same order: fields AND samples are bitwise equal,
    so a member's series does not depend on the ensemble size that selects the kernel."""
    C0 = inputs.initial_state(range(80, 80 + M), N, 2, -0.3, 0.2)
    a, sa = run_gpu(B, C0, 1.0, 0.01, 40, 4, options={"fuse": 6, "resident_lines": 1})
    b, sb = run_gpu(B, C0, 1.0, 0.01, 40, 4, options={"fuse": 6, "resident_lines": 2})
    assert np.array_equal(a, b) and np.array_equal(sa, sb)
    a, sa = run_gpu(B, C0, 66.4, 7.97, 20, 5, options={"fuse": 6, "resident_lines": 1})
    b, sb = run_gpu(B, C0, 66.4, 7.97, 20, 5, options={"fuse": 6, "resident_lines": 2})
    assert np.array_equal(a, b) and np.array_equal(sa, sb)


def test_resident_stepping_cluster_waves(B):
    """157 members of 128^2 on 2-CTA clusters: more clusters than fit the device at once (74), an odd count; against the
    line kernel's step, and bitwise independent of the member order."""
    C0 = inputs.initial_state(range(6000, 6157), 128, 2, -0.4, 0.05)
    a, sa = run_gpu(B, C0, 1.0, 0.01, 30, 10)
    b, sb = run_gpu(B, C0, 1.0, 0.01, 30, 10, options={"fuse": 3})
    assert np.abs(a - b).max() <= 1e-13
    assert_series_close(sa, sb, 1e-12)
    r, sr = run_gpu(B, C0[::-1].copy(), 1.0, 0.01, 30, 10)
    assert np.array_equal(r[::-1], a) and np.array_equal(sr[:, ::-1], sa)


# ------------------------------------- one-pass local step (option fuse = 5)
def reach_bound(sigma, eps=2.0 ** -56):
    """Independent restatement of the host bound (include/ch.h "local_reach"): smallest H with 2 G T(H) / c0 <= eps
    for the causal factor 1 + p z^-1 + q z^-2 of the symbol of A = I + sigma (delta^2)^2 (roots z, conj z inside the
    unit circle, z + 1/z = 2 + i / sqrt(sigma))."""
    w = 2 + 1j / np.sqrt(sigma)
    z = min((w + np.sqrt(w * w - 4)) / 2, (w - np.sqrt(w * w - 4)) / 2, key=abs)
    p, q = -2 * z.real, abs(z) ** 2
    c0 = sigma / q
    h = [1.0, -p]
    while abs(h[-1]) > 1e-40 or len(h) < 16:
        h.append(-p * h[-1] - q * h[-2])
    h = np.abs(np.array(h))
    G, tails = h.sum(), np.cumsum(h[::-1])[::-1]
    return int(np.argmax(2 * G * tails / c0 <= eps))


def test_local_step_is_selected_from_gamma_dt_with_a_host_bound(B):
    """The one-pass step is legal only while the factor recurrences decay within 18 points to below 2^-56 of the data;
    the library computes that reach on the host, picks the step for shapes without a line kernel, and falls back to the
    exact kernels otherwise (sigma = 529 must never take it)."""
    for sigma, legal in [(0.001, True), (0.005, True), (0.01, True), (0.02, False), (1.0, False), (529.0, False)]:
        e = B.Ensemble(1, 500, 2, sigma / 0.5, 0.5)
        H, mode = B.ch_get_option(e.ctx, "local_reach"), B.ch_get_option(e.ctx, "fuse_mode")
        assert (H >= 0) == legal and (mode == 5) == legal, (sigma, H, mode)
        if legal:
            assert H == max(2, reach_bound(sigma)), (sigma, H, reach_bound(sigma))
        else:
            with pytest.raises(B.ChError):
                B.ch_set_option(e.ctx, "fuse", 5)
        e.close()
    for N, want in [(512, 3), (320, 3), (2048, 4), (768, 5), (1000, 5), (352, 5), (100, 5), (24, 0)]:
        e = B.Ensemble(1, N, 2, 1.0, 0.01)
        assert B.ch_get_option(e.ctx, "fuse_mode") == want, N
        e.close()
    e = B.Ensemble(1, 32, 3, 1.0, 0.01)                      # 3D: never
    assert B.ch_get_option(e.ctx, "local") == 0
    e.close()


@pytest.mark.parametrize("name,members,nsteps", [("cfg1", [0], 1000), ("cfg2", [0, 31, 63], 1000), ("cfg3", [0, 77, 127], 1000)])
def test_local_step_parity_1000_steps(B, oracle, name, members, nsteps):
    """north_star bar on the one-pass step: cfg1, cfg2 and cfg3 (full ensembles on the GPU, member subsets on the
    oracle), 1000 steps, field 1e-10, series 1e-9."""
    c = inputs.CONFIGS[name]
    C0 = inputs.config_state(name)
    C, s = run_gpu(B, C0, c["gamma"], c["dt"], nsteps, c["stride"], options={"fuse": 5})
    Co, so = oracle.run(C0[members], c["gamma"], c["dt"], nsteps, c["stride"])
    assert np.abs(C[members] - Co).max() <= FIELD_TOL
    assert_series_close(s[:, members], so)
    mass = s[:, :, 3]
    assert np.abs(mass - mass[0]).max() <= 1e-9 * max(np.abs(mass[0]).max(), 1.0)


@pytest.mark.parametrize("M,N,nsteps,gamma,dt", [
    (3, 100, 300, 1.0, 0.01),        # N % 16 != 0: strips narrower than a CTA, idle warps, tile-kernel sampling
    (2, 68, 200, 1.0, 0.01),         # the C window of a strip wraps around the whole member
    (1, 500, 200, 1.0, 0.01),        # three ragged strips (168, 168, 164 columns)
    (1, 1000, 100, 0.5, 0.01),       # reach 15
    (5, 768, 60, 1.0, 0.01),         # spans that cut strips and members at arbitrary rows
    (2, 1536, 40, 2.0, 0.005),
    (37, 256, 50, 1.0, 0.01),        # more segments than CTAs: several segments per CTA
    (1, 2048, 30, 1.0, 0.001),       # reach 12: different geometry (wider strips)
])
def test_local_step_shapes(B, oracle, M, N, nsteps, gamma, dt):
    C0 = inputs.initial_state(range(900, 900 + M), N, 2, [(-0.4, 0.0, 0.3)[k % 3] for k in range(M)], 0.2)
    C, s = run_gpu(B, C0, gamma, dt, nsteps, 10, options={"fuse": 5})
    sub = sorted({0, M // 2, M - 1})
    Co, so = oracle.run(C0[sub], gamma, dt, nsteps, 10)
    assert np.abs(C[sub] - Co).max() <= FIELD_TOL
    assert_series_close(s[:, sub], so)
    if M > 3:                         # every member against the exact two-kernel / three-pass step
        R, sr = run_gpu(B, C0, gamma, dt, nsteps, 10, options={"fuse": 1})
        assert np.abs(C - R).max() <= 1e-13
        assert_series_close(s, sr, 1e-12)


@pytest.mark.parametrize("M,N,steps", [(128, 512, 12), (9, 1000, 8), (3, 2048, 6), (74, 352, 16)])
def test_local_step_is_deterministic(B, M, N, steps):
    """Warps of the one-pass kernel synchronise through per-warp mbarriers and three CTA barriers per block and drift
    apart in between: 20 repeats, half of them with a second stream keeping the GPU busy, must agree bitwise."""
    import torch
    C0 = torch.from_numpy(inputs.initial_state(range(300, 300 + M), N, 2, -0.3, 0.1)).cuda()
    side, junk = torch.cuda.Stream(), torch.empty(32 << 20, dtype=torch.float32, device="cuda")
    e = B.Ensemble(M, N, 2, 1.0, 0.01, options={"fuse": 5})
    ref = None
    for rep in range(20):
        e.set_state(C0)
        if rep % 2:
            with torch.cuda.stream(side):
                for _ in range(10):
                    junk.mul_(1.0001)
        e.step(steps)
        out = torch.empty_like(C0)
        B.ch_get_state(e.ctx, out)
        torch.cuda.synchronize()
        assert bool(torch.isfinite(out).all())
        if ref is None:
            ref = out
        else:
            assert bool((out == ref).all()), rep
    e.close()


def test_local_step_member_independence_and_graph(B):
    C0 = inputs.initial_state(range(40, 47), 320, 2, -0.2, 0.1)
    a, sa = run_gpu(B, C0, 1.0, 0.01, 64, 16, options={"fuse": 5, "graph": 1})
    g, sg = run_gpu(B, C0, 1.0, 0.01, 64, 16, options={"fuse": 5, "graph": 2})
    assert np.array_equal(a, g) and np.array_equal(sa, sg)             # CUDA graph of 8 ping-pong steps
    # a member's result does not depend on the ensemble around it -- up to the truncation (< 2^-56 of the local max |w|
    # per sweep): where the CTA spans cut the strips depends on the ensemble size, so this is round-off, not bitwise
    one, s1 = run_gpu(B, C0[4:5].copy(), 1.0, 0.01, 64, 16, options={"fuse": 5})
    assert np.abs(one[0] - a[4]).max() <= 1e-15
    assert_series_close(s1[:, :1], sa[:, 4:5], 1e-13)


@pytest.mark.parametrize("M,N,steps", [
    (7, 512, 12), (8, 512, 12), (9, 512, 12), (16, 512, 8), (17, 512, 8), (41, 512, 6),     # 130, 148, 167, 296, 315, 759 tiles on 148 CTAs
    (33, 256, 10), (75, 128, 10),                                                           # two line-kernel CTAs per SM
    (3, 1024, 8), (5, 1024, 6), (2, 2048, 6), (3, 2048, 5), (1, 4096, 4),                    # clusters of 2, 4, 8 CTAs per line
])
def test_flag_synchronised_kernels_repeat_bitwise_under_load(B, M, N, steps):
    """compute-sanitizer is closed on this pool, so the hand-rolled release/acquire protocols of the line kernel
    (per-warp sequence flags, single-buffered slots, packed leftover tiles for odd M) and of the cluster line kernel
    (st.release.cluster / ld.acquire.cluster ghost slots) are exercised instead: 20 repeats per shape -- tile counts
    just below, at and just above multiples of the 148 resident CTAs, odd ensembles -- every other one with a second
    stream keeping the SMs busy so that CTA scheduling and warp drift vary; all must agree bitwise."""
    import torch
    C0 = torch.from_numpy(inputs.initial_state(range(700, 700 + M), N, 2, -0.3, 0.1)).cuda()
    side, junk = torch.cuda.Stream(), torch.empty(32 << 20, dtype=torch.float32, device="cuda")
    e = B.Ensemble(M, N, 2, 1.0, 0.01, options={"fuse": 3} if N <= 128 else None)
    assert B.ch_get_option(e.ctx, "fuse_mode") in (3, 4)
    ser = torch.empty((steps // 2 + 1, M, 4), dtype=torch.float64, device="cuda")
    ref = None
    for rep in range(20):
        e.set_state(C0)
        e.set_series(2, steps // 2 + 1)                     # sampling variants (CTA barriers) interleaved with the flag kernels
        if rep % 2:
            with torch.cuda.stream(side):
                for _ in range(8):
                    junk.mul_(1.0001)
        e.step(steps)
        out = torch.empty_like(C0)
        B.ch_get_state(e.ctx, out)
        ser.copy_(e._series)
        torch.cuda.synchronize()
        if ref is None:
            ref, sref = out, ser.clone()
            assert bool(torch.isfinite(out).all())
        else:
            assert bool((out == ref).all()) and bool((ser == sref).all()), rep
    e.close()


@pytest.mark.parametrize("M,N,D,nsteps,stride,chunk,opts", [
    (12, 256, 2, 37, 10, 5, None),            # uneven chunks (5, 5, 2), line kernel, sampling inside and at the end
    (9, 512, 2, 20, 5, 0, None),              # default chunking
    (5, 1024, 2, 7, 3, 2, None),              # cluster line kernel
    (6, 64, 3, 12, 4, 4, None),               # 3D
    (7, 352, 2, 15, 5, 3, None),              # one-pass local step (auto), odd number of steps: arrays end up swapped
    (3, 24, 2, 9, 3, 1, None),                # generic path
    (11, 64, 2, 23, 5, 4, None),              # member-resident stepping (auto): one launch per chunk
])
def test_run_host_is_set_state_step_get_state(B, M, N, D, nsteps, stride, chunk, opts):
    """ch_run_host (host -> chunk-pipelined H2D / steps / D2H on three streams -> host) against the plain
    ch_set_state + ch_step + ch_get_state job: same final field, same series, same context state afterwards."""
    import torch
    C0 = inputs.initial_state(range(60, 60 + M), N, D, -0.2, 0.2)
    ref, sref = run_gpu(B, C0, 1.0, 0.01, nsteps, stride, options=opts)
    hin = torch.from_numpy(C0.copy()).pin_memory()
    hout = torch.empty_like(hin).pin_memory()
    e = B.Ensemble(M, N, D, 1.0, 0.01, options=opts)
    local = D == 2 and B.ch_get_option(e.ctx, "fuse_mode") == 5
    e.set_series(stride, nsteps // stride + 1)
    B.ch_run_host(e.ctx, hin, hout, nsteps, chunk)
    out, s = hout.numpy().copy(), e.series()
    assert B.ch_step_count(e.ctx) == nsteps and B.ch_series_count(e.ctx) == nsteps // stride + 1
    state_after = e.get_state()
    # the context goes on from there like any other
    e.set_series(stride, 8)
    e.step(2 * stride)
    cont = e.get_state()
    e.close()
    if local:                                   # chunking moves the CTA spans: equal to the truncation, not bitwise
        assert np.abs(out - ref).max() <= 1e-15 and np.abs(s - sref).max() <= 1e-12 * np.abs(sref).max()
    else:
        assert np.array_equal(out, ref) and np.array_equal(s, sref)
    assert np.array_equal(state_after, out)
    ref2, _ = run_gpu(B, out, 1.0, 0.01, 2 * stride, stride, options=opts)
    assert np.abs(cont - ref2).max() <= (1e-15 if local else 0.0)


def test_flag_protocol_invariants_in_the_debug_build(B, tmp_path):
    """libch_debugsync.so (-DCH_DEBUG_SYNC) checks inside the kernels that every warp publishes tile numbers in steps of
    exactly one and that a waiter never finds its neighbour a whole tile ahead (ch_line2d.cuh, ch_cline2d.cuh); a violation
    traps.  The stress shapes run against it in a separate process (the library path is fixed at import) and must finish
    and reproduce the production library's fields bitwise."""
    import os
    import subprocess
    import sys
    from paper_1911_03386_b200 import build
    lib = build.build_debug_sync()
    shapes = [(9, 512, 12), (17, 512, 8), (33, 256, 10), (5, 1024, 6), (3, 2048, 5), (1, 4096, 4)]
    refs = {}
    for M, N, steps in shapes:
        C0 = inputs.initial_state(range(700, 700 + M), N, 2, -0.3, 0.1)
        refs[(M, N)], _ = run_gpu(B, C0, 1.0, 0.01, steps, 2)
        np.save(tmp_path / f"ref_{M}_{N}.npy", refs[(M, N)])
    script = f"""
import sys, numpy as np
sys.path.insert(0, {str(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))!r})
from paper_1911_03386_b200 import binding as B, inputs
assert B._LIBPATH.endswith("libch_debugsync.so")
for M, N, steps in {shapes!r}:
    C0 = inputs.initial_state(range(700, 700 + M), N, 2, -0.3, 0.1)
    for rep in range(3):
        e = B.Ensemble(M, N, 2, 1.0, 0.01)
        assert B.ch_get_option(e.ctx, "fuse_mode") in (3, 4)
        e.set_state(C0); e.set_series(2, steps // 2 + 1); e.step(steps)
        C = e.get_state(); e.close()
        assert np.array_equal(C, np.load({str(tmp_path)!r} + f"/ref_{{M}}_{{N}}.npy")), (M, N, rep)
print("debug build ok")
"""
    r = subprocess.run([sys.executable, "-c", script], env={**os.environ, "CH_LIBCH": lib}, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0 and "debug build ok" in r.stdout, r.stdout[-2000:] + r.stderr[-2000:]


def test_equivariances_on_gpu(B):
    C0 = inputs.initial_state([3, 4], 128, 2, [0.0, -0.3], 0.2)
    base, _ = run_gpu(B, C0, 1.0, 0.01, 50, 50)
    sh, _ = run_gpu(B, np.roll(C0, (37, -70), axis=(1, 2)).copy(), 1.0, 0.01, 50, 50)   # straddles tiles and chunks
    assert np.abs(np.roll(sh, (-37, 70), axis=(1, 2)) - base).max() <= 1e-13
    neg, _ = run_gpu(B, -C0, 1.0, 0.01, 50, 50)
    assert np.array_equal(neg, -base)
    tr, _ = run_gpu(B, np.ascontiguousarray(C0.transpose(0, 2, 1)), 1.0, 0.01, 50, 50)
    assert np.abs(tr.transpose(0, 2, 1) - base).max() <= 1e-13


def test_steady_state_and_split_calls(B, oracle):
    e = B.Ensemble(1, 64, 2, 1.0, 0.01)
    C0 = np.full((1, 64, 64), 0.37)
    e.set_state(C0)
    e.step(5)
    assert np.array_equal(e.get_state(), C0)
    e.close()
    # ch_step(a) + ch_step(b) == ch_step(a + b), series included, also across a sampling step
    C0 = inputs.initial_state([21], 64, 2, 0.0, 0.1)
    whole, sw = run_gpu(B, C0, 1.0, 0.01, 60, 10)
    e = B.Ensemble(1, 64, 2, 1.0, 0.01)
    e.set_state(C0)
    e.set_series(10, 7)
    for k in (0, 7, 3, 10, 25, 15):
        e.step(k)
    assert np.array_equal(e.get_state(), whole) and np.array_equal(e.series(), sw)
    assert B.ch_step_count(e.ctx) == 60 and B.ch_series_count(e.ctx) == 7
    e.close()


@pytest.mark.parametrize("M,N,D", [(1, 64, 2), (3, 256, 2), (2, 32, 3), (1, 64, 3), (2, 24, 2)])
def test_cuda_graph_replay_is_bitwise_the_plain_launches(B, M, N, D):
    """Small ensembles are launch bound: ch_step replays a CUDA graph of 8 plain steps between sampling steps.
    Same field, same series, same launch count as plain launches, also across split calls and odd step counts."""
    C0 = inputs.initial_state(range(90, 90 + M), N, D, -0.2, 0.1)
    out = {}
    for g in (1, 2):
        e = B.Ensemble(M, N, D, 1.0, 0.01, options={"graph": g})
        e.set_state(C0)
        e.set_series(40, 6)
        for k in (37, 1, 90, 16, 33):                    # 177 steps: graphs start at every phase of the stride
            e.step(k)
        out[g] = (e.get_state(), e.series(), B.ch_launch_count(e.ctx))
        e.close()
    assert np.array_equal(out[1][0], out[2][0]) and np.array_equal(out[1][1], out[2][1])
    assert out[1][2] == out[2][2] and out[1][1].shape[0] == 5


def test_errors_and_edge_cases(B):
    e = B.Ensemble(1, 16, 2, 1.0, 0.01)
    with pytest.raises(B.ChError) as ei:
        e.step(1)
    assert ei.value.code == B.CH_ESTATE
    with pytest.raises(B.ChError):
        e.energy()
    C0 = inputs.initial_state([1], 16, 2, 0.0, 0.1)
    e.set_state(C0)
    with pytest.raises(B.ChError) as ei:
        B.ch_step(e.ctx, -1)
    assert ei.value.code == B.CH_EINVAL
    e.set_series(5, 2)
    e.step(5)                                   # samples n = 0 and n = 5: exactly full
    with pytest.raises(B.ChError) as ei:
        e.step(5)                               # would need a third sample
    assert ei.value.code == B.CH_EINVAL and "series full" in str(ei.value)
    assert B.ch_step_count(e.ctx) == 5          # nothing was enqueued
    e.step(4)                                   # no new sample needed
    bad = C0.copy()
    bad[0, 3, 3] = np.nan
    e.set_state(bad)
    with pytest.raises(B.ChError) as ei:
        e.energy()
    assert ei.value.code == B.CH_ENONFINITE
    with pytest.raises(B.ChError):
        B.ch_set_option(e.ctx, "nonsense", 1)
    e.close()


def test_attached_workspace_and_device_pointers(B):
    import torch
    M, N = 4, 64
    C0 = inputs.initial_state(range(M), N, 2, 0.0, 0.1)
    ref, sref = run_gpu(B, C0, 1.0, 0.01, 40, 10)
    ws = torch.empty(B.ch_workspace_bytes(M, N, 2), dtype=torch.uint8, device="cuda")
    stream = torch.cuda.Stream()
    e = B.Ensemble(M, N, 2, 1.0, 0.01, stream=stream.cuda_stream)
    B.ch_attach_workspace(e.ctx, ws)
    with torch.cuda.stream(stream):
        d = torch.from_numpy(C0).cuda()
    stream.synchronize()
    e.set_state(d)
    e.set_series(10, 5)
    e.step(40)
    out = torch.empty_like(d)
    B.ch_get_state(e.ctx, out)
    en = torch.empty((M, 4), dtype=torch.float64, device="cuda")
    B.ch_energy(e.ctx, en)
    stream.synchronize()
    assert np.array_equal(out.cpu().numpy(), ref)
    assert np.array_equal(e.series(), sref)
    assert np.array_equal(en.cpu().numpy(), sref[-1])
    assert B.ch_launch_count(e.ctx) > 0
    e.close()


# ---------------------------------------------------- ensemble statistics
def test_ensemble_statistics_against_the_oracle(B, oracle):
    """eq. (41), (42), P:548 on a real series: 48 members x 128^2 (mixed mixtures), 600 steps sampled every 20;
    moments, window average, slope and histogram against oracle/stats_oracle.py; integer counts bit-exact."""
    import torch
    from oracle import stats_oracle as so
    M, N = 48, 128
    C0 = inputs.initial_state(range(7000, 7000 + M), N, 2, [0.0, -0.4] * (M // 2), 0.05)
    e = B.Ensemble(M, N, 2, 1.0, 0.01)
    e.set_state(C0)
    e.set_series(20, 31)
    e.step(600)
    series = e._series[: B.ch_series_count(e.ctx)].contiguous()
    S = series.shape[0]
    assert S == 31
    mom = torch.empty((S, 4), dtype=torch.float64, device="cuda")
    hist = torch.empty((S, 40), dtype=torch.int32, device="cuda")
    fit = torch.empty(3, dtype=torch.float64, device="cuda")
    B.ch_stats_moments(series, mom)
    B.ch_stats_hist(series, -0.05, 0.0125, 40, hist)
    B.ch_stats_fit(mom, 0.0, 0.2, 2.0, 5.0, fit)
    torch.cuda.synchronize()
    sh = series.cpu().numpy()
    e.close()
    ref = so.moments(sh)
    got = mom.cpu().numpy()
    scale = np.abs(sh[:, :, 2]).max(axis=1)[:, None] ** np.arange(1, 5)[None, :] + 1e-300
    assert (np.abs(got - ref) / scale).max() <= 1e-12
    assert np.array_equal(hist.cpu().numpy(), so.hist(sh, -0.05, 0.0125, 40))
    f = fit.cpu().numpy()
    assert abs(f[0] - so.beta0(ref, 0.0, 0.2, 2.0, 5.0)) <= 1e-12 * max(1e-3, abs(f[0]))
    assert abs(f[1] - so.slope_k(ref, 0.0, 0.2, 2.0, 5.0)) <= 1e-12 * max(1e-6, abs(f[1]))
    assert f[2] == 16


def test_ensemble_statistics_edge_cases(B):
    import torch
    from oracle import stats_oracle as so
    rng = np.random.default_rng(2)
    for S, M in [(1, 1), (3, 2), (5, 1000), (2, 257)]:
        sh = rng.normal(0.3, 0.1, size=(S, M, 4))
        series = torch.from_numpy(sh).cuda()
        mom = torch.empty((S, 4), dtype=torch.float64, device="cuda")
        hist = torch.empty((S, 7), dtype=torch.int32, device="cuda")
        fit = torch.empty(3, dtype=torch.float64, device="cuda")
        B.ch_stats_moments(series, mom)
        B.ch_stats_hist(series, 0.0, 0.1, 7, hist)
        B.ch_stats_fit(mom, 1.0, 0.5, 0.0, 100.0, fit)
        torch.cuda.synchronize()
        ref = so.moments(sh)
        assert np.allclose(mom.cpu().numpy(), ref, rtol=1e-11, atol=1e-17)
        assert np.array_equal(hist.cpu().numpy(), so.hist(sh, 0.0, 0.1, 7))
        f = fit.cpu().numpy()
        assert np.isclose(f[0], so.beta0(ref, 1.0, 0.5, 0.0, 100.0), rtol=1e-12)
        assert np.isclose(f[1], so.slope_k(ref, 1.0, 0.5, 0.0, 100.0), rtol=1e-12)
    with pytest.raises(B.ChError):
        B.ch_stats_hist(series, 0.0, -1.0, 7, hist)


# ---------------------------------------------------- grid-doubling convergence
def test_grid_doubling_error_kernel(B):
    import torch
    from oracle import stats_oracle as so
    rng = np.random.default_rng(4)
    for M, n in [(1, 1), (3, 8), (2, 37), (1, 256)]:
        fine, coarse = rng.standard_normal((M, 2 * n, 2 * n)), rng.standard_normal((M, n, n))
        out = torch.empty(M, dtype=torch.float64, device="cuda")
        B.ch_grid_doubling_error(torch.from_numpy(fine).cuda(), torch.from_numpy(coarse).cuda(), out)
        assert np.allclose(out.cpu().numpy(), so.grid_doubling_error(fine, coarse), rtol=1e-12)


def test_grid_doubling_study_first_order_and_oracle_parity(B, oracle):
    """Appendix A: elliptical droplet on [0, 2 pi]^2, gamma = 0.01, dt = 0.1 dx, T = 10
    (gamma dt / dx^4 = 2.1 at n = 128 ... 1082 at n = 1024).  The n = 128 run is checked against the oracle
    step by step in the rescaled h = 1 units.  Error = O(dx^2) + O(dt) with dt ~ dx: the observed order
    log2(E_n / E_2n) must fall from 2 towards 1; halving dt at fixed n isolates the first order in time."""
    import math
    import torch
    from paper_1911_03386_b200 import convergence as cv
    from oracle import stats_oracle as so
    L = 2 * math.pi
    g, d, nsteps = cv.scaled_parameters(128, L, 0.01, 10.0, 0.1)
    Co, _ = oracle.run(inputs.droplet_state(128, L, 0.01, 1.8, 0.9), g, d, nsteps, nsteps)
    f128 = cv.final_state(128).cpu().numpy()
    assert np.abs(f128 - Co).max() <= FIELD_TOL
    rows = cv.study([128, 256, 512, 1024])
    ns, E, order = zip(*rows)
    assert ns == (256, 512, 1024)
    assert E[0] > E[1] > E[2] > 0                                   # converges
    assert 1.0 <= order[2] < order[1] <= 2.05, rows                  # between first and second order, falling
    assert abs(E[0] - so.grid_doubling_error(cv.final_state(256).cpu().numpy(), f128)[0]) <= 1e-12
    # the paper's Table A.6 (tests/golden/table_A6.txt): at n = 2048, 4096 its order is 1.00; with a different (readable)
    # initial condition only the asymptote is comparable: within 0.25 of the printed orders on the two finest grids
    import os
    paper = {int(l.split()[0]): float(l.split()[2]) for l in open(os.path.join(os.path.dirname(__file__), "golden", "table_A6.txt"))
             if l.strip() and not l.startswith("#")}
    fine = dict((n, o) for n, _, o in cv.study([1024, 2048, 4096]))
    assert abs(fine[4096] - paper[2048]) <= 0.25 and abs(fine[4096] - paper[4096]) <= 0.25, fine
    # time refinement at fixed n = 256: differences of successive halvings of dt halve (first order)
    a, b, c = (cv.final_state(256, dt_factor=f) for f in (0.2, 0.1, 0.05))
    d1, d2 = float((a - b).abs().mean()), float((b - c).abs().mean())
    assert 0.9 <= math.log2(d1 / d2) <= 1.1, (d1, d2)
