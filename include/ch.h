/*
 * ch.h -- C ABI of libch: ensemble Cahn-Hilliard semi-implicit ADI stepper for
 * NVIDIA B200 (sm_100a), fp64, one GPU per context.
 *
 * Citations: P:nnn = line nnn of the paper text (arXiv 1911.03386, PAPER.md);
 * Gk = reading k in DESIGN.md ("Readings of the paper").
 *
 * The method (eq.(3); "semi-implicit ADI finite-difference
 * method, periodic boundary conditions"; scheme left open by the paper and fixed by
 * reading G1/G2).  Grid spacing h = 1, periodic N^D grid per ensemble member:
 *
 *     mu^n    = (C^n)^3 - C^n - gamma Lap_h C^n
 *     r       = dt Lap_h mu^n
 *     w       = A_z^-1 A_y^-1 A_x^-1 r       A_d = I + gamma dt (delta_d^2)^2, cyclic pentadiagonal,
 *                                            rows (s,-4s,1+6s,-4s,s), s = gamma dt; A_z only if D = 3
 *     C^{n+1} = C^n + w
 *
 * which is (I + s dxx^2)(I + s dyy^2) C^{n+1} = C^n + dt Lap_h[(C^n)^3 - C^n]
 * - 2 s dxx dyy C^n + s^2 dxx^2 dyy^2 C^n  (three factors in 3D) with C^n subtracted
 * from both sides.  Diagnostics of a state at time t (eq.(4) with the bulk
 * prefactor 1/4, G3; forward differences, G4; eq.(6); eq.(43)):
 *
 *     F    = sum_i [ (C_i^2 - 1)^2 / 4 + gamma/2 sum_d (C_{i+e_d} - C_i)^2 ]
 *     Fdot = - sum_i sum_d (mu_{i+e_d} - mu_i)^2
 *     mass = sum_i C_i
 *     beta = - t Fdot / F                    (0 when F == 0)
 *
 * A physical run with spacing h maps onto h = 1 by gamma' = gamma/h^2, dt' = dt/h^2,
 * F = h^D F', beta unchanged.
 *
 * Layout: every state / field pointer is ensemble * N^D contiguous doubles,
 * C[m][y][x] (D = 2) or C[m][z][y][x] (D = 3), x fastest, member stride N^D.
 * "on_device" arguments say whether a caller pointer is device (1) or host (0) memory.
 *
 * Ownership: the context owns its factorisation tables and, unless a workspace is
 * attached, its device arrays.  State passed in or out is copied.  A series buffer
 * is caller-owned device memory and must outlive every ch_step that writes it.
 *
 * Errors: every call returns CH_OK (0) or a negative code; nothing throws or aborts
 * across the boundary.  ch_last_error() gives a message for the last failure on a
 * context.  There is no CPU fallback: without a CUDA device ch_create fails with
 * CH_ECUDA.
 *
 * Determinism: same inputs give bitwise-same outputs run to run; the result of a
 * member does not depend on the ensemble size or on its position in the ensemble
 * (bitwise for the exact kernels; to within the stated truncation, < 2^-56 of the
 * local max |w| per sweep, for the one-pass local step, option "fuse" = 5).
 */
#ifndef CH_H
#define CH_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ch_ctx ch_ctx;   /* opaque; created by ch_create, freed by ch_destroy */

enum {
    CH_OK = 0,
    CH_EINVAL = -1,      /* null pointer, ensemble < 1, D not in {2,3}, N < 8, gamma <= 0, dt <= 0,
                            nsteps < 0, workspace too small, series full, unknown option */
    CH_ENOMEM = -2,      /* host or device allocation failed */
    CH_ECUDA = -3,       /* CUDA runtime error (message in ch_last_error) */
    CH_ESTATE = -4,      /* step / energy / get_state before set_state */
    CH_ENONFINITE = -5   /* ch_energy found a non-finite F (state has blown up) */
};

/* Create a context for `ensemble` independent members on an N^D periodic grid (D = 2 or 3,
 * N >= 8, any N; N a multiple of 16 takes the fast kernels) with parameters gamma, dt of
 * eq.(3) at h = 1.  Computes the periodic (circulant) LU factorisation of A_d on the host
 * (DESIGN.md "Factorisation").  Uses the current CUDA device.  *out is set on success. */
int ch_create(ch_ctx **out, int ensemble, int N, int D, double gamma, double dt);

/* Free the context and everything it owns (not an attached workspace, not the series). */
int ch_destroy(ch_ctx *ctx);

/* Stream on which every later call enqueues its work (a cudaStream_t, e.g.
 * torch.cuda.current_stream().cuda_stream).  Default: the legacy default stream. */
int ch_set_stream(ch_ctx *ctx, void *cuda_stream);

/* Bytes of device memory a context of this shape needs (state, work array, reduction
 * partials).  0 on invalid arguments. */
size_t ch_workspace_bytes(int ensemble, int N, int D);

/* Use caller-owned device memory (256-byte aligned, >= ch_workspace_bytes) instead of
 * cudaMalloc.  Must be called before ch_set_state; the buffer must outlive the context. */
int ch_attach_workspace(ch_ctx *ctx, void *dev, size_t bytes);

/* Copy ensemble*N^D doubles into the context (stream-ordered; synchronises if the source
 * is host memory).  Resets the step counter n = 0, the time origin t0 = 0 and the series cursor. */
int ch_set_state(ch_ctx *ctx, const double *C, int on_device);

/* Time origin for beta after a restart: samples are taken at t = t0 + n dt (G6). */
int ch_set_time(ch_ctx *ctx, double t0);

/* Per-member time series, caller-owned DEVICE buffer series[capacity][ensemble][4] =
 * {F, dF/dt, beta, mass}.  A sample is written for the state after n steps whenever
 * n % stride == 0, including n = 0 (sample k at t = t0 + k stride dt).
 * Pass NULL to switch sampling off.  Resets the series cursor. */
int ch_set_series(ch_ctx *ctx, double *series_dev, int stride, int capacity);

/* Advance every member by nsteps steps.  Asynchronous: work is enqueued on the stream and
 * the call returns.  CH_EINVAL (nothing enqueued) if the series would overflow. */
int ch_step(ch_ctx *ctx, int nsteps);

/* {F, dF/dt, beta, mass} of the current state, out[ensemble][4].  With a host pointer the
 * call synchronises the stream and returns CH_ENONFINITE if any F is not finite. */
int ch_energy(ch_ctx *ctx, double *out, int on_device);

/* The same {F, dF/dt, beta, mass} (eq. (4), eq. (6); readings G3-G6) WITHOUT A CONTEXT AND WITHOUT ANY
 * ALLOCATION -- for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid it).  C_dev: DEVICE field [ensemble][N^D] (layout as ch_set_state), out_dev: DEVICE double[ensemble][4],
 * t: the time beta is taken at (beta = -t dF/dt / F, 0 if F == 0); h = 1; enqueued on cuda_stream (a cudaStream_t, NULL =
 * the legacy default stream), nothing synchronises; the CUDA device that is current must own both buffers.  The reduction
 * partials live in a file-scope __device__ array of CH_ENERGY_STATIC_MAX_PARTS x 3 doubles (1.5 MiB, held by every GPU
 * that loads the library until the process exits); a call needs ensemble * ceil(N^D / CH_ENERGY_STATIC_PART_POINTS) of
 * them and is REJECTED with CH_EINVAL (nothing enqueued) beyond that, e.g. above 1024 members of 512^2, 64 of 2048^2 or 128 of
 * 128^3 (2 GiB of state): use ch_energy, or split the ensemble over several calls.  The array is shared by every call and keeps the
 * last call's contents (nothing in it has to start at zero: a call writes every slot it reads), so CALLS THAT OVERLAP ON
 * THE GPU -- different streams without ordering, or different host threads -- RACE; calls ordered on one stream do not.
 * The first call on a device looks the array's device address up (cudaGetSymbolAddress; make that call outside graph
 * capture).  Calls no cudaMalloc, cudaFree or allocating library routine.  Slower than ch_energy (no shared-memory
 * tiles); same values to round-off.  Errors: CH_EINVAL (NULL pointer, ensemble < 1, N < 8, D not in {2, 3}, gamma <= 0,
 * too large), CH_ECUDA; the message goes to errbuf (may be NULL) as a NUL-terminated string of at most errlen bytes. */
#define CH_ENERGY_STATIC_PART_POINTS 4096
#define CH_ENERGY_STATIC_MAX_PARTS 65536
int ch_energy_static(const double *C_dev, int ensemble, int N, int D, double gamma, double t, double *out_dev,
                     void *cuda_stream, char *errbuf, size_t errlen);

/* Copy the current state out (stream-ordered; synchronises if the target is host memory). */
int ch_get_state(ch_ctx *ctx, double *C, int on_device);

/* The whole job from and to HOST memory: equivalent to ch_set_state(C_in, host) + ch_step(nsteps) + ch_get_state(C_out, host)
 * (bitwise for the exact kernels; the series buffer registered with ch_set_series is filled the same way; afterwards the
 * context holds the final state, n = nsteps, t0 = 0), but done member chunk by member chunk -- members are independent
 * -- so that the host-to-device copy of chunk k + 1, the steps of chunk k and the device-to-host copy of
 * chunk k - 1 overlap on three internal streams (ordered after everything already enqueued on the context's stream).
 * `chunk` = members per chunk, 0 = library default (about 4 Mi grid points, 2 Mi for jobs of <= 30 steps; at least 4 chunks).  C_in and C_out
 * (ensemble * N^D doubles each, may be the same buffer) should be pinned host memory for the copies to be asynchronous.
 * Synchronous: returns when everything has completed.  CUDA graphs are not used inside. */
int ch_run_host(ch_ctx *ctx, const double *C_in, double *C_out, int nsteps, int chunk);

/* Number of series samples written (enqueued) so far, steps taken since ch_set_state. */
int ch_series_count(const ch_ctx *ctx);
long long ch_step_count(const ch_ctx *ctx);

/* Components of one step, exported for per-kernel parity tests and profiling.
 * ch_rhs:   r = dt Lap_h mu(C) of the CURRENT state into r_out (device or host).
 * ch_sweep: w := A_axis^-1 w on a caller field of the context's shape (axis 0 = x, 1 = y, 2 = z),
 *           in place, device or host.  Neither touches the state or the step counter. */
int ch_rhs(ch_ctx *ctx, double *r_out, int on_device);
int ch_sweep(ch_ctx *ctx, double *w, int axis, int on_device);

/* Kernel-variant options (measurement knobs; every variant computes the same step to round-off):
 *   "sweep"    0 auto, 1 force the generic thread-per-line sweeps, 2 force the chunked periodic-LU sweeps,
 *              3 parallel cyclic reduction for the x-axis of ch_sweep (N a power of two <= 4096)
 *   "fuse"     which 2D step runs: 0 auto, 1 three passes (RHS, x-sweep, y-sweep + update; 56 B per update),
 *              2 RHS fused into a cluster/st.async y-sweep, 3 the line kernel (N in {32, 64, 96, 128, 160, 192, 224,
 *              256, 320, 384, 448, 512}), 4 the cluster line kernel (N in {1024, 2048, 4096}); modes 2-4 finish with the
 *              x-sweep fused with C += w (40 B per update); 5 the one-pass local step:
 *              RHS, y-sweep, x-sweep and update in one kernel that reads C^n once and writes C^{n+1} once (16 B per
 *              update), legal when the recurrences of the factorisation decay within 18 points to below 2^-56 of the
 *              data (gamma dt <~ 0.012; the bound is computed on the host, "local_reach"); auto picks it for D = 2,
 *              N >= 256 when it is legal and the exact modes otherwise; 6 member-resident stepping (SURVEY.md 8(f)
 *              NEXT-3 (ii); D = 2; one CTA per member for N in {32, 64, 96}, a cluster of 2 / 8 CTAs for N = 128 / 256):
 *              a whole ch_step(nsteps) call, with the samples
 *              that fall inside it, is ONE launch that keeps each member and its work array in shared memory (exact
 *              periodic solves, any gamma dt; global memory is read and written once per call, so the bound is the
 *              fp64 / shared-memory pipe, not HBM); auto picks it for N <= 128 (measured 1.1 - 2.3 x the line kernel;
 *              at N = 256 it measures slower than the line kernel and is explicit only).  A mode the shape does not support is CH_EINVAL.
 *   "resident_lines" one-CTA member-resident kernel (N <= 96): 0 auto (two lines per thread when at least two CTAs share an SM, i.e.
 *              ensemble >= 2 x multiprocessors, or N = 96), 1 one line per thread, 2 two lines per thread (half the shared-
 *              memory traffic, half the warps); fields and samples are bitwise the same either way
 *   "pdl"      0 (default): the stepping kernels of the fast paths are launched as programmatic dependents (they may start
 *              while their predecessor on the stream drains and wait inside the kernel before touching memory; same results),
 *              1 plain launches
 *   "linesync" line kernel: 0 auto (neighbour-warp flags when the closure is truncated to 2 chunks), 1 CTA barriers
 *   "scan"     closure of the chunk states: 0 auto (log-depth shuffle scan when the K-term sum is long), 1 K-term
 *              sum always, 2 scan wherever it is available
 *   "graph"    0 auto = 2 (plain steps between sampling steps are replayed as a CUDA graph of 8 steps, captured on first use;
 *              bitwise the same results and launch count; not while profiling), 1 plain launches, 2 graphs always
 *   "rhs3"     3D RHS: 0 auto (z-marching kernel for N in {64, 128}), 1 tile kernel
 *   "sweep3"   3D x/y sweeps: 0 auto (one pass per z-plane in shared memory for N in {64, 128}; cluster pairs at
 *              N = 128), 1 separate x- and y-sweeps, 2 one CTA per plane
 * ch_get_option answers these and, read-only: "chunked" (chunk length of the fast sweeps, 0 if N needs the generic
 * path), "K" (chunks summed by the periodic closure), "fused" / "line" / "cline" / "rhs3_stream" / "sweep_xy"
 * (non-zero if this shape has that kernel), "local" (non-zero if the one-pass local step is legal for this shape and
 * gamma dt), "local_reach" (its decay reach H in points, -1 if above the limit), "resident" (CTAs per member if member-resident
 * stepping is available for this shape, else 0), "fuse_mode" (the 2D step that will run: 0, 2, 3, 4, 5 or 6). */
int ch_set_option(ch_ctx *ctx, const char *key, int value);
int ch_get_option(const ch_ctx *ctx, const char *key, int *value);

/* Per-kernel device timing.  ch_profile(ctx, 1) makes every later launch be bracketed by CUDA
 * events on the context's stream; ch_profile_read synchronises, returns the summed milliseconds
 * and launch counts per kernel kind (ch_kernel_kinds() kinds, named by ch_kernel_kind_name:
 * rhs, rhs_diag, finish, sweep_x, sweep_y, sweep_z, rhs_sweep_y, rhs_sweep_y_diag, sweep_x_update, sweep_xy, step_local,
 * step_resident -- one record per ch_step call in that mode)
 * and clears the records. */
int ch_profile(ch_ctx *ctx, int enable);
int ch_profile_read(ch_ctx *ctx, double *ms, long long *counts, int nkinds);
int ch_kernel_kinds(void);
const char *ch_kernel_kind_name(int kind);

/* Kernel launches enqueued by this context since creation (each graph node counts once per replay). */
long long ch_launch_count(const ch_ctx *ctx);

/* ---- Ensemble statistics of the coarsening rate (off the hot path) ----
 * Input everywhere: the series buffer ch_step writes, series[nsamples][ensemble][4] = {F, dF/dt, beta, mass},
 * on the device.  Members gathered from several ranks are simply concatenated along the member axis first.
 * All calls are asynchronous on `stream` (a cudaStream_t, NULL = default stream); outputs are device pointers
 * owned by the caller.  Return CH_OK, CH_EINVAL (null pointer, sizes < 1, bad window or bins), CH_ECUDA.
 *
 * ch_stats_moments: eq. (41a,b): moments[s] = {mu_1, mu_2, mu_3, mu_4} of beta over the members at
 *   sample s, mu_1 = (1/M) sum_j beta_j, mu_p = (1/M) sum_j (beta_j - mu_1)^p.  moments_dev is [nsamples][4].
 * ch_stats_hist: histogram of beta at every sample time (Figs 9, 14, 18): hist[s][b] = number of members with
 *   floor((beta - lo) / width) == b, 0 <= b < nbins (values outside are dropped).  hist_dev is int[nsamples][nbins].
 * ch_stats_fit: over the samples with t1 <= t_s <= t2, t_s = t0 + s * dt_sample: out[0] = beta_0, the time average of
 *   mu_1 (eq. (42); trapezoid rule over the samples, divided by the span they cover), out[1] = k, the
 *   least-squares slope of mu_2 = k t through the origin, k = sum t mu_2 / sum t^2, out[2] = number of
 *   samples in the window.  moments_dev is the output of ch_stats_moments; out_dev is double[3]. */
int ch_stats_moments(const double *series_dev, int nsamples, int ensemble, double *moments_dev, void *stream);
int ch_stats_hist(const double *series_dev, int nsamples, int ensemble, double lo, double width, int nbins,
                  int *hist_dev, void *stream);
int ch_stats_fit(const double *moments_dev, int nsamples, double t0, double dt_sample, double t1, double t2,
                 double *out_dev, void *stream);

/* ch_grid_doubling_error: the self-convergence measure of eq. (A.1), P:672-674:
 *   out[m] = (1/|Omega|) sum_{i,j} | (1/4) (the four fine-grid values in coarse cell (i,j)) - coarse[m][i][j] | dx_c^2
 *          = (1/n_coarse^2) sum_{i,j} | ... |
 * for 2D fields fine[ensemble][2 n_coarse][2 n_coarse] and coarse[ensemble][n_coarse][n_coarse] on cell-centred grids
 * of the same periodic domain (device pointers, caller-owned; out_dev is double[ensemble]); asynchronous on stream. */
int ch_grid_doubling_error(const double *fine_dev, const double *coarse_dev, int ensemble, int n_coarse,
                           double *out_dev, void *stream);

/* Message for the last error on this context (never NULL); ch_create failures: pass NULL. */
const char *ch_last_error(const ch_ctx *ctx);

/* ---- Model 1: ensembles of droplet populations (off the hot path) ----
 * `realisations` independent populations of N droplets each (the paper: M = 100, N = 128 ... 8192, Table 1),
 *     dR_i/dt = H(R_i + eps) (-1/R_i^2 + ubar/R_i),   ubar = sum_i H(R_i) / sum_i H(R_i) R_i     eq. (39), eq. (14)
 * (H(s) = 1 for s > 0, else 0; eps = 1e-3 in the paper), integrated with the Dormand-Prince 5(4) pair -- the method of the
 * paper's ODE45, P:368 -- one CTA per realisation, the whole time loop in one launch.  Step controller (the paper states
 * none; reading G21): err = max_i |e_i| / (atol + rtol max(|R_i|, |R_i^new|)), accept iff err <= 1,
 * h_new = h min(5, max(0.2, 0.9 err^(-1/5))), the step clipped to land on t_end.
 * Layout: R[realisation][droplet], contiguous doubles.  Every call is asynchronous on the context's stream unless it
 * copies to or from host memory.  Errors as above (CH_EINVAL, CH_ENOMEM, CH_ECUDA, CH_ESTATE).
 *
 * ch_droplet_set_state: copies realisations * N radii in and resets every realisation's time to 0.
 * ch_droplet_integrate: advance every realisation from its current time to t_end (at most max_steps attempted steps,
 *   first trial step h0).  steps_dev (may be NULL): device double[realisations][max_record], receives the ACCEPTED step
 *   sizes; nsteps_dev (may be NULL): device int[realisations], their number.
 * ch_droplet_replay: advance by GIVEN step sizes without error control: steps_dev is device double[realisations][stride],
 *   the first nsteps entries of a row are used, a non-positive entry ends the row early.  (With the step sequence of a
 *   reference integration this reproduces it to round-off: the parity test.)
 * ch_droplet_energy: out[realisations][4] = {F, dF/dt, beta, V} at each realisation's current time t:
 *   F = sum_i H(R_i) R_i^2 / 2 (eq. (31)), dF/dt = -sum_i H(R_i) (1 - ubar R_i)^2 / R_i (eq. (33)),
 *   beta = -(t/F) dF/dt (eq. (36)), V = sum_i H(R_i) R_i^3 / 3 (the conserved volume). */
typedef struct ch_droplet_ctx ch_droplet_ctx;
int ch_droplet_create(ch_droplet_ctx **out, int realisations, int N, double eps);
int ch_droplet_destroy(ch_droplet_ctx *ctx);
int ch_droplet_set_stream(ch_droplet_ctx *ctx, void *cuda_stream);
int ch_droplet_set_state(ch_droplet_ctx *ctx, const double *R, int on_device);
int ch_droplet_get_state(ch_droplet_ctx *ctx, double *R, int on_device);
int ch_droplet_integrate(ch_droplet_ctx *ctx, double t_end, double rtol, double atol, double h0, long long max_steps,
                         double *steps_dev, int max_record, int *nsteps_dev);
int ch_droplet_replay(ch_droplet_ctx *ctx, const double *steps_dev, int nsteps, int stride);
int ch_droplet_energy(ch_droplet_ctx *ctx, double *out, int on_device);
const char *ch_droplet_last_error(const ch_droplet_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* CH_H */
