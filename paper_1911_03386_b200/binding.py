"""Thin ctypes binding over the C ABI of include/ch.h (argument marshalling only).

Every step of the path runs in the CUDA kernels of libch.so; there is no CPU fallback:
loading fails loudly if the library has not been built (python -m paper_1911_03386_b200.build),
and ch_create fails without a CUDA device.  Module-level functions carry the C names;
`Ensemble` is a convenience wrapper holding the context.  Arrays may be numpy (host)
or torch CUDA tensors (device); torch is used only for device memory and streams.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

CH_OK, CH_EINVAL, CH_ENOMEM, CH_ECUDA, CH_ESTATE, CH_ENONFINITE = 0, -1, -2, -3, -4, -5

EXPORTS = [
    "ch_create", "ch_destroy", "ch_set_stream", "ch_workspace_bytes", "ch_attach_workspace",
    "ch_set_state", "ch_set_time", "ch_set_series", "ch_step", "ch_run_host", "ch_energy", "ch_energy_static", "ch_get_state",
    "ch_series_count", "ch_step_count", "ch_rhs", "ch_sweep", "ch_set_option", "ch_get_option",
    "ch_droplet_create", "ch_droplet_destroy", "ch_droplet_set_stream", "ch_droplet_set_state", "ch_droplet_get_state",
    "ch_droplet_integrate", "ch_droplet_replay", "ch_droplet_energy", "ch_droplet_last_error",
    "ch_launch_count", "ch_last_error", "ch_profile", "ch_profile_read", "ch_kernel_kinds",
    "ch_kernel_kind_name", "ch_stats_moments", "ch_stats_hist", "ch_stats_fit", "ch_grid_doubling_error",
]

# CH_LIBCH selects another build of the library (the debug build with in-kernel synchronisation assertions, build.py)
_LIBPATH = os.environ.get("CH_LIBCH") or os.path.join(os.path.dirname(os.path.abspath(__file__)), "libch.so")
_lib = None


class ChError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libch error {code}: {msg}")
        self.code = code


def lib():
    """Load libch.so (raises if it is missing: the CUDA path is the only path)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIBPATH):
            raise RuntimeError(f"{_LIBPATH} not built; run `python -m paper_1911_03386_b200.build` "
                               "(there is no CPU fallback)")
        L = ctypes.CDLL(_LIBPATH)
        vp, dp, ci, cd = ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_double
        L.ch_create.argtypes = [ctypes.POINTER(vp), ci, ci, ci, cd, cd]
        L.ch_destroy.argtypes = [vp]
        L.ch_set_stream.argtypes = [vp, vp]
        L.ch_workspace_bytes.argtypes = [ci, ci, ci]
        L.ch_workspace_bytes.restype = ctypes.c_size_t
        L.ch_attach_workspace.argtypes = [vp, vp, ctypes.c_size_t]
        L.ch_set_state.argtypes = [vp, dp, ci]
        L.ch_set_time.argtypes = [vp, cd]
        L.ch_set_series.argtypes = [vp, dp, ci, ci]
        L.ch_step.argtypes = [vp, ci]
        L.ch_run_host.argtypes = [vp, dp, dp, ci, ci]
        L.ch_energy.argtypes = [vp, dp, ci]
        L.ch_energy_static.argtypes = [dp, ci, ci, ci, cd, cd, dp, vp, ctypes.c_char_p, ctypes.c_size_t]
        L.ch_get_state.argtypes = [vp, dp, ci]
        L.ch_series_count.argtypes = [vp]
        L.ch_step_count.argtypes = [vp]
        L.ch_step_count.restype = ctypes.c_longlong
        L.ch_rhs.argtypes = [vp, dp, ci]
        L.ch_sweep.argtypes = [vp, dp, ci, ci]
        L.ch_set_option.argtypes = [vp, ctypes.c_char_p, ci]
        L.ch_get_option.argtypes = [vp, ctypes.c_char_p, ctypes.POINTER(ci)]
        L.ch_launch_count.argtypes = [vp]
        L.ch_launch_count.restype = ctypes.c_longlong
        L.ch_profile.argtypes = [vp, ci]
        L.ch_profile_read.argtypes = [vp, ctypes.POINTER(cd), ctypes.POINTER(ctypes.c_longlong), ci]
        L.ch_kernel_kinds.restype = ci
        L.ch_kernel_kind_name.argtypes = [ci]
        L.ch_kernel_kind_name.restype = ctypes.c_char_p
        L.ch_stats_moments.argtypes = [dp, ci, ci, dp, vp]
        L.ch_stats_hist.argtypes = [dp, ci, ci, cd, cd, ci, vp, vp]
        L.ch_stats_fit.argtypes = [dp, ci, cd, cd, cd, cd, dp, vp]
        L.ch_grid_doubling_error.argtypes = [dp, dp, ci, ci, dp, vp]
        L.ch_last_error.argtypes = [vp]
        L.ch_last_error.restype = ctypes.c_char_p
        L.ch_droplet_create.argtypes = [ctypes.POINTER(vp), ci, ci, cd]
        L.ch_droplet_destroy.argtypes = [vp]
        L.ch_droplet_set_stream.argtypes = [vp, vp]
        L.ch_droplet_set_state.argtypes = [vp, dp, ci]
        L.ch_droplet_get_state.argtypes = [vp, dp, ci]
        L.ch_droplet_integrate.argtypes = [vp, cd, cd, cd, cd, ctypes.c_longlong, dp, ci, vp]
        L.ch_droplet_replay.argtypes = [vp, dp, ci, ci]
        L.ch_droplet_energy.argtypes = [vp, dp, ci]
        L.ch_droplet_last_error.argtypes = [vp]
        L.ch_droplet_last_error.restype = ctypes.c_char_p
        _lib = L
    return _lib


def _ptr(a):
    """(address, on_device) of a C-contiguous float64 numpy array or torch tensor."""
    if isinstance(a, np.ndarray):
        assert a.dtype == np.float64 and a.flags.c_contiguous
        return a.ctypes.data, 0
    import torch
    assert isinstance(a, torch.Tensor) and a.dtype == torch.float64 and a.is_contiguous()
    return a.data_ptr(), 1 if a.is_cuda else 0


def _check(ctx, rc):
    if rc != CH_OK:
        raise ChError(rc, lib().ch_last_error(ctx).decode())


# ---- C names ---------------------------------------------------------------------------
def ch_create(ensemble, N, D, gamma, dt):
    ctx = ctypes.c_void_p()
    rc = lib().ch_create(ctypes.byref(ctx), ensemble, N, D, gamma, dt)
    if rc != CH_OK:
        raise ChError(rc, lib().ch_last_error(None).decode())
    return ctx


def ch_destroy(ctx):
    return lib().ch_destroy(ctx)


def ch_set_stream(ctx, stream):
    _check(ctx, lib().ch_set_stream(ctx, ctypes.c_void_p(stream)))


def ch_workspace_bytes(ensemble, N, D):
    return lib().ch_workspace_bytes(ensemble, N, D)


def ch_attach_workspace(ctx, tensor):
    _check(ctx, lib().ch_attach_workspace(ctx, tensor.data_ptr(), tensor.numel() * tensor.element_size()))


def ch_set_state(ctx, C):
    p, dev = _ptr(C)
    _check(ctx, lib().ch_set_state(ctx, p, dev))


def ch_run_host(ctx, C_in, C_out, nsteps, chunk=0):
    """C_in, C_out: host arrays (numpy, or CPU torch tensors -- pinned for overlap) of the ensemble's shape."""
    pi, di = _ptr(C_in)
    po, do = _ptr(C_out)
    assert di == 0 and do == 0, "ch_run_host takes host buffers"
    _check(ctx, lib().ch_run_host(ctx, pi, po, nsteps, chunk))


def ch_set_time(ctx, t0):
    _check(ctx, lib().ch_set_time(ctx, t0))


def ch_set_series(ctx, series, stride, capacity):
    _check(ctx, lib().ch_set_series(ctx, None if series is None else series.data_ptr(), stride, capacity))


def ch_step(ctx, nsteps):
    _check(ctx, lib().ch_step(ctx, nsteps))


def ch_energy(ctx, out):
    p, dev = _ptr(out)
    _check(ctx, lib().ch_energy(ctx, p, dev))


def ch_energy_static(C, gamma, t, out, stream=None):
    """C: CUDA tensor [ensemble][N]^D, out: CUDA tensor [ensemble][4] (output).  No context, no allocation (include/ch.h)."""
    M, N, D = C.shape[0], C.shape[1], C.dim() - 1
    assert C.is_cuda and out.is_cuda and C.is_contiguous() and out.is_contiguous() and tuple(out.shape) == (M, 4)
    err = ctypes.create_string_buffer(512)
    rc = lib().ch_energy_static(C.data_ptr(), M, N, D, gamma, t, out.data_ptr(), ctypes.c_void_p(stream or 0), err, 512)
    if rc != CH_OK:
        raise ChError(rc, err.value.decode())


def ch_get_state(ctx, C):
    p, dev = _ptr(C)
    _check(ctx, lib().ch_get_state(ctx, p, dev))


def ch_series_count(ctx):
    return lib().ch_series_count(ctx)


def ch_step_count(ctx):
    return lib().ch_step_count(ctx)


def ch_rhs(ctx, r_out):
    p, dev = _ptr(r_out)
    _check(ctx, lib().ch_rhs(ctx, p, dev))


def ch_sweep(ctx, w, axis):
    p, dev = _ptr(w)
    _check(ctx, lib().ch_sweep(ctx, p, axis, dev))


def ch_set_option(ctx, key, value):
    _check(ctx, lib().ch_set_option(ctx, key.encode(), int(value)))


def ch_get_option(ctx, key):
    v = ctypes.c_int()
    rc = lib().ch_get_option(ctx, key.encode(), ctypes.byref(v))
    if rc != CH_OK:
        raise ChError(rc, f"unknown option {key}")
    return v.value


def ch_launch_count(ctx):
    return lib().ch_launch_count(ctx)


def ch_profile(ctx, enable):
    _check(ctx, lib().ch_profile(ctx, int(enable)))


def ch_profile_read(ctx):
    """{kind name: (total ms, launches)} since profiling was switched on / last read."""
    n = lib().ch_kernel_kinds()
    ms = (ctypes.c_double * n)()
    cnt = (ctypes.c_longlong * n)()
    _check(ctx, lib().ch_profile_read(ctx, ms, cnt, n))
    return {lib().ch_kernel_kind_name(k).decode(): (ms[k], cnt[k]) for k in range(n)}


def _stats_check(rc, what):
    if rc != CH_OK:
        raise ChError(rc, what)


def ch_stats_moments(series, moments, stream=None):
    """series: CUDA tensor [S][M][4]; moments: CUDA tensor [S][4] (output)."""
    S, M = series.shape[0], series.shape[1]
    assert series.is_cuda and moments.is_cuda and series.is_contiguous() and tuple(moments.shape) == (S, 4)
    _stats_check(lib().ch_stats_moments(series.data_ptr(), S, M, moments.data_ptr(), ctypes.c_void_p(stream or 0)), "ch_stats_moments")


def ch_stats_hist(series, lo, width, nbins, hist, stream=None):
    """hist: CUDA int32 tensor [S][nbins] (output)."""
    S, M = series.shape[0], series.shape[1]
    assert series.is_cuda and hist.is_cuda and series.is_contiguous() and tuple(hist.shape) == (S, nbins)
    _stats_check(lib().ch_stats_hist(series.data_ptr(), S, M, lo, width, nbins, hist.data_ptr(), ctypes.c_void_p(stream or 0)), "ch_stats_hist")


def ch_stats_fit(moments, t0, dt_sample, t1, t2, out, stream=None):
    """out: CUDA tensor [3] = {beta_0, k, samples in the window} (output)."""
    assert moments.is_cuda and out.is_cuda and out.numel() == 3
    _stats_check(lib().ch_stats_fit(moments.data_ptr(), moments.shape[0], t0, dt_sample, t1, t2, out.data_ptr(),
                                    ctypes.c_void_p(stream or 0)), "ch_stats_fit")


def ch_grid_doubling_error(fine, coarse, out, stream=None):
    """fine: CUDA tensor [M][2n][2n], coarse: [M][n][n], out: [M] (output): eq. (A.1)."""
    M, n = coarse.shape[0], coarse.shape[1]
    assert fine.is_cuda and coarse.is_cuda and out.is_cuda and fine.is_contiguous() and coarse.is_contiguous()
    assert tuple(fine.shape) == (M, 2 * n, 2 * n) and tuple(coarse.shape) == (M, n, n) and out.numel() == M
    _stats_check(lib().ch_grid_doubling_error(fine.data_ptr(), coarse.data_ptr(), M, n, out.data_ptr(),
                                              ctypes.c_void_p(stream or 0)), "ch_grid_doubling_error")


# ---- Model 1: droplet populations (include/ch.h, ch_droplet_*) ---------------------------
def _dcheck(ctx, rc):
    if rc != CH_OK:
        raise ChError(rc, lib().ch_droplet_last_error(ctx).decode())


def ch_droplet_create(realisations, N, eps):
    ctx = ctypes.c_void_p()
    rc = lib().ch_droplet_create(ctypes.byref(ctx), realisations, N, eps)
    if rc != CH_OK:
        raise ChError(rc, lib().ch_droplet_last_error(None).decode())
    return ctx


def ch_droplet_destroy(ctx):
    return lib().ch_droplet_destroy(ctx)


def ch_droplet_set_stream(ctx, stream):
    _dcheck(ctx, lib().ch_droplet_set_stream(ctx, ctypes.c_void_p(stream)))


def ch_droplet_set_state(ctx, R):
    p, dev = _ptr(R)
    _dcheck(ctx, lib().ch_droplet_set_state(ctx, p, dev))


def ch_droplet_get_state(ctx, R):
    p, dev = _ptr(R)
    _dcheck(ctx, lib().ch_droplet_get_state(ctx, p, dev))


def ch_droplet_integrate(ctx, t_end, rtol=1e-6, atol=1e-9, h0=1e-4, max_steps=10_000_000, steps=None, nsteps=None):
    """steps: CUDA float64 tensor [M][max_record] or None; nsteps: CUDA int32 tensor [M] or None (outputs)."""
    _dcheck(ctx, lib().ch_droplet_integrate(ctx, t_end, rtol, atol, h0, max_steps,
                                            None if steps is None else steps.data_ptr(), 0 if steps is None else steps.shape[1],
                                            None if nsteps is None else nsteps.data_ptr()))


def ch_droplet_replay(ctx, steps):
    """steps: CUDA float64 tensor [M][nsteps]; a non-positive entry ends a row early."""
    assert steps.is_cuda and steps.is_contiguous()
    _dcheck(ctx, lib().ch_droplet_replay(ctx, steps.data_ptr(), steps.shape[1], steps.shape[1]))


def ch_droplet_energy(ctx, out):
    p, dev = _ptr(out)
    _dcheck(ctx, lib().ch_droplet_energy(ctx, p, dev))


# ---- convenience wrapper ---------------------------------------------------------------
class Ensemble:
    """Context holder: Ensemble(ensemble, N, D, gamma, dt); methods mirror the C calls."""

    def __init__(self, ensemble, N, D, gamma, dt, stream=None, options=None):
        self.shape = (ensemble,) + (N,) * D
        self.ensemble, self.N, self.D, self.gamma, self.dt = ensemble, N, D, gamma, dt
        self.ctx = ch_create(ensemble, N, D, gamma, dt)
        self._series = None
        self.stride = 0
        if stream is not None:
            ch_set_stream(self.ctx, stream)
        for k, v in (options or {}).items():
            ch_set_option(self.ctx, k, v)

    def close(self):
        if self.ctx is not None:
            ch_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_state(self, C):
        assert tuple(C.shape) == self.shape, (tuple(C.shape), self.shape)
        ch_set_state(self.ctx, C)

    def set_series(self, stride, capacity):
        """Allocate a device series buffer [capacity][ensemble][4] (torch) and register it."""
        import torch
        self._series = torch.zeros((capacity, self.ensemble, 4), dtype=torch.float64, device="cuda")
        self.stride = stride
        ch_set_series(self.ctx, self._series, stride, capacity)

    def step(self, nsteps):
        ch_step(self.ctx, nsteps)

    def get_state(self, out=None):
        if out is None:
            out = np.empty(self.shape, dtype=np.float64)
        ch_get_state(self.ctx, out)
        return out

    def energy(self):
        out = np.empty((self.ensemble, 4), dtype=np.float64)
        ch_energy(self.ctx, out)
        return out

    def series(self):
        """Samples written so far, as a host array [count][ensemble][4]."""
        import torch
        torch.cuda.synchronize()
        return self._series[: ch_series_count(self.ctx)].cpu().numpy()

    def rhs(self):
        out = np.empty(self.shape, dtype=np.float64)
        ch_rhs(self.ctx, out)
        return out

    def sweep(self, w, axis):
        w = np.array(w, dtype=np.float64, order="C", copy=True)
        ch_sweep(self.ctx, w, axis)
        return w
