"""ctypes loader for the CPU oracle (oracle/ch_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It never imports the CUDA package's binding.
All arrays are C-contiguous float64 numpy arrays shaped [ensemble][(z)][y][x].
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ch_oracle.c")
_LIB = os.path.join(_HERE, "libch_oracle.so")
_lib = None

_dp = ctypes.POINTER(ctypes.c_double)


def build(force: bool = False) -> str:
    """Compile the oracle with gcc -O2 -fopenmp (OpenMP over members only)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-std=c11", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        L = _lib
        L.cho_num_threads.restype = ctypes.c_int
        L.cho_set_num_threads.argtypes = [ctypes.c_int]
        L.cho_solve_lines.argtypes = [ctypes.c_int, ctypes.c_double, _dp, ctypes.c_long, ctypes.c_int]
        L.cho_rhs.argtypes = [_dp, _dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double]
        L.cho_sweep.argtypes = [_dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_int]
        L.cho_step.argtypes = [_dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double,
                               ctypes.c_long, ctypes.c_int]
        L.cho_step_literal.argtypes = [_dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double,
                                       ctypes.c_double, ctypes.c_long]
        L.cho_energy.argtypes = [_dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double, _dp]
        L.cho_run.argtypes = [_dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double,
                              ctypes.c_long, ctypes.c_long, ctypes.c_double, _dp, ctypes.c_long]
        L.cho_run.restype = ctypes.c_long
    return _lib


def _ptr(a):
    return a.ctypes.data_as(_dp)


def _shape(C):
    C = np.ascontiguousarray(C, dtype=np.float64)
    D = C.ndim - 1
    assert D in (2, 3) and len(set(C.shape[1:])) == 1, "state must be [ensemble][(N,)N,N]"
    return C, C.shape[0], C.shape[1], D


def num_threads() -> int:
    return lib().cho_num_threads()


def set_num_threads(n: int) -> None:
    lib().cho_set_num_threads(int(n))


def solve_lines(b, sigma: float, dense: bool = False) -> np.ndarray:
    """Solve circulant(s,-4s,1+6s,-4s,s) v = b for each row of b[count][N]."""
    x = np.array(b, dtype=np.float64, order="C", copy=True)
    x2 = x.reshape(-1, x.shape[-1])
    rc = lib().cho_solve_lines(x2.shape[1], float(sigma), _ptr(x2), x2.shape[0], int(dense))
    assert rc == 0, rc
    return x


def rhs(C, gamma: float, dt: float) -> np.ndarray:
    C, M, N, D = _shape(C)
    r = np.empty_like(C)
    assert lib().cho_rhs(_ptr(C), _ptr(r), M, N, D, gamma, dt) == 0
    return r


def sweep(w, sigma: float, axis: int) -> np.ndarray:
    """axis 0 = x (fastest), 1 = y, 2 = z."""
    w, M, N, D = _shape(w)
    w = w.copy()
    assert lib().cho_sweep(_ptr(w), M, N, D, float(sigma), axis) == 0
    return w


def step(C, gamma: float, dt: float, nsteps: int = 1, dense: bool = False) -> np.ndarray:
    C, M, N, D = _shape(C)
    C = C.copy()
    assert lib().cho_step(_ptr(C), M, N, D, gamma, dt, nsteps, int(dense)) == 0
    return C


def step_literal(C, gamma: float, dt: float, nsteps: int = 1) -> np.ndarray:
    C, M, N, D = _shape(C)
    C = C.copy()
    assert lib().cho_step_literal(_ptr(C), M, N, D, gamma, dt, nsteps) == 0
    return C


def energy(C, gamma: float, t: float = 0.0) -> np.ndarray:
    """[ensemble][4] = {F, dF/dt, beta, mass} of the state at time t."""
    C, M, N, D = _shape(C)
    out = np.empty((M, 4), dtype=np.float64)
    assert lib().cho_energy(_ptr(C), M, N, D, gamma, float(t), _ptr(out)) == 0
    return out


def run(C, gamma: float, dt: float, nsteps: int, stride: int, t0: float = 0.0):
    """Returns (C_end, series[samples][ensemble][4]); sample k is the state after k*stride steps."""
    C, M, N, D = _shape(C)
    C = C.copy()
    cap = nsteps // stride + 1
    series = np.zeros((cap, M, 4), dtype=np.float64)
    k = lib().cho_run(_ptr(C), M, N, D, gamma, dt, nsteps, stride, float(t0), _ptr(series), cap)
    assert k == cap, (k, cap)
    return C, series
