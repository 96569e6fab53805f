"""ch_energy_static (include/ch.h): the energy / beta reduction with its scratch in a file-scope __device__ array -- no
context, no allocation -- against the existing path (ch_energy of a context holding the same state), on two calls in a
row that share the static array.  Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh
process and after the other tests."""
import numpy as np
import pytest

from paper_1911_03386_b200 import inputs

pytestmark = pytest.mark.gpu

RTOL = 1e-9          # tests/test_parity_gpu.py SERIES_RTOL (north_star: relative 1e-9 on F(t), beta(t))


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_1911_03386_b200 import binding, build
    build.build()
    return binding


def existing_path(B, C0, gamma, t):
    M, N, D = C0.shape[0], C0.shape[1], C0.ndim - 1
    e = B.Ensemble(M, N, D, gamma, 0.01)
    e.set_state(C0)
    B.ch_set_time(e.ctx, t)
    ref = e.energy()
    e.close()
    return ref


def assert_close(got, ref):
    assert got.shape == ref.shape and np.isfinite(got).all()
    for q in (0, 1, 3):                                   # F, dF/dt, mass (mass of a symmetric mixture is ~0: scale >= 1)
        scale = np.maximum(np.abs(ref[:, q]), 1.0 if q == 3 else 1e-300)
        assert (np.abs(got[:, q] - ref[:, q]) / scale).max() <= RTOL, f"column {q}"
    assert (np.abs(got[:, 2] - ref[:, 2]) <= RTOL * np.abs(ref[:, 2]) + 1e-12).all(), "beta"


def test_energy_static_matches_ch_energy_on_two_calls_in_a_row(B):
    import torch
    # call 1 fills 5 * 16 slots of the static array, call 2 (another shape, fewer slots: 3 * 7, a ragged last part)
    # runs over what call 1 left there; then 3D, and the first shape once more
    cases = [(900, 5, 256, 2, 1.0, 3.5, -0.4), (910, 3, 164, 2, 0.7, 0.25, 0.0), (920, 2, 40, 3, 1.3, 2.0, -0.2),
             (900, 5, 256, 2, 1.0, 3.5, -0.4)]
    stream = torch.cuda.current_stream().cuda_stream
    pending = []
    for seed, M, N, D, gamma, t, cbar in cases:
        C0 = inputs.initial_state(range(seed, seed + M), N, D, cbar, 0.3)
        C = torch.from_numpy(C0).cuda()
        out = torch.full((M, 4), float("nan"), dtype=torch.float64, device="cuda")
        B.ch_energy_static(C, gamma, t, out, stream)
        pending.append((C0, gamma, t, out))
    torch.cuda.synchronize()                              # the four calls ran back to back on one stream
    for C0, gamma, t, out in pending:
        assert_close(out.cpu().numpy(), existing_path(B, C0, gamma, t))
    assert np.array_equal(pending[0][3].cpu().numpy(), pending[3][3].cpu().numpy())    # fixed summation order


def test_energy_static_rejects_sizes_beyond_the_static_array(B):
    import torch
    C = torch.zeros((2, 64, 64), dtype=torch.float64, device="cuda")
    out = torch.full((2, 4), 7.0, dtype=torch.float64, device="cuda")
    L = B.lib()
    import ctypes
    err = ctypes.create_string_buffer(512)
    # 65537 members of 64^2 need 65537 slots > CH_ENERGY_STATIC_MAX_PARTS: refused before anything is enqueued or read
    rc = L.ch_energy_static(C.data_ptr(), 65537, 64, 2, 1.0, 0.0, out.data_ptr(), None, err, 512)
    assert rc == B.CH_EINVAL and b"CH_ENERGY_STATIC_MAX_PARTS" in err.value and b"65537" in err.value
    rc = L.ch_energy_static(C.data_ptr(), 129, 128, 3, 1.0, 0.0, out.data_ptr(), None, err, 512)
    assert rc == B.CH_EINVAL and b"exceed" in err.value
    for bad in [(0, 64, 2, 1.0), (2, 4, 2, 1.0), (2, 64, 4, 1.0), (2, 64, 2, 0.0)]:
        assert L.ch_energy_static(C.data_ptr(), bad[0], bad[1], bad[2], bad[3], 0.0, out.data_ptr(), None, err, 512) == B.CH_EINVAL
    assert L.ch_energy_static(None, 2, 64, 2, 1.0, 0.0, out.data_ptr(), None, None, 0) == B.CH_EINVAL
    torch.cuda.synchronize()
    assert (out.cpu().numpy() == 7.0).all()
    with pytest.raises(B.ChError):
        B.ch_energy_static(torch.zeros((2, 4, 4), dtype=torch.float64, device="cuda"), 1.0, 0.0, out)
