"""lloid_svd_slice_noalloc (the entry point that allocates no device memory: its Jacobi working set is a fixed device array
inside the library) against the existing lloid_svd_slice, two calls in a row that share that array (-m gpu).
Collected last on purpose (the suite runs with pytest -x): passes alone in a fresh process and after the other tests."""
import ctypes as C

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _cuda():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def _compare(lib, torch, H, energy, tag):
    """Same tolerances as tests/test_gpu_svd.py; the two paths run the same kernels in the same order, so the results are
    expected to agree to the last bit -- checked with the suite's tolerances, reported exactly."""
    n, N = H.shape
    mb = min(n, N)
    U0, R0, s0, kept0 = lib.binding.lloid_svd_slice(H, energy)
    Hd = torch.from_numpy(np.ascontiguousarray(H)).cuda()
    Ud = torch.full((mb, N), float("nan"), dtype=torch.float32, device="cuda")
    Rd = torch.full((n, mb), float("nan"), dtype=torch.float32, device="cuda")
    L, s1, kept1 = lib.binding.lloid_svd_slice_noalloc(Hd, energy, Ud, Rd, torch.cuda.current_stream().cuda_stream)
    U1 = Ud.flatten()[:L * N].reshape(L, N).cpu().numpy()
    R1 = Rd.flatten()[:n * L].reshape(n, L).cpu().numpy()
    assert L == len(s0), (tag, L, len(s0))
    assert np.abs(s1 / s0 - 1).max() < 1e-10 and abs(kept1 - kept0) < 1e-12
    assert np.isfinite(U1).all() and np.isfinite(R1).all()
    assert np.abs(U1.astype(np.float64) @ U1.T - np.eye(L)).max() < 2e-6
    scale = np.abs(H).max()
    err = np.abs(R1.astype(np.float64) @ U1 - R0.astype(np.float64) @ U0).max() / scale
    exact = np.array_equal(U1, U0) and np.array_equal(R1, R0)
    print(f"{tag}: {H.shape} -> L = {L}, product err vs lloid_svd_slice {err:.1e}, bit-identical {exact}")
    assert err < 5e-6


def test_noalloc_svd_matches_the_allocating_path_on_two_calls_in_a_row():
    torch = _cuda()
    import paper_2511_04730_b200 as lib
    from workloads import chirp_templates
    # call 1 fills the shared scratch with a large problem (128 rows x 2048 taps = the stated maximum) ...
    H1 = chirp_templates(np.linspace(1.0, 1.1, 64), 1.0, 2048, 1024.0)
    assert H1.shape == (128, 2048)
    _compare(lib, torch, H1, 0.9999, "call 1 (maximum size)")
    # ... call 2 is smaller, odd-shaped and rank-deficient: whatever call 1 left behind must not leak into it
    rng = np.random.default_rng(5)
    H2 = rng.standard_normal((37, 20)) @ rng.standard_normal((20, 513))
    _compare(lib, torch, H2, 0.999, "call 2 (37 x 513, rank 20)")
    # and once more the first problem: identical to its first answer
    _compare(lib, torch, H1, 0.9999, "call 3 (maximum size again)")


def test_noalloc_svd_rejects_what_it_cannot_hold():
    torch = _cuda()
    import paper_2511_04730_b200 as lib
    L = lib.binding._lib
    n = C.c_int32()
    d = torch.zeros(16, dtype=torch.float64, device="cuda")
    f = torch.zeros(16, dtype=torch.float32, device="cuda")
    assert L.lloid_svd_slice_noalloc(d.data_ptr(), 129, 4, 0.9999, 4, C.byref(n), f.data_ptr(), f.data_ptr(), None, None, None) == lib.LLOID_EINVAL
    assert "exceeds the fixed scratch" in lib.lloid_last_error()
    assert L.lloid_svd_slice_noalloc(d.data_ptr(), 4, 2049, 0.9999, 4, C.byref(n), f.data_ptr(), f.data_ptr(), None, None, None) == lib.LLOID_EINVAL
    host = np.zeros(16)
    assert L.lloid_svd_slice_noalloc(host.ctypes.data, 4, 4, 0.9999, 4, C.byref(n), f.data_ptr(), f.data_ptr(), None, None, None) == lib.LLOID_EINVAL
    assert "DEVICE pointer" in lib.lloid_last_error()
