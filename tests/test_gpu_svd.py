"""GPU parity of lloid_svd_slice (one-sided Jacobi SVD on the GPU) against oracle/svd_oracle.py (-m gpu)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _cuda():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def _check(H, energy, tag):
    import paper_2511_04730_b200 as lib
    from oracle import svd_slice
    U, R, s, kept = lib.binding.lloid_svd_slice(H, energy)
    Uo, Ro, so, kepto = svd_slice(H, energy)
    assert len(s) == len(so), (tag, len(s), len(so))
    assert np.abs(s / so - 1).max() < 1e-10 and abs(kept - kepto) < 1e-12
    L = len(s)
    assert np.abs(U.astype(np.float64) @ U.T - np.eye(L)).max() < 2e-6          # fp32 outputs
    # singular vectors are unique up to sign / rotations inside clusters: compare the subspace and the unique product
    C = U.astype(np.float64) @ Uo.T
    assert np.abs(C @ C.T - np.eye(L)).max() < 1e-5
    scale = np.abs(H).max()
    err = np.abs(R.astype(np.float64) @ U - Ro @ Uo).max() / scale
    print(f"{tag}: {H.shape} -> L = {L}, sigma rel err {np.abs(s / so - 1).max():.1e}, product err {err:.1e}")
    assert err < 5e-6
    return U, R


def test_svd_of_chirp_slices_against_the_oracle():
    _cuda()
    from workloads import chirp_templates
    # full-rate slice of a 120-template bank (rank-deficient: 240 rows of strongly correlated chirps)
    H = chirp_templates(np.linspace(1.0, 1.1, 120), 0.5, 2048, 1024.0)
    _check(H, 0.9999, "chirps 0.5 s")
    _check(H[:, 200:713], 0.999, "odd shapes")                                   # N = 513
    _check(H[:7], 1.0, "odd row count, full rank")                               # n = 7 -> padded to 8
    rng = np.random.default_rng(3)
    _check(rng.standard_normal((64, 40)), 1.0, "more rows than taps")             # rank 40 < 64 rows


def test_gpu_built_bank_filters_like_the_oracle_built_one():
    """A bank whose slices are decomposed ON THE GPU goes through the stream; its SNR equals the float64 LLOID oracle's SNR
    for that same bank (gate 2e-3) and the SNR of the numpy-built bank up to the truncation residual."""
    _cuda()
    import paper_2511_04730_b200 as lib
    from oracle import lloid_snr
    from workloads import Bank, Slice, bank_from_layout, make_strain, slice_template_matrices
    f0 = 2048
    mc = np.linspace(1.3, 1.5, 30)
    lay = [(2048, 0, 1024), (1024, 1024, 3072), (512, 3072, 8192)]
    ref_bank = bank_from_layout(mc, 4.0, lay, f0=f0)
    slices = []
    for (rate, s0, e0), Hs, sl in zip(lay, slice_template_matrices(mc, 4.0, lay, f0=f0), ref_bank.slices):
        U, R, s, kept = lib.binding.lloid_svd_slice(Hs, 0.9999)
        assert U.shape[0] == sl.n_basis and abs(kept - sl.kept_energy) < 1e-9
        slices.append(Slice(rate=rate, n_taps=sl.n_taps, delay=sl.delay, U=U.astype(np.float64), R=R.astype(np.float64), kept_energy=kept))
    bank = Bank(f0=f0, M=len(mc), slices=slices, mchirp=mc, T=4.0).as_f32()
    strain = make_strain(77, 6 * f0)[None]
    st = lib.LloidStream([bank], 1, 2048)
    rho = np.concatenate([st.push(strain[:, p * 2048:(p + 1) * 2048], want_snr_bank=0)[1][0] for p in range(6)], axis=1)
    st.close()
    ref = lloid_snr(bank, strain[0])
    rms = np.sqrt(np.mean(ref ** 2) * 2)
    assert np.abs(rho - ref).max() / rms < 2e-3
    ref2 = lloid_snr(ref_bank.as_f32(), strain[0])
    assert np.abs(ref - ref2).max() / rms < 1e-4          # same rank-L approximation of H up to fp32 rounding of U, R
