"""CPU pins of oracle/svd_oracle.py (SVD bank construction): closed forms and the properties the north star
names (orthonormality to 1e-12, residual = 1 - kept energy)."""
import numpy as np

from oracle import svd_slice


def test_rank_two_closed_form():
    rng = np.random.default_rng(0)
    u1 = rng.standard_normal(50); u1 /= np.linalg.norm(u1)
    u2 = rng.standard_normal(50); u2 -= u1 * (u1 @ u2); u2 /= np.linalg.norm(u2)
    v1 = rng.standard_normal(8); v1 /= np.linalg.norm(v1)
    v2 = rng.standard_normal(8); v2 -= v1 * (v1 @ v2); v2 /= np.linalg.norm(v2)
    H = 5.0 * np.outer(v1, u1) + 0.5 * np.outer(v2, u2)
    U, R, s, kept = svd_slice(H, 1.0)
    assert len(s) == 2 and np.allclose(s, [5.0, 0.5], rtol=1e-13)
    assert abs(abs(U[0] @ u1) - 1) < 1e-13 and abs(abs(U[1] @ u2) - 1) < 1e-13
    assert np.allclose(R @ U, H, atol=1e-13)
    U, R, s, kept = svd_slice(H, 0.98)                       # 25 / 25.25 = 0.990 >= 0.98: one filter is enough
    assert len(s) == 1 and abs(kept - 25.0 / 25.25) < 1e-14


def test_orthonormality_residual_and_truncation_rule_on_a_chirp_slice():
    from workloads import chirp_templates
    H = chirp_templates(np.linspace(1.0, 1.2, 24), 0.5, 2048, 1024.0)
    U, R, s, kept = svd_slice(H, 0.9999)
    assert np.abs(U @ U.T - np.eye(len(s))).max() < 1e-12                       # north star: orthonormal to 1e-12
    res = np.linalg.norm(H - R @ U) ** 2 / np.linalg.norm(H) ** 2
    assert abs(res - (1.0 - kept)) < 1e-12 and kept >= 0.9999                   # residual energy = 1 - kept energy
    s_all = np.linalg.svd(H, compute_uv=False)
    assert np.sum(s_all[:len(s) - 1] ** 2) < 0.9999 * np.sum(s_all ** 2)        # one filter fewer would not be enough
    # the same subspace as the eigenvectors of the Gram matrix (an independent route)
    w, Q = np.linalg.eigh(H @ H.T)
    assert np.allclose(np.sort(w)[::-1][:len(s)], s ** 2, rtol=1e-9)
