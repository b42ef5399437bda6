"""TEST INFRASTRUCTURE -- float64 oracle of the SVD bank construction (Eq. 3): truncated singular value
decomposition of one time slice's template matrix through numpy.linalg.svd (the library routine IS the definition).

    H (2M x N) = V diag(sigma) U ;  keep the smallest L with sum_{l<L} sigma_l^2 >= energy * sum sigma^2 ;
    basis U_L = first L rows of U (orthonormal),  reconstruction R_L = V[:, :L] diag(sigma_L)  (readings 4, 5).
"""
import numpy as np


def svd_slice(H: np.ndarray, energy: float = 0.9999):
    """-> (U [L][N], R [2M][L], sigma [L], kept_energy)."""
    H = np.asarray(H, dtype=np.float64)
    V, s, U = np.linalg.svd(H, full_matrices=False)
    e = np.cumsum(s ** 2)
    L = int(np.searchsorted(e, energy * e[-1] * (1.0 - 1e-15)) + 1)
    L = min(L, len(s))
    return U[:L], V[:, :L] * s[:L], s[:L], float(e[L - 1] / e[-1])
