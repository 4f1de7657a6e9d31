"""Normal-mode transformation of the oracle (test infrastructure; see oracle/__init__.py).

PAPER.md:L429-448 (Appendix B, Eqs. B1-B3).  B1 is garbled in the extracted text (the cosine
range is printed "1 <= i <= floor(n/2)", overlapping the i = n/2 row; the index line reads
"i = 0..n-1" where the bead index j is meant).  DESIGN R-2 fixes the reading used here:

  row k = mode, column j = bead, j = 0..P-1
    k = 0            : 1/sqrt(P)
    1 <= k < P/2     : sqrt(2/P) cos(2 pi k j / P)
    k = P/2 (P even) : (-1)^j / sqrt(P)
    P/2 < k <= P-1   : sqrt(2/P) sin(2 pi k j / P)

lambda_k = 4 sin^2(k pi / P) (Eq. B2) are the eigenvalues of the ring Laplacian that M
diagonalises, with lambda_k belonging to row k (L441 calls them "eigenvalues of M").
"""
import math
import numpy as np

from .constants import HBAR, KB


def nm_matrix(P):
    """The orthogonal matrix M of Eq. B1 as a (P, P) float64 array, written
    out entry by entry."""
    M = np.zeros((P, P), dtype=np.float64)
    for k in range(P):
        for j in range(P):
            if k == 0:
                M[k, j] = 1.0 / math.sqrt(P)
            elif P % 2 == 0 and k == P // 2:
                M[k, j] = (1.0 if j % 2 == 0 else -1.0) / math.sqrt(P)
            elif 2 * k < P:
                M[k, j] = math.sqrt(2.0 / P) * math.cos(2.0 * math.pi * k * j / P)
            else:
                M[k, j] = math.sqrt(2.0 / P) * math.sin(2.0 * math.pi * k * j / P)
    return M


def lambdas(P):
    """lambda_k = 4 sin^2(k pi / P), k = 0..P-1 (Eq. B2)."""
    return np.array([4.0 * math.sin(k * math.pi / P) ** 2 for k in range(P)], dtype=np.float64)


def omega_P(P, T):
    """omega_n = n / (beta hbar), beta = 1/(k_B T) (Eq. 2); in 1/ps."""
    return P * KB * T / HBAR


def omegas(P, T):
    """omega_k = sqrt(lambda_k) omega_n."""
    return np.sqrt(lambdas(P)) * omega_P(P, T)


def to_nm(M, a):
    """a~_k = sum_j M_kj a_j over the leading (bead) axis of a [P, ...] (Eq. B1)."""
    return np.tensordot(M, a, axes=(1, 0))


def from_nm(M, a):
    """a_j = sum_k M_kj a~_k  (Eq. B3: M^-1 = M^T)."""
    return np.tensordot(M.T, a, axes=(1, 0))
