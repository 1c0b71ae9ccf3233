"""Oracle (test infrastructure): SU(3) link compression, PAPER.md:L46-50 (section 2.1, eq. 2.3).

12 parameters (eq. 2.3): keep two columns a, b of U = (a b c); c = (a x b)^*.
The same identity holds for rows of an SU(3) matrix (U^T is also SU(3)); both are provided.

8 parameters (PAPER.md:L46 only points to refs [3, 9]; the formula is absent - DESIGN.md reading R8):
with ROWS a, b, c of U store the complex numbers a2, a3, b1 and the phases theta1 = arg a1,
theta2 = arg c1 (3*2 + 2 = 8 reals).  Reconstruction, N = |a2|^2 + |a3|^2:
    a1 = sqrt(1 - N) e^{i theta1}                    (row a has unit norm)
    c1 = sqrt(N - |b1|^2) e^{i theta2}               (column 1 has unit norm: |a1|^2+|b1|^2+|c1|^2 = 1)
    b2 = -(a1^* a2 b1 + a3^* c1^*) / N      b3 = (a2^* c1^* - a1^* a3 b1) / N
    c2 = (a3^* b1^* - a1^* a2 c1) / N       c3 = -(a2^* b1^* + a1^* a3 c1) / N
(derivation: b and c are orthogonal to a and to each other, and det U = 1).  Singular as N -> 0, which
includes unit links.

Arrays: U[..., row, col] complex128.
"""
import numpy as np


def compress12_cols(U):
    """eq. 2.3: the two columns a = U[:,0], b = U[:,1] -> [..., 2, 3]."""
    return np.stack([U[..., :, 0], U[..., :, 1]], axis=-2)


def reconstruct12_cols(ab):
    a, b = ab[..., 0, :], ab[..., 1, :]
    c = np.conj(np.cross(a, b))                 # c = (a x b)^*, eq. 2.3
    return np.stack([a, b, c], axis=-1)


def compress12_rows(U):
    return U[..., :2, :].copy()


def reconstruct12_rows(ab):
    a, b = ab[..., 0, :], ab[..., 1, :]
    c = np.conj(np.cross(a, b))
    return np.stack([a, b, c], axis=-2)


def compress8(U):
    """-> (z[..., 3] complex = (a2, a3, b1), theta[..., 2] real = (arg a1, arg c1)), rows a, b, c."""
    z = np.stack([U[..., 0, 1], U[..., 0, 2], U[..., 1, 0]], axis=-1)
    th = np.stack([np.angle(U[..., 0, 0]), np.angle(U[..., 2, 0])], axis=-1)
    return z, th


def reconstruct8(z, th):
    a2, a3, b1 = z[..., 0], z[..., 1], z[..., 2]
    N = np.abs(a2) ** 2 + np.abs(a3) ** 2
    a1 = np.sqrt(np.maximum(1.0 - N, 0.0)) * np.exp(1j * th[..., 0])
    c1 = np.sqrt(np.maximum(N - np.abs(b1) ** 2, 0.0)) * np.exp(1j * th[..., 1])
    cj = np.conj
    b2 = -(cj(a1) * a2 * b1 + cj(a3) * cj(c1)) / N
    b3 = (cj(a2) * cj(c1) - cj(a1) * a3 * b1) / N
    c2 = (cj(a3) * cj(b1) - cj(a1) * a2 * c1) / N
    c3 = -(cj(a2) * cj(b1) + cj(a1) * a3 * c1) / N
    U = np.stack([np.stack([a1, a2, a3], -1), np.stack([b1, b2, b3], -1), np.stack([c1, c2, c3], -1)], -2)
    return U


def recon8_min_N(U):
    """Smallest N = |a2|^2+|a3|^2 over the field: the conditioning of the 8-parameter form."""
    return float(np.min(np.abs(U[..., 0, 1]) ** 2 + np.abs(U[..., 0, 2]) ** 2))
