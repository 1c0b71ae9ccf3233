"""Oracle (test infrastructure): the index of the Neuberger-Dirac operator by zero-mode counting ("the
calculation of the index of our Neuberger-Dirac operator via zero-mode counting [7]").

D_N = c (1 + gamma5 sign(Q)) (eq. 2.4) obeys the Ginsparg-Wilson relation, so its zero modes have definite chirality;
    index = n_+ - n_-,   n_+- = number of zero modes with gamma5 psi = +-psi.
The plain definition, on a lattice small enough for dense algebra: build D_N with the EXACT sign function from the dense
eigendecomposition of Q, take the null space of D_N^dagger D_N, count the chiralities.  D_N^dagger D_N commutes with
gamma5, and on the sector gamma5 = sigma it equals 2 c^2 (1 + sigma P_sigma S P_sigma), P_sigma = (1 + sigma gamma5)/2:
this is the operator whose lowest eigenvalues the CUDA path computes sector by sector; `sector_spectrum` gives them densely.
"""
import numpy as np


def gamma5_diag(nsites):
    """gamma5 = diag(1,1,-1,-1) on spin (chiral basis, R2), identity on colour: the diagonal for [site][spin][colour]."""
    return np.tile(np.repeat(np.array([1.0, 1.0, -1.0, -1.0]), 3), nsites)


def exact_sign(Qmat):
    lam, W = np.linalg.eigh(0.5 * (Qmat + Qmat.conj().T))
    return (W * np.sign(lam)) @ W.conj().T, lam


def zero_mode_count(Qmat, c=1.0, tol=1e-8):
    """(n_plus, n_minus) of D_N = c (1 + gamma5 S): eigenvectors of D^dagger D with eigenvalue <= tol c^2, sorted into
    chiralities by <v, gamma5 v> (which is +-1 on them up to rounding, else the count is refused)."""
    S, _ = exact_sign(Qmat)
    n = Qmat.shape[0]
    g5 = gamma5_diag(n // 12)
    D = c * (np.eye(n) + g5[:, None] * S)
    w, v = np.linalg.eigh(D.conj().T @ D)
    zero = v[:, w <= tol * c * c]
    if zero.shape[1] == 0:
        return 0, 0
    # the null space may mix chiralities only if both are present: diagonalise gamma5 inside it
    chi = np.linalg.eigvalsh(zero.conj().T @ (g5[:, None] * zero))
    assert np.all(np.abs(np.abs(chi) - 1.0) < 1e-6), chi
    return int(np.sum(chi > 0)), int(np.sum(chi < 0))


def index(Qmat, c=1.0):
    np_, nm = zero_mode_count(Qmat, c)
    return np_ - nm


def sector_spectrum(Qmat, sigma):
    """Eigenvalues (ascending) of B_sigma = 1 + sigma P_sigma S P_sigma restricted to the chirality sector sigma = +-1:
    D_N^dagger D_N / (2 c^2) on that sector; zero modes of D_N of chirality sigma are its zero eigenvalues."""
    S, _ = exact_sign(Qmat)
    g5 = gamma5_diag(Qmat.shape[0] // 12)
    keep = np.flatnonzero(g5 == sigma)
    B = np.eye(len(keep)) + sigma * S[np.ix_(keep, keep)]
    return np.linalg.eigvalsh(0.5 * (B + B.conj().T))
