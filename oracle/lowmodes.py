"""Oracle (test infrastructure): the low-lying modes of Q^2, section 2.3 (L77-93).

"The spectrum of Q in the vicinity of the origin can be reliably determined by minimizing the Ritz
functional of Q^2" - what is determined is the set of the l lowest eigenpairs of Q^2.
The oracle therefore takes the plain definition: a dense Hermitian eigendecomposition where that is
possible (4^4), a library Lanczos (`scipy.sparse.linalg.eigsh`) on the oracle's own Q^2 otherwise.
Eigenvectors are unique only up to rotations inside (near-)degenerate clusters, so tests compare
eigenvalues, residues and projector actions, never raw vectors (reading R10).
"""
import numpy as np


def lowest_modes_dense(Qmat, l):
    """l lowest eigenpairs of Q^2 from the dense matrix of Q: Q = W Lambda W^dagger => Q^2 has the same
    eigenvectors with eigenvalues Lambda^2.  Returns (theta[l] ascending, V[N, l])."""
    lam, W = np.linalg.eigh(Qmat)
    order = np.argsort(lam * lam)[:l]
    return (lam[order] ** 2), W[:, order]


def lowest_modes_eigsh(Q, shape, l, tol=1e-10, ncv=None, seed=7, maxiter=None):
    """l lowest eigenpairs of Q^2 by library Lanczos on the callable Q (shape = field shape)."""
    from scipy.sparse.linalg import LinearOperator, eigsh

    n = int(np.prod(shape))
    count = [0]

    def mv(x):
        count[0] += 2
        return Q(Q(x.reshape(shape))).reshape(n)

    op = LinearOperator((n, n), matvec=mv, dtype=np.complex128)
    rng = np.random.Generator(np.random.PCG64(seed))
    v0 = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    theta, vec = eigsh(op, k=l, which="SA", tol=tol, ncv=ncv, v0=v0, maxiter=maxiter)
    order = np.argsort(theta)
    return theta[order], [vec[:, i].reshape(shape) for i in order], count[0]


def orthonormalise(V):
    """Modified Gram-Schmidt (twice) on a list of vectors."""
    out = []
    for v in V:
        w = v.copy()
        for _ in range(2):
            for u in out:
                w = w - np.vdot(u.reshape(-1), w.reshape(-1)) * u
        out.append(w / np.linalg.norm(w.reshape(-1)))
    return out


def approximate_low_space(Q, shape, l, qnorm, cut, degree=24, sweeps=3, seed=11):
    """A cheap, APPROXIMATE low-mode space of Q^2 for the large lattices where a converged CPU
    eigen-solve takes too long: `sweeps` rounds of a degree-`degree` Chebyshev filter in Q^2 that damps
    the interval [cut, qnorm^2], each followed by orthonormalisation.  The result is an orthonormal set
    V that is only roughly invariant under Q; eq. 2.11 is well defined for ANY orthonormal V (its
    Rayleigh-Ritz pairs (nu_k, u_k) are then inputs shared by oracle and CUDA path), so this is an
    input-preparation step for the D_N parity test at 16^3x32, not a statement about eigenvectors."""
    rng = np.random.Generator(np.random.PCG64(seed))
    V = [rng.standard_normal(shape) + 1j * rng.standard_normal(shape) for _ in range(l)]
    V = orthonormalise(V)
    a, b = cut, qnorm * qnorm
    e, c0 = (b - a) / 2.0, (b + a) / 2.0

    def filt(v):
        # T_degree((Q^2 - c0)/e) v by the three-term recurrence
        t0 = v
        t1 = (Q(Q(v)) - c0 * v) / e
        for _ in range(degree - 1):
            t0, t1 = t1, 2.0 * (Q(Q(t1)) - c0 * t1) / e - t0
        return t1

    for _ in range(sweeps):
        V = orthonormalise([filt(v) for v in V])
    return V


# ----------------------------------------------------------------------------- error control, eq. 2.8-2.10
def distances_d(nu, spectrum_rest):
    """d_k of PAPER.md:L90: the distance of nu_k from the spectrum of Q in the subspace orthogonal to the range of
    (P_+)_exact if nu_k > 0, of (P_-)_exact if nu_k < 0.  `spectrum_rest` = the eigenvalues of Q NOT represented in
    V (all modes outside the l projected ones).  For nu_k > 0 the complement of range((P_+)_exact) carries those plus
    the projected NEGATIVE eigenvalues (approximated by the negative nu_j), and vice versa."""
    nu = np.asarray(nu, dtype=np.float64)
    rest = np.asarray(spectrum_rest, dtype=np.float64)
    d = np.empty_like(nu)
    for k, v in enumerate(nu):
        other = nu[nu < 0] if v > 0 else nu[nu > 0]
        cand = np.concatenate([rest, other])
        d[k] = np.min(np.abs(cand - v))
    return d


def kappa_pm(nu, rho, d):
    """kappa_+-^2 = sum_{+-nu_k > 0} rho_k^2 / d_k^2 (eq. 2.9).  Returns (kappa_+, kappa_-)."""
    nu, rho, d = (np.asarray(a, dtype=np.float64) for a in (nu, rho, d))
    kp = np.sqrt(np.sum((rho[nu > 0] / d[nu > 0]) ** 2))
    km = np.sqrt(np.sum((rho[nu < 0] / d[nu < 0]) ** 2))
    return float(kp), float(km)


def projector_bound(kappa):
    """|| P_+- - (P_+-)_exact || <= kappa (1 + 2 kappa) / (1 - 2 kappa (1 + 2 kappa)) (eq. 2.10);
    +inf when the denominator is not positive (the bound says nothing there)."""
    x = 2.0 * kappa * (1.0 + 2.0 * kappa)
    return float(kappa * (1.0 + 2.0 * kappa) / (1.0 - x)) if x < 1.0 else float("inf")


# ----------------------------------------------------------------------------- dynamic choice of l
def choose_l(abs_nu, l_min, l_max):
    """"The number of low modes included in the projector will be determined dynamically in such a way that the
    spectral distance from the other modes is not accidentally small".  Reading (R17): given
    the ascending moduli a_1 <= a_2 <= ... of the Ritz values of Q in the block (projected candidates AND guard vectors),
    the cut l' in [l_min, l_max] is put at the LARGEST gap a_{l'+1} - a_{l'}; ties go to the smallest l'.
    Needs len(abs_nu) >= l_max + 1 (at least one value beyond the last candidate)."""
    a = np.asarray(abs_nu, dtype=np.float64)
    assert np.all(np.diff(a) >= 0) and 1 <= l_min <= l_max < len(a)
    best, best_gap = l_min, -1.0
    for l in range(l_min, l_max + 1):
        gap = a[l] - a[l - 1]
        if gap > best_gap:
            best, best_gap = l, gap
    return best, best_gap


def error_control(nu_block, rho_block, l_min, l_max):
    """The whole error control of PAPER.md:L86-110 on a block of Ritz pairs (nu_j, u_j) of Q with their residues rho_j
    (eq. 2.8), ordered by the modulus estimate a_j = ||Q u_j|| = sqrt(nu_j^2 + rho_j^2) - for a converged pair a_j = |nu_j|;
    a spurious small Ritz value of the indefinite Q comes with a large residue and sorts to the end (R17).
    l' by `choose_l` on the a_j (made monotone by a running maximum: only unconverged guard pairs are affected); d_k (L90)
    from the moduli outside the cut, a_j for j >= l', taken with BOTH signs because a poorly converged guard vector does
    not fix its sign, and from the projected values of the opposite sign; kappa_+- (2.9); bound (2.10).
    Returns dict(l, gap, d, kappa, bound)."""
    nu = np.asarray(nu_block, dtype=np.float64)
    rho = np.asarray(rho_block, dtype=np.float64)
    a = np.maximum.accumulate(np.sqrt(nu * nu + rho * rho))
    l, gap = choose_l(a, l_min, l_max)
    rest = np.concatenate([a[l:], -a[l:]])
    d = distances_d(nu[:l], rest)
    kp, km = kappa_pm(nu[:l], rho[:l], d)
    return dict(l=l, gap=gap, d=d, kappa=(kp, km), bound=(projector_bound(kp), projector_bound(km)))
