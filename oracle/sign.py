"""Oracle (test infrastructure): Chebyshev approximation of sign(Q), the projected sign function and the
Neuberger-Dirac operator, section 2.2-2.3 (L54-118), followed step by step.

    D_N = (1 + gamma5 sign(Q)) / abar,   Q = gamma5 (a D_W - 1 - s)                          (2.4)
    sign(Q) ~ X P_n(X^2),  X = Q/||Q||,  P_n(y) = sum_{k=0}^n c_k T_k(.)                     (2.5)
    delta = max_{eps<=y<=1} |1 - sqrt(y) P(y)|                                               (2.6)
    P_+- = sum_{nu_k ><0} u_k (x) u_k^dagger,   PP Q u_k = nu_k u_k                           (2.7)
    sign(Q) ~ P_+ - P_- + (1 - P_+ - P_-) X P_n(X^2)                                        (2.11)

Readings: R4 the kernel mass is m = -(1+s) = -rho; R5 the prefactor 1/abar is an
explicit scalar `c`; R6 ||Q|| is an input `qnorm` >= the true norm; R7 T_k is evaluated at
z = (2y - 1 - eps)/(1 - eps) and c_0 is NOT halved, coefficients = Chebyshev interpolation of
y^{-1/2} at the n+1 Chebyshev nodes, delta is measured; R9 Clenshaw on vectors as written in
`clenshaw_P`; R12 projector applied after the polynomial, literally as eq. 2.11.

The operator enters only through the callable `Q(psi) -> psi` (e.g. a closure over oracle.wilson.apply_Q
or the plain-C oracle); vectors are complex128 arrays of any shape.
"""
import numpy as np


# ----------------------------------------------------------------------------- coefficients, eq. 2.5-2.6
def cheb_coeffs(n, eps):
    """c_0..c_n with P(y) = sum_k c_k T_k(z(y)), z = (2y-1-eps)/(1-eps), interpolating y^{-1/2} at the
    n+1 zeros of T_{n+1} in z (reading R7).  long double accumulation."""
    ld = np.longdouble
    j = np.arange(n + 1, dtype=ld)
    theta = ld(np.pi) * (j + ld(0.5)) / ld(n + 1)
    z = np.cos(theta)
    y = (ld(1.0 - eps) * z + ld(1.0 + eps)) / ld(2.0)
    f = ld(1.0) / np.sqrt(y)
    k = np.arange(n + 1, dtype=ld)
    c = (ld(2.0) / ld(n + 1)) * (np.cos(np.outer(k, theta)) @ f)
    c[0] = c[0] / ld(2.0)          # full c_0 convention: P = sum_{k=0}^n c_k T_k (eq. 2.5 as printed)
    return np.asarray(c, dtype=np.float64)


def z_of_y(y, eps):
    return (2.0 * y - 1.0 - eps) / (1.0 - eps)


def eval_P_scalar(c, eps, y):
    """Scalar Clenshaw for P(y) = sum c_k T_k(z): b_k = c_k + 2 z b_{k+1} - b_{k+2}; P = c_0 + z b_1 - b_2."""
    z = z_of_y(np.asarray(y, dtype=np.float64), eps)
    b1 = np.zeros_like(z)
    b2 = np.zeros_like(z)
    for k in range(len(c) - 1, 0, -1):
        b1, b2 = c[k] + 2.0 * z * b1 - b2, b1
    return c[0] + z * b1 - b2


def measure_delta(c, eps, npts=200001):
    """delta of eq. 2.6 measured on a geometric + a linear grid of [eps, 1] (reading R7)."""
    y = np.concatenate([np.geomspace(eps, 1.0, npts), np.linspace(eps, 1.0, npts)])
    return float(np.max(np.abs(1.0 - np.sqrt(y) * eval_P_scalar(c, eps, y))))


# ----------------------------------------------------------------------------- polynomial on vectors
def clenshaw_P(Q, eta, c, eps, qnorm):
    """P_n(X^2) eta by the Clenshaw recurrence (reading R9), X = Q/qnorm:
        Z = alpha Q^2 + beta,  alpha = 2/((1-eps) qnorm^2),  beta = -(1+eps)/(1-eps)      [Z = z(X^2)]
        b_n = c_n eta, b_{n+1} = 0;   b_k = c_k eta + 2 Z b_{k+1} - b_{k+2}  (k = n-1..1)
        P eta = c_0 eta + Z b_1 - b_2
    n applications of Q^2."""
    n = len(c) - 1
    alpha = 2.0 / ((1.0 - eps) * qnorm * qnorm)
    beta = -(1.0 + eps) / (1.0 - eps)

    def Z(v):
        return alpha * Q(Q(v)) + beta * v

    if n == 0:
        return c[0] * eta
    b1 = c[n] * eta                # b_n
    b2 = np.zeros_like(eta)        # b_{n+1}
    for k in range(n - 1, 0, -1):
        b1, b2 = c[k] * eta + 2.0 * Z(b1) - b2, b1
    return c[0] * eta + Z(b1) - b2


def sign_poly(Q, eta, c, eps, qnorm):
    """sign(Q) eta ~ X P_n(X^2) eta (eq. 2.5): 2n+1 applications of Q."""
    return Q(clenshaw_P(Q, eta, c, eps, qnorm)) / qnorm


# ----------------------------------------------------------------------------- low modes, eq. 2.7-2.8, 2.11
def vdot(a, b):
    return np.vdot(a.reshape(-1), b.reshape(-1))


def rayleigh_ritz_Q(Q, V):
    """PP Q u_k = nu_k u_k: V = list of l orthonormal vectors spanning the low-mode space;
    diagonalise the l x l Hermitian matrix M_ij = <v_i, Q v_j>, rotate back.  Returns (nu[l] ascending,
    U = list of l vectors)."""
    l = len(V)
    QV = [Q(v) for v in V]
    M = np.array([[vdot(V[i], QV[j]) for j in range(l)] for i in range(l)])
    M = 0.5 * (M + M.conj().T)
    nu, W = np.linalg.eigh(M)
    U = [sum(W[i, k] * V[i] for i in range(l)) for k in range(l)]
    return nu, U


def residues(Q, nu, U):
    """rho_k = ||(Q - nu_k) u_k|| (eq. 2.8)."""
    return np.array([np.linalg.norm((Q(u) - n * u).reshape(-1)) for n, u in zip(nu, U)])


def sign_projected(Q, eta, c, eps, qnorm, nu, U):
    """eq. 2.11 literally (reading R12):
        sign(Q) eta ~ sum_k sign(nu_k) u_k <u_k, eta> + (1 - sum_k u_k u_k^dagger) [X P_n(X^2) eta]."""
    chi = sign_poly(Q, eta, c, eps, qnorm)
    s = np.zeros_like(eta)
    for n, u in zip(nu, U):
        s = s + np.sign(n) * vdot(u, eta) * u
    for u in U:
        chi = chi - vdot(u, chi) * u
    return s + chi


def apply_DN(Q, gamma5, eta, c, eps, qnorm, prefactor, nu=None, U=None):
    """D_N eta = prefactor * (eta + gamma5 sign(Q) eta) (eq. 2.4; `prefactor` = 1/abar, R5)."""
    if U is None or len(U) == 0:
        s = sign_poly(Q, eta, c, eps, qnorm)
    else:
        s = sign_projected(Q, eta, c, eps, qnorm, nu, U)
    return prefactor * (eta + gamma5(s))



# ----------------------------------------------------------------------------- min-max coefficients, eq. 2.6
def minmax_coeffs(n, eps, max_iter=60, tol=1e-3):
    """The polynomial that MINIMISES delta = max_{eps<=y<=1} |1 - sqrt(y) P(y)| (eq. 2.6: "minmax
    polynomials"), by the Remez exchange algorithm for the weighted problem  w(y) (f(y) - P(y)),  f = y^{-1/2}, w = y^{1/2}:
      1. reference y_0 < ... < y_{n+1} (start: the extrema of T_{n+1} in z);
      2. solve  sum_k c_k T_k(z_i) + (-1)^i E / w(y_i) = f(y_i),  i = 0..n+1,  for (c_0..c_n, E)   [long double elimination];
      3. new reference = the alternating local extrema of the error e(y) = 1 - sqrt(y) P(y) on a fine grid;
      repeat until max|e| <= (1 + tol) |E|  (de la Vallee-Poussin: |E| <= delta_min <= max|e|).
    Same conventions as cheb_coeffs (z = (2y-1-eps)/(1-eps), full c_0).  Returns (c[0..n], delta = max|e| measured, |E|)."""
    ld = np.longdouble
    m = n + 2
    i = np.arange(m, dtype=ld)
    z = -np.cos(ld(np.pi) * i / ld(m - 1))                      # ascending in z: -1 .. 1
    # fine grid, Chebyshev-distributed in z (dense at both ends, where the extrema crowd)
    ng = 60 * m
    zg = -np.cos(np.pi * (np.arange(ng) + 0.5) / ng)
    zg = np.concatenate([[-1.0], zg, [1.0]])
    yg = ((1.0 - eps) * zg + 1.0 + eps) / 2.0
    c = None
    E = ld(0)
    for _ in range(max_iter):
        y = (ld(1.0 - eps) * z + ld(1.0 + eps)) / ld(2.0)
        A = np.empty((m, m), dtype=ld)
        theta = np.arccos(np.clip(z, -1, 1))
        A[:, :n + 1] = np.cos(np.outer(theta, np.arange(n + 1, dtype=ld)))
        A[:, n + 1] = np.where(np.arange(m) % 2 == 0, ld(1), ld(-1)) / np.sqrt(y)
        b = ld(1.0) / np.sqrt(y)
        # Gaussian elimination with partial pivoting in long double
        M = np.concatenate([A, b[:, None]], axis=1)
        for k in range(m):
            p = k + int(np.argmax(np.abs(M[k:, k])))
            if p != k:
                M[[k, p]] = M[[p, k]]
            M[k + 1:] -= np.outer(M[k + 1:, k] / M[k, k], M[k])
        sol = np.empty(m, dtype=ld)
        for k in range(m - 1, -1, -1):
            sol[k] = (M[k, m] - M[k, k + 1:m] @ sol[k + 1:]) / M[k, k]
        c = np.asarray(sol[:n + 1], dtype=np.float64)
        E = sol[n + 1]
        e = 1.0 - np.sqrt(yg) * eval_P_scalar(c, eps, yg)
        emax = float(np.max(np.abs(e)))
        if emax <= (1.0 + tol) * abs(float(E)):
            break
        # alternating extrema: split the grid where the error changes sign, take the largest |e| of every piece
        sgn = np.sign(e)
        sgn[sgn == 0] = 1
        cuts = np.flatnonzero(sgn[1:] != sgn[:-1]) + 1
        pieces = np.split(np.arange(len(e)), cuts)
        ext = np.array([p[np.argmax(np.abs(e[p]))] for p in pieces])
        while len(ext) > m:                                       # drop the smaller end extremum until n+2 are left
            ext = ext[1:] if abs(e[ext[0]]) < abs(e[ext[-1]]) else ext[:-1]
        if len(ext) < m:
            break                                                 # (degree too high for this grid / precision)
        z = np.asarray(zg[ext], dtype=ld)
    delta = float(np.max(np.abs(1.0 - np.sqrt(yg) * eval_P_scalar(c, eps, yg))))
    return c, max(delta, measure_delta(c, eps, 100001)), abs(float(E))
