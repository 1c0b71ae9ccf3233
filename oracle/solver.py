"""Oracle (test infrastructure): the massive Neuberger-Dirac operator and its inversion, PAPER.md:L115-118 (eq. 2.12)
and L146 ("inversion").

PAPER.md never writes D_N^m down; the bound (2.12), ||D~_N^m - D_N^m|| <= (2/a)(1 + s - a m/2)(kappa_+ + kappa_-),
fixes it (reading R16): an error E in sign(Q) (||E|| <= kappa_+ + kappa_-, eq. 2.10-2.11) enters
D_N = (1/abar)(1 + gamma5 sign(Q)) as (1/abar) gamma5 E, so the factor in front of D_N must be
abar (2/a)(1 + s - a m/2)/2... with abar = a/(1+s) this is (1 - abar m/2): the convention of the paper's ref. [10],
    D_N^m = (1 - abar m/2) D_N + m.
`DN` is any callable eta -> D_N eta built with prefactor 1/abar (oracle.sign.apply_DN or a dense matrix).
"""
import numpy as np


def apply_DNm(DN, eta, abar, mq):
    """D_N^m eta = (1 - abar mq/2) D_N eta + mq eta."""
    return (1.0 - 0.5 * abar * mq) * DN(eta) + mq * eta


def cg_normal_equations(D, Ddag, b, tol, maxit):
    """Textbook conjugate gradients on D^dagger D x = D^dagger b from x = 0 (Hestenes-Stiefel):
        r = D^dagger b, p = r;  alpha = <r,r>/<Dp,Dp>;  x += alpha p;  r -= alpha D^dagger D p;
        beta = <r',r'>/<r,r>;  p = r' + beta p;  stop when |r| <= tol |D^dagger b|.
    Returns (x, iterations, |b - D x| / |b|)."""
    x = np.zeros_like(b)
    r = Ddag(b)
    p = r.copy()
    rr = np.vdot(r.ravel(), r.ravel()).real
    stop = tol * tol * rr
    it = 0
    while it < maxit and rr > 0.0:
        t = D(p)
        q = Ddag(t)
        alpha = rr / np.vdot(t.ravel(), t.ravel()).real
        x = x + alpha * p
        r = r - alpha * q
        rn = np.vdot(r.ravel(), r.ravel()).real
        it += 1
        if rn <= stop:
            break
        p = r + (rn / rr) * p
        rr = rn
    res = np.linalg.norm((b - D(x)).ravel()) / np.linalg.norm(b.ravel())
    return x, it, float(res)
