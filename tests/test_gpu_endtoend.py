"""End-to-end parity a10 -> a7 -> a8 ("higher-degree reference"; VERDICT r1 task 2): the low
modes come from the library's OWN eigen-solver (nd_lowmodes_compute with the dynamic choice of l), go into
nd_set_lowmodes, and nd_apply_DN is compared with a reference that uses NO projection at all:

  * 4^4:    the exact D_N = c (1 + gamma5 sign(Q)) from the dense eigendecomposition of the oracle's Q;
  * 8^3x16: the oracle's sign_poly (eq. 2.5 alone) at a degree so high that its own delta is <= 1e-10 on the WHOLE spectrum
            (eps = lambda_min(Q^2)/||Q||^2 from a library Lanczos on the oracle's Q^2).

The statement under test is eq. 2.12 at m = 0 together with eq. 2.6: the projected operator deviates from
the exact one by at most  c (delta + 2 (b_+ + b_-)) ||eta||,  b_+- = the bound (2.10) on ||P_+- - (P_+-)_exact|| (to first
order kappa_+-).  An eigen-solver that returns a wrong projector (round 1 at 16^3x32: kappa ~ 29) fails this test."""
import numpy as np
import pytest

from lattice_inputs import gaussian_spinor
from oracle import lowmodes as olow
from oracle import sign as osign
from oracle import wilson, wilson_c
from tests.gpu_common import make_context

pytestmark = pytest.mark.gpu

RHO = 1.6
M = -RHO
PREF = 1.0 / RHO
QNORM = abs(4.0 + M) + 4.0


def gpu_DN_with_own_modes(ctx, eta, lo, hi, guard, bound_tol, n, degree, maxit=80):
    u, nu, resid, st = ctx.lowmodes_compute(lo, M, tol=bound_tol, maxit=maxit, lextra=guard, degree=degree, l_max=hi, stop="bound")
    assert st["converged"], st
    eps = 0.99 * float((nu ** 2).max()) / QNORM ** 2          # DESIGN.md R11
    c = osign.cheb_coeffs(n, eps)
    delta = osign.measure_delta(c, eps)
    ctx.set_sign_poly(c, eps, QNORM, M)
    ctx.set_lowmodes(u, nu)
    x, out, work = ctx.pack_spinor(eta), ctx.new_spinor(), ctx.new_spinor(3)
    ctx.apply_DN(out, x, PREF, work, use_graph=True)
    return ctx.unpack_spinor(out), delta, st


def test_4x4_solver_modes_vs_exact_dense_sign(dense_4x4_smooth):
    d = dense_4x4_smooth
    ctx, U = make_context(d["dims"], 64, 12, -1, "smooth", eps=0.3)
    eta = gaussian_spinor(d["dims"])
    got, delta, st = gpu_DN_with_own_modes(ctx, eta, 6, 14, 8, 1e-8, n=60, degree=30)
    lam, W = d["lam"], d["W"]
    S = (W * np.sign(lam)) @ W.conj().T
    exact = PREF * (eta + wilson.apply_gamma5((S @ eta.reshape(-1)).reshape(eta.shape)))
    err = np.linalg.norm((got - exact).ravel())
    tol = PREF * (delta + 2.0 * float(st["bound"].sum())) * np.linalg.norm(eta.ravel())
    assert 1e-9 < delta < 1e-4 and err <= tol, (err, tol, delta, st["bound"])
    assert err >= 1e-4 * PREF * delta * np.linalg.norm(eta.ravel())     # not vacuous: the polynomial error is really there


def test_8c16_solver_modes_vs_projection_free_reference():
    dims = (16, 8, 8, 8)
    ctx, U = make_context(dims, 64, 12, -1, "smooth", eps=0.3)
    Q = wilson_c.make_Q(U, M, -1)
    eta = gaussian_spinor(dims)
    got, delta, st = gpu_DN_with_own_modes(ctx, eta, 16, 24, 8, 1e-7, n=100, degree=60)
    # projection-free reference: eps from the lowest eigenvalue of the oracle's Q^2 (library Lanczos), delta_ref <= 1e-10
    theta, _, _ = olow.lowest_modes_eigsh(Q, dims + (4, 3), 2, tol=1e-8, ncv=64)
    eps_ref = 0.98 * theta[0] / QNORM ** 2
    n_ref = 200
    c_ref = osign.cheb_coeffs(n_ref, eps_ref)
    delta_ref = osign.measure_delta(c_ref, eps_ref)
    assert delta_ref <= 1e-10, delta_ref
    ref = osign.apply_DN(Q, wilson.apply_gamma5, eta, c_ref, eps_ref, QNORM, PREF)
    err = np.linalg.norm((got - ref).ravel())
    tol = PREF * (delta + delta_ref + 2.0 * float(st["bound"].sum())) * np.linalg.norm(eta.ravel())
    assert 1e-9 < delta < 1e-5 and err <= tol, (err, tol, delta, st["bound"])
    # the library's lowest |nu| agrees with the Lanczos value the reference's eps was taken from
    assert abs(float((st["nu_block"] ** 2).min()) - theta[0]) <= 1e-6
