"""the massive operator D_N^m (R16) and its CG inversion on the CUDA path against the oracle's
operator and textbook CG with the same polynomial coefficients."""
import numpy as np
import pytest

from lattice_inputs import gaussian_spinor
from oracle import sign as osign
from oracle import solver as osolver
from oracle import wilson, wilson_c
from tests.gpu_common import assert_field_close, make_context, rel_l2, round_to

pytestmark = pytest.mark.gpu

RHO = 1.6
M = -RHO
QNORM = 6.4


def setup(prec, dims=(8, 4, 4, 8), n=60, eps=0.004):
    ctx, U = make_context(dims, prec, 12, -1, "smooth", eps=0.3)
    c = osign.cheb_coeffs(n, eps)
    ctx.set_sign_poly(c, eps, QNORM, M)
    ctx.set_lowmodes(None, [])
    Q = wilson_c.make_Q(U, M, -1)
    DN = lambda v: osign.apply_DN(Q, wilson.apply_gamma5, v, c, eps, QNORM, RHO)     # prefactor 1/abar = rho
    return ctx, DN


@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("mq", [0.0, 0.1, 0.5])
def test_apply_DNm(prec, mq):
    ctx, DN = setup(prec)
    eta = round_to(gaussian_spinor(ctx.dims), prec)
    out, work = ctx.new_spinor(), ctx.new_spinor(3)
    ctx.apply_DNm(out, ctx.pack_spinor(eta), RHO, mq, work, use_graph=True)
    ref = osolver.apply_DNm(DN, eta, 1.0 / RHO, mq)
    assert_field_close(ctx.unpack_spinor(out), ref, (1e-11 if prec == 64 else 1e-5), ctx=ctx)


def test_solve_fp64_matches_oracle_cg():
    ctx, DN = setup(64)
    mq, tol = 0.2, 1e-9
    b = gaussian_spinor(ctx.dims)
    x = ctx.new_spinor()
    relres, iters, ok = ctx.solve_DNm(x, ctx.pack_spinor(b), RHO, mq, tol=tol, maxit=300)
    assert ok and relres < 1e-7
    D = lambda v: osolver.apply_DNm(DN, v, 1.0 / RHO, mq)
    Dd = lambda v: wilson.apply_gamma5(D(wilson.apply_gamma5(v)))
    xr, itr, resr = osolver.cg_normal_equations(D, Dd, b, tol, 300)
    got = ctx.unpack_spinor(x)
    assert abs(iters - itr) <= 2
    assert rel_l2(got, xr) <= 1e-7
    assert np.linalg.norm((b - D(got)).ravel()) <= 1e-7 * np.linalg.norm(b.ravel())     # the oracle's operator agrees


def test_solve_fp32_and_failure_reporting():
    import paper_1010_5636_b200 as nd

    ctx, DN = setup(32)
    mq = 0.3
    b = round_to(gaussian_spinor(ctx.dims), 32)
    x, bd = ctx.new_spinor(), ctx.pack_spinor(b)
    relres, iters, ok = ctx.solve_DNm(x, bd, RHO, mq, tol=1e-4, maxit=200)
    assert ok and relres < 1e-3
    D = lambda v: osolver.apply_DNm(DN, v, 1.0 / RHO, mq)
    assert np.linalg.norm((b - D(ctx.unpack_spinor(x))).ravel()) <= 2e-3 * np.linalg.norm(b.ravel())
    relres2, iters2, ok2 = ctx.solve_DNm(x, bd, RHO, mq, tol=1e-12, maxit=2)     # cannot converge in 2 iterations
    assert not ok2 and iters2 == 2 and 0 < relres2 < 1
    with pytest.raises(nd.NDError):
        ctx.solve_DNm(bd, bd, RHO, mq)                                            # aliasing
    # zero right-hand side
    z = ctx.new_spinor()
    z.zero_()
    assert ctx.solve_DNm(x, z, RHO, mq) == (0.0, 0, True)


def test_mixed_precision_refinement_reaches_fp64_accuracy():
    """fp32 inner CG + fp64 residual (BASELINE config 4's 'fp32 inner, fp64 accumulation' applied to the inversion):
    the solution must agree with the oracle's all-fp64 CG far below the fp32 floor, with a handful of fp64 applications."""
    import paper_1010_5636_b200 as nd
    from lattice_inputs import gauge_field

    dims, n, eps, mq = (8, 4, 4, 8), 60, 0.004, 0.2
    ctx64, DN = setup(64, dims, n, eps)
    U = gauge_field(dims, "smooth", eps=0.3)
    ctx32 = nd.Context(dims, prec=32, recon=12, bc_time=-1)
    ctx32.set_gauge(U.astype(np.complex64))
    ctx32.set_sign_poly(osign.cheb_coeffs(n, eps), eps, QNORM, M)
    b = gaussian_spinor(dims)
    x = ctx64.new_spinor()
    relres, outer, inner, ok = ctx64.solve_DNm_mixed(ctx32, x, ctx64.pack_spinor(b), RHO, mq, tol=1e-10, inner_tol=1e-3)
    assert ok and relres <= 1e-10 and 2 <= outer <= 8 and inner > outer
    D = lambda v: osolver.apply_DNm(DN, v, 1.0 / RHO, mq)
    Dd = lambda v: wilson.apply_gamma5(D(wilson.apply_gamma5(v)))
    xr, _, _ = osolver.cg_normal_equations(D, Dd, b, 1e-12, 400)
    got = ctx64.unpack_spinor(x)
    assert rel_l2(got, xr) <= 1e-9
    assert np.linalg.norm((b - D(got)).ravel()) <= 1e-9 * np.linalg.norm(b.ravel())
    # precision conversion round trip and rejection of mismatched contexts
    y32, y64 = ctx32.new_spinor(), ctx64.new_spinor()
    ctx64.convert_spinor(y32, 32, x, 64)
    ctx64.convert_spinor(y64, 64, y32, 32)
    assert rel_l2(ctx64.unpack_spinor(y64), got) <= 1e-7
    other = nd.Context((4, 4, 4, 4), prec=32, recon=12)
    with pytest.raises(nd.NDError):
        ctx64.solve_DNm_mixed(other, x, y64, RHO, mq)
