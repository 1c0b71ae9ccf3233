"""nd_apply_DN_multi / nd_apply_sign_multi (several right-hand sides per launch; VERDICT r1 task 7) against the single-source
calls and the CPU oracle recipe, on lattices that take each of the three stencil paths (hop-parallel, site-per-thread with
blockIdx.y = source, tiled kernel looped over sources), with projected low modes."""
import numpy as np
import pytest

from lattice_inputs import gaussian_spinor
from oracle import sign as osign
from oracle import wilson, wilson_c
from tests.gpu_common import assert_field_close, make_context, rel_l2, round_to
from tests.test_gpu_sign import M, PREF, QNORM, low_space, upload_modes

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("dims,prec,nrhs,l", [((8, 4, 4, 4), 64, 5, 6), ((8, 8, 16, 16), 32, 3, 4), ((40, 8, 16, 32), 32, 2, 3),
                                              ((8, 4, 4, 4), 32, 16, 0)])
def test_multi_rhs_matches_single_and_oracle(dims, prec, nrhs, l):
    ctx, U = make_context(dims, prec, 12, -1, "smooth", eps=0.3)
    Q = wilson_c.make_Q(U, M, -1)
    etas = [round_to(gaussian_spinor(dims, seed=100 + j), prec) for j in range(nrhs)]
    n, eps = 30, 0.004
    c = osign.cheb_coeffs(n, eps)
    ctx.set_sign_poly(c, eps, QNORM, M)
    if l:
        nu, Us = low_space(Q, etas[0].shape, l, cut=1.0, degree=6)
        Us = [round_to(u, prec) for u in Us]
        ctx.set_lowmodes(upload_modes(ctx, Us, prec), nu)
    else:
        nu, Us = None, None
    X, OUT, work = ctx.new_spinor(nrhs), ctx.new_spinor(nrhs), ctx.new_spinor(3 * nrhs)
    for j in range(nrhs):
        ctx.pack_spinor(etas[j], out=X[j])
    single, w1 = ctx.new_spinor(), ctx.new_spinor(3)
    tol = 1e-12 if prec == 64 else 5e-6
    for use_graph in (False, True, True):
        OUT.zero_()
        l0 = ctx.launch_count()
        ctx.apply_DN_multi(OUT, X, PREF, work, use_graph=use_graph)
        ctx.synchronize()
        batch_launches = ctx.launch_count() - l0
        for j in range(nrhs):
            l1 = ctx.launch_count()
            ctx.apply_DN(single, X[j], PREF, w1)
            single_launches = ctx.launch_count() - l1
            got, one = ctx.unpack_spinor(OUT[j]), ctx.unpack_spinor(single)
            assert rel_l2(got, one) <= (1e-13 if prec == 64 else 1e-6), (j, rel_l2(got, one))
            if j in (0, nrhs - 1):
                ref = osign.apply_DN(Q, wilson.apply_gamma5, etas[j], c, eps, QNORM, PREF, nu, Us)
                assert_field_close(got, ref, tol, tag=j)
    # the batch is ONE launch sequence on lattices where the stencil takes the batch as a grid dimension
    if ctx.get_stencil_variant() == "site":
        assert batch_launches <= 2 * n + 2 + 4 * nrhs and batch_launches < 0.5 * nrhs * single_launches
    # sign alone
    ctx.apply_sign_multi(OUT, X, work)
    ref = osign.sign_projected(Q, etas[1], c, eps, QNORM, nu, Us) if l else osign.sign_poly(Q, etas[1], c, eps, QNORM)
    assert_field_close(ctx.unpack_spinor(OUT[1]), ref, tol, ctx=ctx)


def test_multi_rhs_argument_checks():
    import paper_1010_5636_b200 as nd

    ctx, _ = make_context((4, 4, 4, 4), 64, 12)
    ctx.set_sign_poly(osign.cheb_coeffs(4, 0.1), 0.1, QNORM, M)
    X, OUT, work = ctx.new_spinor(17), ctx.new_spinor(17), ctx.new_spinor(51)
    with pytest.raises(nd.NDError) as e:
        ctx.apply_DN_multi(OUT, X, PREF, work)            # more than 16 right-hand sides
    assert e.value.code == -1
