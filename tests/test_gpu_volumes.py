"""lattices shaped like the paper's own benchmark volumes, L = 24 (not a power of two),
against the plain-C oracle - tile / block generality of every kernel on extents 24 and odd block tails."""
import numpy as np
import pytest

from lattice_inputs import gaussian_spinor
from oracle import sign as osign
from oracle import wilson, wilson_c
from tests.gpu_common import TOL, assert_field_close, make_context, rel_l2, round_to

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("recon", [12, 8])
@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("dims", [(8, 24, 24, 24), (6, 12, 24, 12)])
def test_Q_on_24_cubed(prec, recon, dims):
    ctx, U = make_context(dims, prec, recon, -1, "smooth", eps=0.3)
    psi = round_to(gaussian_spinor(dims), prec)
    y = ctx.new_spinor()
    ctx.apply_Q(y, ctx.pack_spinor(psi), -1.6)
    assert_field_close(ctx.unpack_spinor(y), wilson_c.apply_Q(psi, U, -1.6, -1), TOL[prec], ctx=ctx)


def test_DN_on_24_cubed():
    dims = (8, 24, 24, 24)
    ctx, U = make_context(dims, 64, 12, -1, "smooth", eps=0.3)
    eta = gaussian_spinor(dims)
    n, eps, qnorm, pref = 30, 0.004, 6.4, 1 / 1.6
    c = osign.cheb_coeffs(n, eps)
    ctx.set_sign_poly(c, eps, qnorm, -1.6)
    out, work = ctx.new_spinor(), ctx.new_spinor(3)
    ctx.apply_DN(out, ctx.pack_spinor(eta), pref, work, use_graph=True)
    Q = wilson_c.make_Q(U, -1.6, -1)
    ref = osign.apply_DN(Q, wilson.apply_gamma5, eta, c, eps, qnorm, pref)
    assert_field_close(ctx.unpack_spinor(out), ref, 1e-11, ctx=ctx)
