"""Parity at BASELINE.json's full size in the launch configuration bench.py times: the 32^3x64 Haar lattice (config 2),
fp32 and fp64, recon 12 (headline) and 8.  Q is compared with the plain-C oracle on EVERY site (the oracle finishes in
about a second at this volume); D_N, which the oracle cannot recompute in reasonable time at degree 100, is checked
through properties that hold at any size (Hermiticity of gamma5 D_N, |sign(Q) eta| <= (1+delta)|eta|, linearity) and
against the oracle on a reduced degree."""
import numpy as np
import pytest

from lattice_inputs import gauge_field, gaussian_spinor
from oracle import sign as osign
from oracle import wilson, wilson_c
from tests.gpu_common import TOL, assert_field_close, rel_l2, round_to

pytestmark = pytest.mark.gpu

DIMS = (64, 32, 32, 32)
M = -1.6
QNORM = 6.4


@pytest.fixture(scope="module")
def haar_field():
    return gauge_field(DIMS, "haar")


@pytest.mark.parametrize("prec,recon", [(32, 12), (64, 12), (32, 8), (64, 8)])
def test_config2_Q_every_site(haar_field, prec, recon):
    import paper_1010_5636_b200 as nd

    U = round_to(haar_field, prec)
    psi = round_to(gaussian_spinor(DIMS), prec)
    ctx = nd.Context(DIMS, prec=prec, recon=recon, bc_time=-1)
    ctx.set_gauge(U if prec == 64 else U.astype(np.complex64))
    x, y = ctx.pack_spinor(psi), ctx.new_spinor()
    ctx.apply_Q(y, x, M)
    got = ctx.unpack_spinor(y)
    ref = wilson_c.apply_Q(psi, U, M, -1)
    assert rel_l2(got, ref) <= TOL[prec]
    # worst single site, relative to the field's rms site norm: no isolated wrong site hides in the L2 norm
    site_err = np.sqrt((np.abs(got - ref) ** 2).sum(axis=(4, 5)))
    rms = np.sqrt((np.abs(ref) ** 2).sum(axis=(4, 5)).mean())
    # recon 8 amplifies rounding by ~1/N, N = |a2|^2 + |a3|^2 (R8): among 8.4M Haar links min N ~ 3e-4
    min_n = ctx.gauge_stats()[2]
    unit = 2.0 ** -53 if prec == 64 else 2.0 ** -24
    tol_site = (1e-12 if prec == 64 else 2e-5) + (unit / min_n if recon == 8 else 0.0)
    assert site_err.max() <= tol_site * rms
    ctx.close()


def test_config2_DN_bench_configuration(haar_field):
    """The bench step itself: fp32, recon 12, degree 100, l = 8, CUDA graph."""
    import paper_1010_5636_b200 as nd

    U = round_to(haar_field, 32)
    ctx = nd.Context(DIMS, prec=32, recon=12, bc_time=-1)
    ctx.set_gauge(U.astype(np.complex64))
    Q = wilson_c.make_Q(U, M, -1)
    eps, pref = 0.002, 1 / 1.6
    eta = round_to(gaussian_spinor(DIMS), 32)
    chi = round_to(gaussian_spinor(DIMS, seed=77), 32)
    x, z = ctx.pack_spinor(eta), ctx.pack_spinor(chi)
    out, out2, work = ctx.new_spinor(), ctx.new_spinor(), ctx.new_spinor(3)
    # (1) reduced degree against the oracle recipe, same coefficients, whole field
    n = 6
    c = osign.cheb_coeffs(n, eps)
    ctx.set_sign_poly(c, eps, QNORM, M)
    ctx.apply_DN(out, x, pref, work, use_graph=True)
    ref = osign.apply_DN(Q, wilson.apply_gamma5, eta, c, eps, QNORM, pref)
    assert_field_close(ctx.unpack_spinor(out), ref, 1e-5, ctx=ctx)
    # (2) degree 100 (the bench's polynomial): properties
    n = 100
    c = osign.cheb_coeffs(n, eps)
    delta = osign.measure_delta(c, eps)
    ctx.set_sign_poly(c, eps, QNORM, M)
    ctx.apply_sign(out, x, work, use_graph=True)
    ctx.apply_sign(out2, z, work, use_graph=False)
    ne, ns = np.sqrt(ctx.norm2(x)), np.sqrt(ctx.norm2(out))
    assert ns <= (1 + delta + 1e-5) * ne                      # |x P(x^2)| <= 1 + delta on the whole spectrum
    # Hermiticity of the polynomial sign function: <chi, S eta> = <S chi, eta>
    a, b = ctx.dot(z, out), ctx.dot(out2, x)
    assert abs(a - b) <= 2e-5 * np.sqrt(ctx.norm2(z)) * ne
    # graph replay and plain enqueue give the same bits
    ctx.apply_sign(out2, x, work, use_graph=False)
    assert np.array_equal(ctx.unpack_spinor(out), ctx.unpack_spinor(out2))
    ctx.close()


def test_config2_DN_with_lowmodes_every_site(haar_field):
    """The step bench.py times - 32^3x64, fp32, recon 12, l = 8 projected vectors, CUDA graph - against the oracle's eq. 2.11
    on every site (the headline configuration had no oracle comparison with low modes).  The block of eq. 2.11 is
    any orthonormal set with its Rayleigh quotients (bench.py's build_modes makes such a set); here it is built on the CPU -
    Gaussian vectors orthonormalised with numpy, nu_k = <v_k, Q v_k> from the plain-C oracle - and handed to both sides, so no
    oracle input comes from the CUDA path.  Degree 6 keeps the oracle at 13 + 8 stencils; the projection kernels
    (block_dot_cols_kernel<float,2>, block_axpy_kernel<float,1>, lowmode_coef_kernel) do not depend on the degree."""
    import paper_1010_5636_b200 as nd

    l, n, eps, pref = 8, 6, 0.002, 1 / 1.6
    U = round_to(haar_field, 32)
    Q = wilson_c.make_Q(U, M, -1)
    vs = []
    for k in range(l):
        v = gaussian_spinor(DIMS, seed=300 + k)
        for _ in range(2):
            for u in vs:
                v = v - np.vdot(u.ravel(), v.ravel()) * u
        vs.append(v / np.linalg.norm(v.ravel()))
    vs = [round_to(v, 32) for v in vs]                     # orthonormal to fp32 rounding; eq. 2.11 is applied to these very vectors
    nu = np.array([np.vdot(v.ravel(), Q(v).ravel()).real for v in vs])
    assert (nu > 0).any() and (nu < 0).any()               # both signs occur: sign(nu_k) matters
    eta = round_to(gaussian_spinor(DIMS), 32)
    c = osign.cheb_coeffs(n, eps)
    ref = osign.apply_DN(Q, wilson.apply_gamma5, eta, c, eps, QNORM, pref, nu, vs)

    ctx = nd.Context(DIMS, prec=32, recon=12, bc_time=-1)
    ctx.set_gauge(U.astype(np.complex64))
    assert ctx.get_stencil_variant_for(False, 1) == "tile" and ctx.get_stencil_variant_for(True, 1) == "tile"
    ctx.set_sign_poly(c, eps, QNORM, M)
    Vd = ctx.new_spinor(l)
    for k in range(l):
        ctx.pack_spinor(vs[k], out=Vd[k])
    ctx.set_lowmodes(Vd, nu)
    x, out, work = ctx.pack_spinor(eta), ctx.new_spinor(), ctx.new_spinor(3)
    for use_graph in (True, False):
        out.zero_()
        ctx.apply_DN(out, x, pref, work, use_graph=use_graph)
        # north_star: relative L2 <= 1e-5 per operator application in fp32; worst site within 4x that of the rms site norm
        assert_field_close(ctx.unpack_spinor(out), ref, 1e-5, ctx=ctx, tag=("graph", use_graph))
    # the projected part is really there: without the low modes the result differs by far more than the tolerance
    ctx.set_lowmodes(None, [])
    ctx.apply_DN(out, x, pref, work, use_graph=False)
    assert rel_l2(ctx.unpack_spinor(out), ref) > 1e-4
    ctx.close()
