"""Parity of the CUDA sign function / Neuberger-Dirac operator (fused Clenshaw recurrence, low-mode projection, D_N
epilogue) with the CPU oracle recipe on the same seeded inputs, coefficients and low modes.
BASELINE.json configs 3 (8^3x16 fp64, l=20, n~100) and 4 (16^3x32 fp32 stencil + fp64 accumulation, l=50, n~200).
Tolerances (R15): |D_N eta - oracle| <= c*max(delta, 1e-11)*|eta| (fp64), <= c*max(delta, 5e-6)*|eta| (fp32)."""
import numpy as np
import pytest

from lattice_inputs import gauge_field, gaussian_spinor
from oracle import sign as osign
from oracle import wilson, wilson_c
from tests.gpu_common import assert_field_close, make_context, rel_l2, round_to

pytestmark = pytest.mark.gpu

RHO = 1.6
M = -RHO
PREF = 1.0 / RHO
QNORM = abs(4.0 + M) + 4.0


def low_space(Q, shape, l, cut, degree, seed=11):
    """Input preparation (no method arithmetic of the CUDA path): an orthonormal, roughly Q-invariant block V from one
    Chebyshev-filter sweep with the ORACLE's Q, orthonormalised by a library QR, and its Rayleigh-Ritz pairs (nu, u)
    of Q (eq. 2.7) in matrix form.  Eq. 2.11 is defined for any orthonormal V; (nu, u) are shared inputs."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n = int(np.prod(shape))
    a, b = cut, QNORM * QNORM
    e, c0 = (b - a) / 2.0, (b + a) / 2.0
    cols = []
    for _ in range(l):
        v = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
        t0, t1 = v, (Q(Q(v)) - c0 * v) / e
        for _ in range(degree - 1):
            t0, t1 = t1, 2.0 * (Q(Q(t1)) - c0 * t1) / e - t0
        cols.append(t1.reshape(n))
    Vm, _ = np.linalg.qr(np.stack(cols, axis=1))
    QV = np.stack([Q(Vm[:, j].reshape(shape)).reshape(n) for j in range(l)], axis=1)
    Mm = Vm.conj().T @ QV
    nu, W = np.linalg.eigh(0.5 * (Mm + Mm.conj().T))
    Um = Vm @ W
    return nu, [np.ascontiguousarray(Um[:, j]).reshape(shape) for j in range(l)]


def upload_modes(ctx, U, prec):
    V = ctx.new_spinor(len(U))
    for k, u in enumerate(U):
        ctx.pack_spinor(round_to(u, prec), out=V[k])
    return V


@pytest.mark.parametrize("use_graph", [False, True])
@pytest.mark.parametrize("prec,recon", [(64, 12), (64, 8), (32, 12)])
def test_sign_small_no_modes(prec, recon, use_graph):
    """sign(Q) eta ~ X P_n(X^2) eta (eq. 2.5), 2n+1 stencils (pin P10 on the CUDA side via the launch counter)."""
    dims = (8, 4, 4, 4)
    ctx, U = make_context(dims, prec, recon, -1, "smooth", eps=0.3)
    eta = round_to(gaussian_spinor(dims), prec)
    n, eps = 60, 0.004
    c, delta = osign.cheb_coeffs(n, eps), None
    ctx.set_sign_poly(c, eps, QNORM, M)
    ctx.set_lowmodes(None, [])
    x, out, work = ctx.pack_spinor(eta), ctx.new_spinor(), ctx.new_spinor(3)
    l0 = ctx.launch_count()
    ctx.apply_sign(out, x, work, use_graph=use_graph)
    ctx.synchronize()
    assert ctx.launch_count() - l0 == 2 * n + 1            # 2n+1 stencils and nothing else (b_n = c_n eta is never materialised)
    Q = lambda v: wilson.apply_Q(v, U, M, -1)
    ref = osign.sign_poly(Q, eta, c, eps, QNORM)
    assert_field_close(ctx.unpack_spinor(out), ref, (1e-12 if prec == 64 else 5e-6), ctx=ctx)
    # replay (graph cache hit) gives the same bits
    first = ctx.unpack_spinor(out)
    ctx.apply_sign(out, x, work, use_graph=use_graph)
    assert np.array_equal(first, ctx.unpack_spinor(out))


@pytest.mark.parametrize("n", [0, 1, 2, 3])
def test_sign_degenerate_degrees(n):
    """The first two Clenshaw steps are special (b_n = c_n eta and b_{n+1} = 0 are never materialised): degrees at which they
    are the last steps too.  The work vectors start as NaN: nothing may be read from them before it has been written."""
    dims = (4, 4, 4, 4)
    ctx, U = make_context(dims, 64, 12, -1, "smooth")
    eta = gaussian_spinor(dims)
    eps = 0.01
    c = osign.cheb_coeffs(n, eps)
    ctx.set_sign_poly(c, eps, QNORM, M)
    x, out, work = ctx.pack_spinor(eta), ctx.new_spinor(), ctx.new_spinor(3)
    import torch

    with torch.cuda.stream(ctx.stream):
        work.fill_(float("nan"))
    ctx.apply_sign(out, x, work)
    Q = lambda v: wilson.apply_Q(v, U, M, -1)
    assert_field_close(ctx.unpack_spinor(out), osign.sign_poly(Q, eta, c, eps, QNORM), 1e-13, ctx=ctx)


def test_config3_DN_8c16_fp64_l20():
    """BASELINE config 3: D_N on 8^3x16, fp64, exp(0.3 i H) links, l = 20 projected modes, degree ~100."""
    dims = (16, 8, 8, 8)
    ctx, U = make_context(dims, 64, 12, -1, "smooth", eps=0.3)
    Q = wilson_c.make_Q(U, M, -1)
    eta = gaussian_spinor(dims)
    nu, Us = low_space(Q, eta.shape, 20, cut=0.6, degree=30)
    eps = 0.99 * 0.20 / QNORM ** 2          # lowest Q^2 eigenvalue of this field ~0.202
    n = 100
    c = osign.cheb_coeffs(n, eps)
    delta = osign.measure_delta(c, eps)
    ctx.set_sign_poly(c, eps, QNORM, M)
    ctx.set_lowmodes(upload_modes(ctx, Us, 64), nu)
    x, out, work = ctx.pack_spinor(eta), ctx.new_spinor(), ctx.new_spinor(3)
    for g in (False, True, True):
        ctx.apply_DN(out, x, PREF, work, use_graph=g)
        got = ctx.unpack_spinor(out)
        ref = osign.apply_DN(Q, wilson.apply_gamma5, eta, c, eps, QNORM, PREF, nu, Us)
        err = np.linalg.norm((got - ref).ravel())
        assert err <= PREF * max(delta, 1e-11) * np.linalg.norm(eta.ravel())
        assert_field_close(got, ref, 1e-10)  # same c_k, V, nu
    # the projected sign itself, and sign(Q) u_k = sign(nu_k) u_k up to the non-invariance of V
    ctx.apply_sign(out, x, work)
    refs = osign.sign_projected(Q, eta, c, eps, QNORM, nu, Us)
    assert_field_close(ctx.unpack_spinor(out), refs, 1e-10, ctx=ctx)
    # Ginsparg-Wilson (P9) on the CUDA path: gamma5 D + D gamma5 - (1/c) D gamma5 D = c gamma5 (1 - S^2) ~ small
    g5 = wilson.apply_gamma5
    def D(v):
        ctx.apply_DN(out, ctx.pack_spinor(v), PREF, work)
        return ctx.unpack_spinor(out)
    lhs = g5(D(eta)) + D(g5(eta)) - (1.0 / PREF) * D(g5(D(eta)))
    Dref = lambda v: osign.apply_DN(Q, g5, v, c, eps, QNORM, PREF, nu, Us)
    lhs_ref = g5(Dref(eta)) + Dref(g5(eta)) - (1.0 / PREF) * Dref(g5(Dref(eta)))
    assert np.linalg.norm((lhs - lhs_ref).ravel()) <= 1e-9 * np.linalg.norm(eta.ravel())


def test_config4_DN_16c32_fp32_l50():
    """BASELINE config 4: D_N on 16^3x32, fp32 stencil / links / Clenshaw vectors with fp64 reductions, exp(0.25 i H)
    links, l = 50 projected modes, degree ~200, against the all-fp64 oracle recipe on the rounded inputs."""
    dims = (32, 16, 16, 16)
    ctx, U = make_context(dims, 32, 12, -1, "smooth", eps=0.25)
    Q = wilson_c.make_Q(U, M, -1)
    eta = round_to(gaussian_spinor(dims), 32)
    nu, Us = low_space(Q, eta.shape, 50, cut=1.0, degree=8)
    Us = [round_to(u, 32) for u in Us]      # the modes are inputs: both sides get the fp32-rounded vectors
    eps, n = 0.004, 200
    c = osign.cheb_coeffs(n, eps)
    delta = osign.measure_delta(c, eps)
    ctx.set_sign_poly(c, eps, QNORM, M)
    ctx.set_lowmodes(upload_modes(ctx, Us, 32), nu)
    x, out, work = ctx.pack_spinor(eta), ctx.new_spinor(), ctx.new_spinor(3)
    ref = osign.apply_DN(Q, wilson.apply_gamma5, eta, c, eps, QNORM, PREF, nu, Us)
    for g in (False, True):
        ctx.apply_DN(out, x, PREF, work, use_graph=g)
        err = np.linalg.norm((ctx.unpack_spinor(out) - ref).ravel())
        assert err <= PREF * max(delta, 5e-6) * np.linalg.norm(eta.ravel())


@pytest.mark.parametrize("prec", [64, 32])
def test_DN_free_field_closed_form(prec):
    """P3 on the CUDA path with no oracle in the loop: on a free-field plane wave
    D_N(p) w = c [1 + (M + i sum gamma_mu sin p_mu)/omega(p)] w."""
    dims = (8, 4, 4, 4)
    ctx, U = make_context(dims, prec, 12, -1, "unit")
    g, g5m = wilson.gamma_matrices()
    lo = np.inf
    for n0 in range(8):
        for n1 in range(4):
            for n2 in range(4):
                for n3 in range(4):
                    p = np.array([(2 * n0 + 1) * np.pi / 8, 2 * np.pi * n1 / 4, 2 * np.pi * n2 / 4, 2 * np.pi * n3 / 4])
                    lo = min(lo, (4 + M - np.cos(p).sum()) ** 2 + (np.sin(p) ** 2).sum())
    eps = 0.99 * lo / QNORM ** 2
    c = osign.cheb_coeffs(100, eps)
    delta = osign.measure_delta(c, eps, 50001)
    rng = np.random.default_rng(3)
    w = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
    n = (1, 1, 0, 3)
    p = np.array([(2 * n[0] + 1) * np.pi / 8] + [2 * np.pi * n[i] / 4 for i in (1, 2, 3)])
    grids = np.meshgrid(*[np.arange(d) for d in dims], indexing="ij")
    phase = np.exp(1j * sum(p[i] * grids[i] for i in range(4)))
    psi = round_to(phase[..., None, None] * w, prec)
    Mp = 4 + M - np.cos(p).sum()
    om = np.sqrt(Mp * Mp + (np.sin(p) ** 2).sum())
    Dp = Mp * np.eye(4) + 1j * sum(g[mu] * np.sin(p[mu]) for mu in range(4))
    expect = phase[..., None, None] * (PREF * (w + (Dp @ w) / om))
    ctx.set_sign_poly(c, eps, QNORM, M)
    out, work = ctx.new_spinor(), ctx.new_spinor(3)
    ctx.apply_DN(out, ctx.pack_spinor(psi), PREF, work)
    err = np.linalg.norm((ctx.unpack_spinor(out) - expect).ravel())
    assert err <= PREF * max(delta, 1e-11 if prec == 64 else 5e-6) * np.linalg.norm(psi.ravel())


def test_state_errors():
    import paper_1010_5636_b200 as nd

    ctx, _ = make_context((4, 4, 4, 4), 64, 12)
    x, out, work = ctx.new_spinor(), ctx.new_spinor(), ctx.new_spinor(3)
    with pytest.raises(nd.NDError) as e:
        ctx.apply_sign(out, x, work)           # polynomial not set
    assert e.value.code == -2
    ctx.set_sign_poly(osign.cheb_coeffs(4, 0.1), 0.1, QNORM, M)
    with pytest.raises(nd.NDError) as e:
        ctx.apply_DN(x, x, PREF, work)         # aliasing
    assert e.value.code == -1
