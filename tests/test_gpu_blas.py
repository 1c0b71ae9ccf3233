"""Parity of the BLAS-1 and block (low-mode projection) kernels with numpy on the same seeded inputs
(pin P13: fp32 data with fp64 accumulation agrees with the fp64 result to ~1e-7)."""
import numpy as np
import pytest

from lattice_inputs import gaussian_spinor
from tests.gpu_common import assert_field_close, make_context, rel_l2, round_to

pytestmark = pytest.mark.gpu

DIMS = [(4, 4, 4, 4), (6, 4, 2, 10), (10, 6, 6, 6), (16, 8, 8, 8)]


@pytest.mark.parametrize("dims", DIMS)
@pytest.mark.parametrize("prec", [64, 32])
def test_axpy_scale_copy_gamma5(prec, dims):
    from oracle import wilson

    ctx, _ = make_context(dims, prec, 12, -1, "smooth")
    tol = 1e-14 if prec == 64 else 2e-7
    a = round_to(gaussian_spinor(dims, seed=1), prec)
    b = round_to(gaussian_spinor(dims, seed=2), prec)
    x, y = ctx.pack_spinor(a), ctx.pack_spinor(b)
    alpha = 0.37 - 1.21j
    ctx.axpy(alpha, x, y)
    assert rel_l2(ctx.unpack_spinor(y), alpha * a + b) <= tol
    ctx.scale(-0.5 + 2j, x)
    assert rel_l2(ctx.unpack_spinor(x), (-0.5 + 2j) * a) <= tol
    z = ctx.new_spinor()
    ctx.copy(z, y)
    assert np.array_equal(ctx.unpack_spinor(z), ctx.unpack_spinor(y))
    ctx.gamma5(z, z)
    assert rel_l2(ctx.unpack_spinor(z), wilson.apply_gamma5(alpha * a + b)) <= tol


@pytest.mark.parametrize("dims", DIMS)
@pytest.mark.parametrize("prec", [64, 32])
def test_dot_norm(prec, dims):
    ctx, _ = make_context(dims, prec, 12, -1, "smooth")
    a = round_to(gaussian_spinor(dims, seed=1), prec)
    b = round_to(gaussian_spinor(dims, seed=2), prec)
    x, y = ctx.pack_spinor(a), ctx.pack_spinor(b)
    ref = np.vdot(a.ravel(), b.ravel())
    # fp64 accumulation of exactly representable products: the rounded inputs give the fp64 result in both precisions
    assert abs(ctx.dot(x, y) - ref) <= 1e-13 * np.linalg.norm(a) * np.linalg.norm(b)
    assert abs(ctx.norm2(x) - np.vdot(a.ravel(), a.ravel()).real) <= 1e-13 * np.linalg.norm(a) ** 2
    # run-to-run bitwise reproducibility (no atomics in the reduction)
    assert ctx.dot(x, y) == ctx.dot(x, y)


@pytest.mark.parametrize("l", [1, 3, 20, 50])
@pytest.mark.parametrize("prec", [64, 32])
def test_block_dot_and_block_axpy(prec, l):
    dims = (6, 4, 6, 10)
    ctx, _ = make_context(dims, prec, 12, -1, "smooth")
    vs = [round_to(gaussian_spinor(dims, seed=100 + k), prec) for k in range(l)]
    xh = round_to(gaussian_spinor(dims, seed=7), prec)
    V = ctx.new_spinor(l)
    for k in range(l):
        ctx.pack_spinor(vs[k], out=V[k])
    x = ctx.pack_spinor(xh)
    got = ctx.block_dot(V, x)
    ref = np.array([np.vdot(v.ravel(), xh.ravel()) for v in vs])
    assert np.abs(got - ref).max() <= 1e-13 * np.linalg.norm(xh) * max(np.linalg.norm(v) for v in vs)
    rng = np.random.default_rng(5)
    a = rng.standard_normal(l) + 1j * rng.standard_normal(l)
    ctx.block_axpy(a, V, x)
    refy = xh + sum(a[k] * vs[k] for k in range(l))
    assert rel_l2(ctx.unpack_spinor(x), refy) <= (1e-14 if prec == 64 else 3e-7)
    # bad block sizes are rejected
    import paper_1010_5636_b200 as nd
    out = np.zeros(2)
    rc = ctx.lib.nd_block_dot(ctx._h, 0, V.data_ptr(), x.data_ptr(), out.ctypes.data_as(nd.binding._pd))
    assert rc == -1 and b"block_dot" in ctx.lib.nd_last_error(ctx._h)


def test_gaussian_moments_and_determinism():
    ctx, _ = make_context((8, 8, 8, 8), 32, 12, -1, "smooth")
    x, y = ctx.new_spinor(), ctx.new_spinor()
    ctx.gaussian(x, 11)
    ctx.gaussian(y, 11)
    ctx.synchronize()
    a = ctx.unpack_spinor(x)
    assert np.array_equal(a, ctx.unpack_spinor(y))
    r = np.concatenate([a.real.ravel(), a.imag.ravel()])
    n = r.size
    assert abs(r.mean()) < 5 / np.sqrt(n) and abs(r.var() - 1) < 5 * np.sqrt(2 / n)
    assert abs((r ** 4).mean() - 3) < 0.1
    ctx.gaussian(y, 12)
    b = ctx.unpack_spinor(y)
    assert abs(np.vdot(a.ravel(), b.ravel())) < 6 * np.sqrt(n)


@pytest.mark.parametrize("prec", [64, 32])
def test_dev_variants_chain_on_the_device(prec):
    """nd_block_dot_dev / nd_dot_dev / nd_norm2_dev / nd_block_axpy_dev (results left in device memory): one
    Gram-Schmidt step x <- x - V (V^dagger x) without any host round trip, against numpy; and the same numbers as the host variants."""
    import torch

    dims, l = (10, 6, 6, 6), 7
    ctx, _ = make_context(dims, prec, 12, -1, "smooth")
    vs = [round_to(gaussian_spinor(dims, seed=40 + k), prec) for k in range(l)]
    xa = round_to(gaussian_spinor(dims, seed=3), prec)
    V = ctx.new_spinor(l)
    for k in range(l):
        ctx.pack_spinor(vs[k], out=V[k])
    x = ctx.pack_spinor(xa)
    with torch.cuda.stream(ctx.stream):
        c = torch.zeros(2 * l, dtype=torch.float64, device=ctx.torch_device)
        d2 = torch.zeros(2, dtype=torch.float64, device=ctx.torch_device)
        n2 = torch.zeros(2, dtype=torch.float64, device=ctx.torch_device)
        ctx.block_dot_dev(V, x, c)
        ctx.dot_dev(V[0], x, d2)
        ctx.norm2_dev(x, n2)
        host_c = ctx.block_dot(V, x)                  # host variant: synchronises, same kernel
        cd = c.cpu().numpy()
        assert np.array_equal(cd[0::2] + 1j * cd[1::2], host_c)
        assert complex(*d2.cpu().numpy()) == host_c[0] and abs(n2.cpu().numpy()[1]) <= 1e-13 * n2.cpu().numpy()[0]
        assert abs(n2.cpu().numpy()[0] - np.vdot(xa.ravel(), xa.ravel()).real) <= 1e-12 * n2.cpu().numpy()[0]
        c.neg_()                                      # on the device, on the context's stream
        ctx.block_axpy_dev(c, V, x)
    want = xa - sum(np.vdot(v.ravel(), xa.ravel()) * v for v in vs)
    assert rel_l2(ctx.unpack_spinor(x), want) <= (1e-13 if prec == 64 else 3e-7)


@pytest.mark.parametrize("dims,l", [((64, 32, 32, 32), 8), ((32, 16, 16, 16), 50), ((32, 16, 16, 16), 3)])
@pytest.mark.parametrize("prec", [64, 32])
def test_block_ops_at_bench_sizes(prec, dims, l):
    """Block dot / block axpy against numpy at the sizes bench.py runs them: 32^3x64 with l = 8 (the headline
    step's projection) and 16^3x32 with l = 50 (config 4) / l = 3 - every branch of block_dot_cols_t's launch logic: ranges
    capped by the partial-sum scratch or not, the block's vectors split over grid.y (small lattice, many vectors) or not."""
    import paper_1010_5636_b200 as nd

    ctx = nd.Context(dims, prec=prec, recon=12, bc_time=-1)          # BLAS-1 needs no gauge field
    V = ctx.new_spinor(l)
    vs = []
    for k in range(l):
        vs.append(round_to(gaussian_spinor(dims, seed=100 + k), prec))
        ctx.pack_spinor(vs[k], out=V[k])
    xh = round_to(gaussian_spinor(dims, seed=7), prec)
    x = ctx.pack_spinor(xh)
    got = ctx.block_dot(V, x)
    ref = np.array([np.vdot(v.ravel(), xh.ravel()) for v in vs])
    scale = np.linalg.norm(xh) * max(np.linalg.norm(v) for v in vs)
    assert np.abs(got - ref).max() <= 1e-13 * scale            # fp64 accumulation of exactly representable products
    # two columns at once (the D_N projection takes <u_k, eta> and <u_k, chi> in one pass): the device-side call
    import torch

    o2 = torch.zeros(2 * l, dtype=torch.float64, device=ctx.torch_device)
    ctx.block_dot_dev(V, x, o2)
    ctx.synchronize()
    h = o2.cpu().numpy()
    assert np.array_equal(h[0::2] + 1j * h[1::2], got)          # same kernel, same bits, result left on the device
    rng = np.random.default_rng(5)
    a = rng.standard_normal(l) + 1j * rng.standard_normal(l)
    ctx.block_axpy(a, V, x)
    refy = xh.copy()
    for k in range(l):
        refy += a[k] * vs[k]
    assert_field_close(ctx.unpack_spinor(x), refy, 1e-14 if prec == 64 else 3e-7)
    ctx.close()
