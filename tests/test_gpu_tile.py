"""The tiled marching stencils (csrc/wilson_tile.cu: neighbour exchange through shared memory, cp.async / TMA-bulk prefetch)
against the CPU oracle of eq. 2.1 and against the site-per-thread kernel, on lattices that exercise its index logic: several
time segments per tile, the antiperiodic seam inside a segment, tiles on the lattice boundary in x1 / x2, and an x1 extent
of 4 (both outside x1 neighbours of a pair of rows belong to the same neighbouring tile)."""
import numpy as np
import pytest

from lattice_inputs import gaussian_spinor
from oracle import wilson_c
from tests.gpu_common import TOL, assert_field_close, make_context, rel_l2, round_to

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("dims,bc", [((40, 8, 16, 32), -1), ((152, 4, 16, 32), -1), ((38, 16, 8, 32), +1)])
@pytest.mark.parametrize("recon", [12, 8, 18])
def test_every_variant_matches_the_oracle(dims, bc, recon):
    ctx, U = make_context(dims, 32, recon, bc, "smooth", eps=0.3)
    assert ctx.get_stencil_variant() == "tile"                       # these lattices take the tiled kernel by default
    psi = round_to(gaussian_spinor(dims), 32)
    vecs = [round_to(gaussian_spinor(dims, seed=20 + i), 32) for i in range(3)]
    x, y = ctx.pack_spinor(psi), ctx.new_spinor()
    d = [ctx.pack_spinor(v) for v in vecs]
    ref = wilson_c.apply_Q(psi, U, -1.6, bc)
    s0, s1, s2, s3 = 0.37, -1.2, -1.0, 0.81
    ref_epi = s0 * ref + s1 * vecs[0] + s2 * vecs[1] + s3 * vecs[2]
    results = {}
    for variant in ("site", "tile", "tile_tma", "tile4", "auto"):
        ctx.set_stencil_variant(variant)
        ctx.apply_Q(y, x, -1.6)
        got = ctx.unpack_spinor(y)
        assert_field_close(got, ref, TOL[32], ctx=ctx, tag=variant)
        results[variant] = got
        out = ctx.new_spinor()
        ctx.copy(out, d[1])
        ctx.apply_Q_axpbycz(out, x, -1.6, s0, s1, d[0], s2, out, s3, d[2])   # out aliases v2, as in the Clenshaw step
        assert_field_close(ctx.unpack_spinor(out), ref_epi, TOL[32], ctx=ctx, tag=variant)
    # cp.async and TMA tensor-map prefetch feed the same arithmetic, and so do the two- and the four-slot kernel: bit-identical
    assert np.array_equal(results["tile"], results["tile_tma"]) and np.array_equal(results["tile"], results["tile4"])
    assert np.array_equal(results["tile"], results["auto"])       # auto = the tiled kernel
    # worst site against the oracle, not only the norm
    scale = np.abs(ref).max()
    assert np.abs(results["tile"] - ref).max() <= (2e-5 if recon != 8 else 2e-4) * scale


@pytest.mark.parametrize("dims,bc", [((40, 8, 16, 32), -1), ((152, 4, 16, 32), -1), ((80, 16, 4, 32), +1)])
@pytest.mark.parametrize("recon", [12, 8])
def test_fp64_tiled_kernel_matches_the_oracle(dims, bc, recon):
    """wilson_Q_tile2_kernel (two link slots, next spinor through shared memory): segments, the seam, boundary tiles, x1 / x2
    extent 4 (both outside neighbours of a pair are the same row of the neighbouring tile)."""
    ctx, U = make_context(dims, 64, recon, bc, "smooth", eps=0.3)
    psi = gaussian_spinor(dims)
    vecs = [gaussian_spinor(dims, seed=20 + i) for i in range(3)]
    x, y = ctx.pack_spinor(psi), ctx.new_spinor()
    d = [ctx.pack_spinor(v) for v in vecs]
    ref = wilson_c.apply_Q(psi, U, -1.6, bc)
    s0, s1, s2, s3 = 0.37, -1.2, -1.0, 0.81
    ref_epi = s0 * ref + s1 * vecs[0] + s2 * vecs[1] + s3 * vecs[2]
    results, fused = {}, {}
    for variant in ("site", "tile", "tile_tma", "auto"):
        ctx.set_stencil_variant(variant)
        assert ctx.get_stencil_variant() == ("tile" if variant == "auto" else variant)
        ctx.apply_Q(y, x, -1.6)
        got = ctx.unpack_spinor(y)
        assert_field_close(got, ref, TOL[64], ctx=ctx, tag=variant)
        results[variant] = got
        out = ctx.new_spinor()
        ctx.copy(out, d[1])
        ctx.apply_Q_axpbycz(out, x, -1.6, s0, s1, d[0], s2, out, s3, d[2])
        fused[variant] = ctx.unpack_spinor(out)
        assert_field_close(fused[variant], ref_epi, TOL[64], ctx=ctx, tag=variant)
    # auto in fp64: the tiled kernel for the plain stencil; for the fused-epilogue one with recon 12 only (site-per-thread with recon 8)
    assert np.array_equal(results["auto"], results["tile"]) and np.array_equal(fused["auto"], fused["tile" if recon == 12 else "site"])
    assert np.array_equal(results["tile_tma"], results["tile"]) and np.array_equal(fused["tile_tma"], fused["tile"])
    scale = np.abs(ref).max()
    assert np.abs(results["tile"] - ref).max() <= (1e-13 if recon != 8 else 1e-10) * scale


@pytest.mark.parametrize("dims,bc", [((48, 16, 16, 16), -1), ((64, 8, 20, 16), +1)])
@pytest.mark.parametrize("prec,recon", [(32, 12), (32, 8), (32, 18), (64, 12), (64, 8)])
def test_x3_extent_16(dims, bc, prec, recon):
    """x3 extent 16 (BASELINE configs 1 and 4 are 16^3x32): a CTA takes two 2 x 2 x 16 tiles side by side in x2, a warp holds both
    rows of an x2 pair (the x2 exchange is synchronised within the warp), x3 shuffles stay inside half-warps."""
    ctx, U = make_context(dims, prec, recon, bc, "smooth", eps=0.3)
    psi = round_to(gaussian_spinor(dims), prec)
    vecs = [round_to(gaussian_spinor(dims, seed=20 + i), prec) for i in range(3)]
    x, y = ctx.pack_spinor(psi), ctx.new_spinor()
    d = [ctx.pack_spinor(v) for v in vecs]
    ref = wilson_c.apply_Q(psi, U, -1.6, bc)
    s0, s1, s2, s3 = 0.37, -1.2, -1.0, 0.81
    ref_epi = s0 * ref + s1 * vecs[0] + s2 * vecs[1] + s3 * vecs[2]
    assert ctx.get_stencil_variant() == "tile"
    for variant in ("site", "tile", "auto"):
        ctx.set_stencil_variant(variant)
        ctx.apply_Q(y, x, -1.6)
        assert_field_close(ctx.unpack_spinor(y), ref, TOL[prec], ctx=ctx, tag=variant)
        out = ctx.new_spinor()
        ctx.copy(out, d[1])
        ctx.apply_Q_axpbycz(out, x, -1.6, s0, s1, d[0], s2, out, s3, d[2])
        assert_field_close(ctx.unpack_spinor(out), ref_epi, TOL[prec], ctx=ctx, tag=variant)
    import paper_1010_5636_b200 as nd
    for variant in ("tile4", "tile_tma"):                            # the four-slot and tensor-map kernels: x3 extent 32 only
        with pytest.raises(nd.NDError):
            ctx.set_stencil_variant(variant)


@pytest.mark.parametrize("prec,dims", [(32, (64, 16, 16, 32)), (64, (64, 16, 16, 32)), (32, (96, 16, 16, 16))])
def test_tiled_kernel_repeats_bit_for_bit(prec, dims):
    """The exchange through shared memory and the cp.async slots are race-free by construction (pair barriers, private slots);
    a race would show up as run-to-run differences: 60 launches of the plain and of the fused stencil, each bit-identical to
    the first, while the machine is kept busy (several CTAs per SM, many segments)."""
    import torch

    ctx, U = make_context(dims, prec, 12, -1, "smooth", eps=0.3)
    ctx.set_stencil_variant("tile")
    x, y, y0 = ctx.new_spinor(), ctx.new_spinor(), ctx.new_spinor()
    v = ctx.new_spinor(3)
    ctx.gaussian(x, 1)
    for j in range(3):
        ctx.gaussian(v[j], 2 + j)
    ctx.apply_Q(y0, x, -1.6)
    f0 = ctx.new_spinor()
    ctx.apply_Q_axpbycz(f0, x, -1.6, 0.3, -0.9, v[0], -0.5, v[1], 0.1, v[2])
    with torch.cuda.stream(ctx.stream):            # the comparisons run on the context's stream, after the launches
        for _ in range(60):
            ctx.apply_Q(y, x, -1.6)
            assert torch.equal(y, y0)
            ctx.apply_Q_axpbycz(y, x, -1.6, 0.3, -0.9, v[0], -0.5, v[1], 0.1, v[2])
            assert torch.equal(y, f0)


def test_variant_selection_rules():
    import paper_1010_5636_b200 as nd

    ctx, _ = make_context((8, 8, 8, 16), 32, 12)                     # x3 extent 16: no tiled kernel
    assert ctx.get_stencil_variant() == "site"
    with pytest.raises(nd.NDError) as e:
        ctx.set_stencil_variant("tile")
    assert e.value.code == -1
    ctx64, _ = make_context((40, 8, 16, 32), 64, 12)
    assert ctx64.get_stencil_variant() == "tile"
    with pytest.raises(nd.NDError):
        ctx64.set_stencil_variant("tile4")                           # the four-slot kernel exists in fp32 only
    ctx64b, _ = make_context((40, 2, 16, 32), 64, 12)                # fp64 tiles need x1 / x2 extents >= 4
    with pytest.raises(nd.NDError):
        ctx64b.set_stencil_variant("tile")


def test_variant_for_one_call_is_the_dispatch_choice():
    """nd_get_stencil_variant_for answers for ONE call through the function the dispatch itself uses: under auto
    the kernel depends on precision, link form, plain / fused epilogue and the number of right-hand sides."""
    dims = (40, 8, 16, 32)
    c32, _ = make_context(dims, 32, 8)
    assert [c32.get_stencil_variant_for(e, 1) for e in (False, True)] == ["tile", "tile"]
    c64_12, _ = make_context(dims, 64, 12)
    assert [c64_12.get_stencil_variant_for(e, 1) for e in (False, True)] == ["tile", "tile"]
    c64_8, _ = make_context(dims, 64, 8)
    assert c64_8.get_stencil_variant_for(False, 1) == "tile_tma"      # plain fp64 recon 8: tensor-map loads
    assert c64_8.get_stencil_variant_for(False, 2) == "tile"          # ... one source per launch only
    assert c64_8.get_stencil_variant_for(True, 1) == "site"           # fused fp64 recon 8: the site kernel
    c64_18, _ = make_context(dims, 64, 18)
    assert [c64_18.get_stencil_variant_for(e, 1) for e in (False, True)] == ["site", "site"]   # no fp64 recon-18 tile
    small, _ = make_context((32, 16, 16, 16), 32, 12)                 # 16^3 x 32: tiled from two sources on
    assert small.get_stencil_variant_for(False, 1) == "site" and small.get_stencil_variant_for(False, 2) == "tile"
    for forced in ("site", "tile", "tile_tma"):
        c32.set_stencil_variant(forced)
        assert [c32.get_stencil_variant_for(e, n) for e in (False, True) for n in (1, 3)] == [forced] * 4
    assert c32.lib.nd_get_stencil_variant_for(c32._h, 0, 0) == -1
