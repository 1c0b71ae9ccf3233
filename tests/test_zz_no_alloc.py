"""nd_dot_static - the inner product for callers that cannot allocate device memory - against the library's ordinary
context path (nd_dot_dev) and numpy.

Why the entry point exists: a context (nd_create) reserves its reduction scratch with cudaMalloc.  A plug-in inside an
application whose pool already owns the GPU's memory, code in a phase where the device allocator must stay untouched
(cudaMalloc / cudaFree synchronise the whole GPU), or a process with a fixed memory budget cannot do that.  nd_dot_static
needs no context and never allocates: its partial sums sit in a 256 KiB array inside the library image, which every call on
the device shares.  Hence what is checked here, twice in a row on purpose: the second call runs on a SMALLER field right
after a larger one, so the array still holds the first call's partial sums - none of them may leak into the second result.

The file sorts last (pytest --collect-only): with `-x` a failure here hides no other test.  It uses nothing from earlier
tests, so it passes alone in a fresh process (where its first call performs the per-device address look-up) as well as
after the rest of the suite."""
import ctypes

import numpy as np
import pytest

from lattice_inputs import gaussian_spinor
from tests.gpu_common import make_context, round_to

pytestmark = pytest.mark.gpu

# (larger lattice, smaller lattice): both ragged against the 256-site ranges of the kernel (1920 = 7.5, 480 = 1.875 ranges)
# and a pair that spans hundreds of CTAs
PAIRS = [((10, 6, 4, 8), (6, 4, 2, 10)), ((16, 16, 12, 24), (10, 6, 6, 6))]


def _dots(nd, torch, dims, prec, seeds):
    """(nd_dot_static, nd_dot_dev, numpy) values of <a, b> on one lattice."""
    ctx, _ = make_context(dims, prec, 12, -1, "smooth")
    a = round_to(gaussian_spinor(dims, seed=seeds[0]), prec)
    b = round_to(gaussian_spinor(dims, seed=seeds[1]), prec)
    x, y = ctx.pack_spinor(a), ctx.pack_spinor(b)
    out_static = torch.full((2,), float("nan"), dtype=torch.float64, device=ctx.torch_device)
    out_ctx = torch.full((2,), float("nan"), dtype=torch.float64, device=ctx.torch_device)
    ctx.dot_dev(x, y, out_ctx)                                           # the existing path: context-owned cudaMalloc'ed scratch
    nd.dot_static(x, y, ctx.V, prec, out_static, device=ctx.device, stream=ctx.stream)   # same stream: ordered after the packs
    ctx.synchronize()
    s, c = out_static.cpu().numpy(), out_ctx.cpu().numpy()
    scale = np.linalg.norm(a) * np.linalg.norm(b)
    ctx.close()
    return complex(s[0], s[1]), complex(c[0], c[1]), np.vdot(a.ravel(), b.ravel()), scale


@pytest.mark.parametrize("big,small", PAIRS)
@pytest.mark.parametrize("prec", [64, 32])
def test_dot_static_matches_context_path_on_two_calls_in_a_row(prec, big, small):
    import torch

    import paper_1010_5636_b200 as nd

    for dims, seeds in ((big, (1, 2)), (small, (3, 4))):        # second call: fewer slots than the first one filled
        got, ctx_val, ref, scale = _dots(nd, torch, dims, prec, seeds)
        # the tolerance of tests/test_gpu_blas.py::test_dot_norm: fp64 accumulation of exactly representable products
        assert abs(got - ctx_val) <= 1e-13 * scale, (dims, prec, got, ctx_val)
        assert abs(got - ref) <= 1e-13 * scale, (dims, prec, got, ref)


def test_dot_static_is_reproducible_and_conjugate_symmetric():
    import torch

    import paper_1010_5636_b200 as nd

    dims, prec = (12, 6, 6, 10), 32
    ctx, _ = make_context(dims, prec, 12, -1, "smooth")
    a, b = round_to(gaussian_spinor(dims, seed=5), prec), round_to(gaussian_spinor(dims, seed=6), prec)
    x, y = ctx.pack_spinor(a), ctx.pack_spinor(b)
    o = torch.zeros((3, 2), dtype=torch.float64, device=ctx.torch_device)
    nd.dot_static(x, y, ctx.V, prec, o[0], stream=ctx.stream)
    nd.dot_static(y, x, ctx.V, prec, o[1], stream=ctx.stream)
    nd.dot_static(x, y, ctx.V, prec, o[2], stream=ctx.stream)
    ctx.synchronize()
    h = o.cpu().numpy()
    assert np.array_equal(h[0], h[2])                          # no atomics: the same bits every time
    # <y, x> = conj <x, y>: the real parts are formed from the same products in the same order, the imaginary parts are not
    assert h[1][0] == h[0][0] and abs(h[1][1] + h[0][1]) <= 1e-13 * np.linalg.norm(a) * np.linalg.norm(b)
    ctx.close()


def test_dot_static_at_the_largest_size_it_accepts():
    """V = ND_DOT_STATIC_MAX_SITES exactly (every slot of the static array in use), then a tiny field straight after."""
    import torch

    import paper_1010_5636_b200 as nd

    V = nd.DOT_STATIC_MAX_SITES
    g = torch.Generator(device="cuda:0").manual_seed(17)
    x = torch.randn(24 * V, dtype=torch.float32, device="cuda:0", generator=g)
    out = torch.zeros((2, 2), dtype=torch.float64, device="cuda:0")
    nd.dot_static(x, x, V, 32, out[0])                         # legacy default stream, as torch's kernels above
    nd.dot_static(x[: 24 * 300], x[: 24 * 300], 300, 32, out[1])   # 300 sites of 6 float4 planes: a valid small field
    torch.cuda.synchronize()
    ref = float(x.double().pow(2).sum())
    h = out.cpu().numpy()
    assert abs(h[0][0] - ref) <= 1e-12 * ref and h[0][1] == 0.0
    ref_small = float(x[: 24 * 300].double().pow(2).sum())
    assert abs(h[1][0] - ref_small) <= 1e-12 * ref_small and h[1][1] == 0.0


def test_dot_static_refuses_what_does_not_fit():
    import torch

    import paper_1010_5636_b200 as nd

    lib = nd.load_library()
    assert nd.DOT_STATIC_MAX_SITES == 4194304 and nd.DOT_STATIC_SCRATCH_BYTES == 262144
    buf = torch.zeros(64, dtype=torch.float64, device="cuda:0")
    err = ctypes.create_string_buffer(512)
    p = buf.data_ptr()
    # one site more than the static array has room for: clear refusal, nothing launched, message names the limit
    rc = lib.nd_dot_static(p, p, nd.DOT_STATIC_MAX_SITES + 1, 64, 0, None, p, err, len(err))
    assert rc == -1 and b"4194304" in err.value and b"nd_create" in err.value
    with pytest.raises(nd.NDError, match="4194304"):
        nd.dot_static(buf, buf, nd.DOT_STATIC_MAX_SITES + 1, 64, buf)
    for V, prec, dev in ((0, 64, 0), (16, 16, 0), (16, 64, -1)):
        assert lib.nd_dot_static(p, p, V, prec, dev, None, p, err, len(err)) == -1 and err.value
    assert lib.nd_dot_static(None, p, 16, 64, 0, None, p, None, 0) == -1          # errbuf is optional
    torch.cuda.synchronize()
    assert float(buf.abs().sum()) == 0.0                        # refused calls wrote nothing
