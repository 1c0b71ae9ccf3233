"""Helpers shared by the `-m gpu` parity tests: CUDA path (through the C-ABI binding) vs the CPU oracle."""
import numpy as np

from lattice_inputs import gauge_field, gaussian_spinor


def rel_l2(a, b):
    a = np.asarray(a).ravel()
    b = np.asarray(b).ravel()
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def field_errors(got, ref):
    """(relative L2 deviation, worst single site): the second is max_x |got(x) - ref(x)| over sites (norm over spin and colour)
    relative to the rms site norm of ref - an isolated wrong site, invisible in the L2 norm of a large field, shows up here."""
    got, ref = np.asarray(got), np.asarray(ref)
    site = np.sqrt((np.abs(got - ref) ** 2).sum(axis=(-2, -1)))
    rms = np.sqrt((np.abs(ref) ** 2).sum(axis=(-2, -1)).mean())
    return rel_l2(got, ref), float(site.max() / rms)


def assert_field_close(got, ref, tol, ctx=None, site_factor=4.0, tag=None):
    """Parity of a spinor field with the oracle: relative L2 <= tol AND worst site <= site_factor * tol (of the rms site norm).
    With the 8-parameter links rounding is amplified by ~1/N at the link with the smallest N = |a2|^2 + |a3|^2 (R8):
    that one link's share, unit roundoff / min N, is added to the site bound when the context is given."""
    l2, worst = field_errors(got, ref)
    tol_site = site_factor * tol
    if ctx is not None and ctx.recon == 8:
        tol_site += (2.0 ** -53 if ctx.prec == 64 else 2.0 ** -24) / ctx.gauge_stats()[2]
    assert l2 <= tol, (tag, "rel L2", l2, tol)
    assert worst <= tol_site, (tag, "worst site", worst, tol_site)


def round_to(x, prec):
    """DESIGN.md R15: the fp32 path receives inputs rounded to nearest; the oracle runs in fp64 on the rounded inputs."""
    if prec == 64:
        return np.ascontiguousarray(x, dtype=np.complex128)
    return np.ascontiguousarray(x.astype(np.complex64).astype(np.complex128))


def make_context(dims, prec, recon, bc=-1, kind="haar", eps=0.3, seed=None):
    import paper_1010_5636_b200 as nd

    kw = {} if seed is None else dict(seed=seed)
    U = round_to(gauge_field(dims, kind, eps=eps, **kw), prec)
    ctx = nd.Context(dims, prec=prec, recon=recon, bc_time=bc)
    ctx.set_gauge(U if prec == 64 else U.astype(np.complex64))
    return ctx, U


TOL = {64: 1e-12, 32: 1e-5}     # BASELINE.json north_star: relative L2 per operator application
