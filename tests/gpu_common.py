"""Helpers shared by the `-m gpu` parity tests: CUDA path (through the C-ABI binding) vs the CPU oracle."""
import numpy as np

from lattice_inputs import gauge_field, gaussian_spinor


def rel_l2(a, b):
    a = np.asarray(a).ravel()
    b = np.asarray(b).ravel()
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


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
