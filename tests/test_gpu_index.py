"""Index of D_N by zero-mode counting on the CUDA path (nd_index_count) against the oracle's dense count
(oracle/index.py, pinned in tests/test_oracle_index.py by the trace identity and the index theorem's closed form on
constant-flux torus fields).  The whole chain is the library's own: low modes of Q from nd_lowmodes_compute (dynamic l: the two
near-zero modes of the flux field sit below a large gap), the projected sign function (eq. 2.11), B_sigma = P_sigma (1 + gamma5
sign Q) P_sigma by Chebyshev-filtered subspace iteration per chirality sector.  Compared: the counts (n_+, n_-) exactly, and the
nvec lowest eigenvalues of B_sigma with the dense sector spectrum within the sign function's error."""
import numpy as np
import pytest

from lattice_inputs import flux_su3, gauge_field
from oracle import index as oindex
from oracle import sign as osign
from oracle import wilson

pytestmark = pytest.mark.gpu

DIMS = (4, 4, 2, 2)
M = -1.6
QNORM = abs(4.0 + M) + 4.0
NVEC = 6
ZERO_TOL = 1e-3


def gpu_index(U, bc, n=80):
    import paper_1010_5636_b200 as nd

    ctx = nd.Context(DIMS, prec=64, recon=12, bc_time=bc)
    ctx.set_gauge(U)
    u, nu, resid, st = ctx.lowmodes_compute(2, M, tol=1e-9, maxit=80, lextra=6, degree=20, l_max=8, stop="residue")
    assert st["converged"], st
    guard = float(np.abs(st["nu_guard"]).min())
    assert guard > np.abs(nu).max()
    eps = 0.99 * guard ** 2 / QNORM ** 2           # the polynomial only has to hold above the projected modes
    c = osign.cheb_coeffs(n, eps)
    delta = osign.measure_delta(c, eps)
    ctx.set_sign_poly(c, eps, QNORM, M)
    ctx.set_lowmodes(u, nu)
    npl, nmi, ist = ctx.index_count(NVEC, ZERO_TOL, degree=8, maxit=40)
    ctx.close()
    return npl, nmi, ist, delta, st


@pytest.mark.parametrize("q23", [1, -1])
def test_flux_field_zero_modes_and_sector_spectra(q23):
    U = flux_su3(DIMS, 1, q23, noise=0.05)
    Q = wilson.dense_Q(U, M)
    want = oindex.zero_mode_count(Q)
    assert abs(want[0] - want[1]) == 2 and min(want) == 0
    npl, nmi, ist, delta, st = gpu_index(U, -1)
    assert st["l_chosen"] == 2                      # the dynamic choice of l found the two near-zero modes of Q
    assert (npl, nmi) == want, (npl, nmi, want, ist)
    assert delta < 1e-5
    for sec, sigma in enumerate((+1, -1)):
        exact = oindex.sector_spectrum(Q, sigma)[:NVEC]
        got = ist["evals"][sec]
        # each Ritz value is within its residue of an eigenvalue; the operators differ by the sign function's error
        assert np.abs(got - exact).max() <= 10 * delta + 2 * ist["resid"][sec].max() + 1e-9, (sigma, got, exact)
    assert ist["sign_applications"] > 0


def test_trivial_field_has_no_zero_modes():
    U = gauge_field(DIMS, "smooth", eps=0.3)
    Q = wilson.dense_Q(U, M)
    assert oindex.zero_mode_count(Q) == (0, 0)
    npl, nmi, ist, delta, st = gpu_index(U, -1)
    assert (npl, nmi) == (0, 0)
    lowest = min(oindex.sector_spectrum(Q, +1)[0], oindex.sector_spectrum(Q, -1)[0])
    assert abs(ist["evals"].min() - lowest) <= 10 * delta + 2 * ist["resid"].max() + 1e-9


def test_block_too_small_is_reported():
    import paper_1010_5636_b200 as nd

    U = flux_su3(DIMS, 1, 1, noise=0.05)
    ctx = nd.Context(DIMS, prec=64, recon=12, bc_time=-1)
    ctx.set_gauge(U)
    with pytest.raises(nd.NDError):
        ctx.index_count(2, ZERO_TOL)                # no polynomial set: ND_ERR_BAD_STATE
    u, nu, resid, st = ctx.lowmodes_compute(2, M, tol=1e-9, maxit=80, lextra=6, degree=20, l_max=8, stop="residue")
    eps = 0.99 * float(np.abs(st["nu_guard"]).min()) ** 2 / QNORM ** 2
    ctx.set_sign_poly(osign.cheb_coeffs(80, eps), eps, QNORM, M)
    ctx.set_lowmodes(u, nu)
    with pytest.raises(nd.NDError, match="enlarge nvec"):
        ctx.index_count(2, ZERO_TOL)                # the sector with two zero modes fills the whole block
    ctx.close()
