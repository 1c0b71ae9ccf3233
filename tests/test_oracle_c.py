"""Pins of the plain-C oracle (oracle/wilson_ref.c via oracle/wilson_c.py) and of oracle/lowmodes.py.  CPU only.

The C file restates eq. 2.1 as a site loop; it is pinned (a) against the numpy oracle, which
is itself pinned by tests/test_oracle_wilson.py, and (b) directly against the invariants again at a size numpy
would be slow at (Hermiticity, free-field closed form at 8^3x16)."""
import numpy as np
import pytest

from lattice_inputs import gauge_field, gaussian_spinor
from oracle import lowmodes, wilson, wilson_c


def rel(a, b):
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel())


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (6, 4, 2, 4), (2, 2, 3, 4)])
@pytest.mark.parametrize("bc", [-1, 1])
@pytest.mark.parametrize("kind", ["haar", "smooth"])
def test_c_equals_numpy(dims, bc, kind):
    U = gauge_field(dims, kind, seed=21)
    psi = gaussian_spinor(dims, 22)
    for m in (0.1, -1.6):
        assert rel(wilson_c.apply_Q(psi, U, m, bc), wilson.apply_Q(psi, U, m, bc)) < 1e-14


def test_c_hermitian_and_free_field_8c16():
    dims = (16, 8, 8, 8)
    U = gauge_field(dims, "smooth", eps=0.3)
    psi, chi = gaussian_spinor(dims, 1), gaussian_spinor(dims, 2)
    Qpsi, Qchi = wilson_c.apply_Q(psi, U, -1.6), wilson_c.apply_Q(chi, U, -1.6)
    assert abs(np.vdot(chi, Qpsi) - np.vdot(Qchi, psi)) <= 1e-13 * np.linalg.norm(chi) * np.linalg.norm(Qpsi)
    # free field: Q^2 on a plane wave = (M^2 + sum sin^2 p) (textbook)
    U1 = gauge_field(dims, "unit")
    n = (3, 1, 5, 2)
    p = np.array([(2 * n[0] + 1) * np.pi / 16] + [2 * np.pi * n[i] / 8 for i in (1, 2, 3)])
    grids = np.meshgrid(*[np.arange(d) for d in dims], indexing="ij")
    w = np.arange(12).reshape(4, 3) + 1j
    pw = np.exp(1j * sum(p[i] * grids[i] for i in range(4)))[..., None, None] * w
    M = 4 - 1.6 - np.cos(p).sum()
    got = wilson_c.apply_Q(wilson_c.apply_Q(pw, U1, -1.6), U1, -1.6)
    assert rel(got, (M * M + (np.sin(p) ** 2).sum()) * pw) < 1e-13


def test_lowmodes_dense_vs_eigsh(dense_4x4_smooth):
    """P12 (oracle side): library Lanczos on the oracle's Q^2 reproduces the dense lowest eigenvalues; the dense
    pairs satisfy Q^2 v = theta v and nu_k^2 = theta_k."""
    d = dense_4x4_smooth
    l = 6
    theta, V = lowmodes.lowest_modes_dense(d["Qmat"], l)
    Q2 = d["Qmat"] @ d["Qmat"]
    assert np.abs(Q2 @ V - V * theta).max() < 1e-11
    assert np.allclose(theta, np.sort(d["lam"] ** 2)[:l], atol=1e-12)
    Q = wilson_c.make_Q(d["U"], d["m"])
    th2, vecs, nmv = lowmodes.lowest_modes_eigsh(Q, d["dims"] + (4, 3), l, tol=1e-10)
    assert np.allclose(th2, theta, atol=1e-8)
    assert nmv > 0
    for t, v in zip(th2, vecs):
        assert np.linalg.norm((Q(Q(v)) - t * v).ravel()) < 1e-6


def test_orthonormalise_and_filter_space():
    dims = (4, 4, 4, 4)
    U = gauge_field(dims, "smooth", eps=0.3)
    Q = wilson_c.make_Q(U, -1.6)
    V = lowmodes.approximate_low_space(Q, dims + (4, 3), 4, wilson.norm_bound_Q(-1.6), cut=1.0, degree=8, sweeps=1)
    G = np.array([[np.vdot(a, b) for b in V] for a in V])
    assert np.abs(G - np.eye(4)).max() < 1e-12
    # the filter lowers the Rayleigh quotient of Q^2 relative to a random vector (mean of spectrum ~ 20)
    rq = [np.vdot(v, Q(Q(v))).real for v in V]
    assert max(rq) < 10.0
