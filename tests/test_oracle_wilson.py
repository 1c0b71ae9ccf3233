"""Pins of the Wilson-Dirac oracle (oracle/wilson.py) against what PAPER.md and the mathematics fix.
SURVEY.md section 8(c) pins P1-P5.  CPU only."""
import itertools

import numpy as np
import pytest

from lattice_inputs import SEED_TRANSFORM, gauge_field, gaussian_spinor, haar_su3
from oracle import wilson

I = 1j
# The chiral basis of DESIGN.md reading R2 typed out entry by entry (independent of oracle.wilson.gamma_matrices).
G_HAND = [
    np.array([[0, 0, -1, 0], [0, 0, 0, -1], [-1, 0, 0, 0], [0, -1, 0, 0]], dtype=complex),
    np.array([[0, 0, 0, -I], [0, 0, -I, 0], [0, I, 0, 0], [I, 0, 0, 0]], dtype=complex),
    np.array([[0, 0, 0, -1], [0, 0, 1, 0], [0, 1, 0, 0], [-1, 0, 0, 0]], dtype=complex),
    np.array([[0, 0, -I, 0], [0, 0, 0, I], [I, 0, 0, 0], [0, -I, 0, 0]], dtype=complex),
]
G5_HAND = np.diag([1, 1, -1, -1]).astype(complex)


def rel(a, b):
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel())


def test_gamma_algebra():
    g, g5 = wilson.gamma_matrices()
    for mu in range(4):
        assert np.array_equal(g[mu], G_HAND[mu])
        assert np.allclose(g[mu], g[mu].conj().T)
        for nu in range(4):
            assert np.allclose(g[mu] @ g[nu] + g[nu] @ g[mu], 2.0 * (mu == nu) * np.eye(4))
        assert np.allclose(g5 @ g[mu] + g[mu] @ g5, 0)
    assert np.allclose(g5, G5_HAND)


@pytest.mark.parametrize("bc", [-1, 1])
@pytest.mark.parametrize("y", [(1, 2, 0, 3), (0, 0, 0, 0), (3, 3, 3, 3)])
def test_point_source_by_hand(bc, y):
    """P1: eq. 2.1 applied to a point source, every non-zero output written out by hand.
    The only pin of hop direction / which of (1 -+ gamma) goes with which hop / link dagger / colour order."""
    dims = (4, 4, 4, 4)
    U = gauge_field(dims, "haar", seed=3)
    m = 0.1
    for beta, b in [(0, 0), (1, 2), (2, 1), (3, 0)]:
        src = np.zeros(dims + (4, 3), dtype=complex)
        src[y + (beta, b)] = 1.0
        e_spin = np.zeros(4, dtype=complex)
        e_spin[beta] = 1
        e_col = np.zeros(3, dtype=complex)
        e_col[b] = 1
        expect = np.zeros_like(src)
        expect[y] += (4 + m) * np.outer(G5_HAND @ e_spin, e_col)
        for mu in range(4):
            # x = y - mu^ receives the forward hop  -1/2 gamma5 U_mu(x) (1 - gamma_mu) psi(x + mu^)
            x = list(y)
            x[mu] -= 1
            ph = 1.0
            if x[mu] < 0:
                x[mu] += dims[mu]
                ph = bc if mu == 0 else 1.0       # x0 = T-1 -> 0 crosses the seam
            x = tuple(x)
            expect[x] += -0.5 * ph * np.outer(G5_HAND @ (np.eye(4) - G_HAND[mu]) @ e_spin, U[(mu,) + x] @ e_col)
            # x = y + mu^ receives the backward hop  -1/2 gamma5 U_mu(x - mu^)^dagger (1 + gamma_mu) psi(x - mu^)
            x = list(y)
            x[mu] += 1
            ph = 1.0
            if x[mu] >= dims[mu]:
                x[mu] -= dims[mu]
                ph = bc if mu == 0 else 1.0       # x0 = 0 -> T-1 crosses the seam
            x = tuple(x)
            expect[x] += -0.5 * ph * np.outer(G5_HAND @ (np.eye(4) + G_HAND[mu]) @ e_spin,
                                              U[(mu,) + y].conj().T @ e_col)
        got = wilson.apply_Q(src, U, m, bc)
        assert np.count_nonzero(np.abs(got).sum(axis=(4, 5))) == 9
        assert np.allclose(got, expect, atol=1e-14)


@pytest.mark.parametrize("kind", ["haar", "smooth"])
def test_hermiticity(kind):
    """P2: Q = gamma5 D_W is Hermitian."""
    dims = (4, 4, 4, 4)
    U = gauge_field(dims, kind)
    psi, chi = gaussian_spinor(dims, 1), gaussian_spinor(dims, 2)
    for m in (0.1, -1.6):
        Qpsi, Qchi = wilson.apply_Q(psi, U, m), wilson.apply_Q(chi, U, m)
        lhs, rhs = np.vdot(chi, Qpsi), np.vdot(Qchi, psi)
        assert abs(lhs - rhs) <= 1e-13 * np.linalg.norm(chi) * np.linalg.norm(Qpsi)


def _plane_wave(dims, n, w, bc):
    """e^{ipx} w with p_0 = (2 n_0 + 1) pi / T (antiperiodic) or 2 pi n_0 / T, p_i = 2 pi n_i / L_i."""
    p = [((2 * n[0] + 1) if bc == -1 else 2 * n[0]) * np.pi / dims[0]] + [2 * np.pi * n[i] / dims[i] for i in (1, 2, 3)]
    grids = np.meshgrid(*[np.arange(d) for d in dims], indexing="ij")
    phase = np.exp(1j * sum(p[i] * grids[i] for i in range(4)))
    return np.array(p), phase[..., None, None] * w


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (8, 4, 4, 4), (6, 4, 2, 4)])
@pytest.mark.parametrize("bc", [-1, 1])
def test_free_field_plane_wave(dims, bc):
    """P3: unit links, D_W(p) = M + i sum gamma_mu sin p_mu, M = 4 + m - sum cos p_mu (textbook closed form)."""
    U = gauge_field(dims, "unit")
    rng = np.random.default_rng(0)
    for n in [(0, 0, 0, 0), (1, 2, 0, 1), (3, 1, 1, 3)]:
        w = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
        for m in (0.1, -1.6):
            p, psi = _plane_wave(dims, n, w, bc)
            M = 4 + m - np.cos(p).sum()
            Dp = M * np.eye(4) + 1j * sum(G_HAND[mu] * np.sin(p[mu]) for mu in range(4))
            Qw = G5_HAND @ Dp @ w
            phase = psi[..., 0, 0] / w[0, 0]
            expect = phase[..., None, None] * Qw
            got = wilson.apply_Q(psi, U, m, bc)
            assert rel(got, expect) < 1e-13
            # Q(p)^2 = (M^2 + sum sin^2 p) 1
            got2 = wilson.apply_Q(got, U, m, bc)
            assert rel(got2, (M * M + (np.sin(p) ** 2).sum()) * psi) < 1e-13


def test_free_field_dense_spectrum():
    """P3/P5: the dense 4^4 free spectrum is +-sqrt(M^2 + sum sin^2 p), six-fold per momentum and sign."""
    dims = (4, 4, 4, 4)
    m = 0.1
    Qmat = wilson.dense_Q(gauge_field(dims, "unit"), m)
    assert np.abs(Qmat - Qmat.conj().T).max() < 1e-14
    lam = np.linalg.eigvalsh(Qmat)
    om = []
    for n in itertools.product(range(4), repeat=4):
        p = np.array([(2 * n[0] + 1) * np.pi / 4] + [2 * np.pi * n[i] / 4 for i in (1, 2, 3)])
        w = np.sqrt((4 + m - np.cos(p).sum()) ** 2 + (np.sin(p) ** 2).sum())
        om += [w] * 6 + [-w] * 6
    assert np.allclose(np.sort(lam), np.sort(om), atol=1e-12)


@pytest.mark.parametrize("kind", ["haar", "smooth"])
def test_gauge_covariance(kind):
    """P4: U'_mu(x) = G(x) U_mu(x) G(x+mu^)^dagger, psi' = G psi  =>  Q[U'] psi' = G Q[U] psi."""
    dims = (4, 4, 4, 4)
    U = gauge_field(dims, kind)
    psi = gaussian_spinor(dims)
    rng = np.random.Generator(np.random.PCG64(SEED_TRANSFORM))
    G = haar_su3(int(np.prod(dims)), rng).reshape(dims + (3, 3))
    Up = np.empty_like(U)
    for mu in range(4):
        Gf = np.roll(G, -1, axis=mu)
        Up[mu] = np.einsum("...ab,...bc,...dc->...ad", G, U[mu], Gf.conj())
    gpsi = np.einsum("...ab,...sb->...sa", G, psi)
    lhs = wilson.apply_Q(gpsi, Up, -1.6)
    rhs = np.einsum("...ab,...sb->...sa", G, wilson.apply_Q(psi, U, -1.6))
    assert rel(lhs, rhs) < 1e-14


@pytest.mark.parametrize("dims", [(4, 3, 2, 2), (2, 2, 3, 4)])
@pytest.mark.parametrize("bc", [-1, 1])
def test_vectorised_equals_literal_site_loop(dims, bc):
    """Brute force: eq. 2.1 + 2.2 read literally (8 signed directions, matrix inverse) on tiny lattices,
    including extent-2 directions where x+mu^ and x-mu^ coincide."""
    U = gauge_field(dims, "haar", seed=5)
    psi = gaussian_spinor(dims, 6)
    a = wilson.apply_Q(psi, U, 0.1, bc)
    b = wilson.apply_Q_literal(psi, U, 0.1, bc)
    assert rel(a, b) < 1e-14


def test_dense_properties():
    """P5: dense 4^4 Haar: Hermitian, ||Q|| <= |4+m|+4, Q(m1) - Q(m2) = (m1 - m2) gamma5, matrix = operator."""
    dims = (4, 4, 4, 4)
    U = gauge_field(dims, "haar")
    Q1 = wilson.dense_Q(U, 0.1)
    assert np.abs(Q1 - Q1.conj().T).max() < 1e-14
    lam = np.linalg.eigvalsh(Q1)
    assert np.abs(lam).max() <= wilson.norm_bound_Q(0.1)
    psi = gaussian_spinor(dims)
    assert rel(Q1 @ psi.ravel(), wilson.apply_Q(psi, U, 0.1).ravel()) < 1e-14
    # mass dependence on a few columns (full second dense build is not needed)
    g5 = np.kron(np.eye(256), np.kron(G5_HAND, np.eye(3)))
    for col in (0, 517, 3071):
        e = np.zeros(3072, dtype=complex)
        e[col] = 1
        d = wilson.apply_Q(e.reshape(dims + (4, 3)), U, -1.6).ravel() - Q1[:, col]
        assert np.allclose(d, (-1.6 - 0.1) * g5[:, col], atol=1e-14)
