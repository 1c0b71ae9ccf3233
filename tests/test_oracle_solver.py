"""Pins of oracle/solver.py (massive operator + CG): the dense 4^4 operator with the EXACT sign function and a library
direct solve, the free-field closed form, gamma5-Hermiticity, and the consistency of the reading R16 with the factor
of eq. 2.12."""
import numpy as np

from lattice_inputs import gauge_field, gaussian_spinor
from oracle import sign, solver, wilson

RHO = 1.6


def test_dense_4x4_direct_solve(dense_4x4_smooth):
    d = dense_4x4_smooth
    lam, W = d["lam"], d["W"]
    S = (W * np.sign(lam)) @ W.conj().T          # exact sign(Q) from the dense eigendecomposition (pin P8)
    shape = tuple(d["dims"]) + (4, 3)
    n = S.shape[0]
    g5 = np.kron(np.eye(n // 12), np.kron(np.diag([1.0, 1.0, -1.0, -1.0]), np.eye(3)))
    abar, mq = 1.0 / RHO, 0.05
    DN = (1.0 / abar) * (np.eye(n) + g5 @ S)
    Dm = (1.0 - 0.5 * abar * mq) * DN + mq * np.eye(n)
    # the function agrees with the matrix, gamma5 D gamma5 = D^dagger
    eta = gaussian_spinor(d["dims"])
    got = solver.apply_DNm(lambda v: (DN @ v.ravel()).reshape(shape), eta, abar, mq)
    assert np.allclose(got.ravel(), Dm @ eta.ravel(), rtol=0, atol=1e-12)
    assert np.abs(g5 @ Dm @ g5 - Dm.conj().T).max() < 1e-12
    # spectrum of D^dagger D: mq^2 <= eig <= (2/abar)^2  (D_N normal with eigenvalues on the circle |z - 1/abar| = 1/abar)
    rng = np.random.default_rng(2)
    for _ in range(4):
        v = rng.standard_normal(n) + 1j * rng.standard_normal(n)
        q = np.linalg.norm(Dm @ v) / np.linalg.norm(v)
        assert mq - 1e-12 <= q <= 2.0 / abar + 1e-12
    # CG = direct solve
    D = lambda v: (Dm @ v.ravel()).reshape(shape)
    Dd = lambda v: (Dm.conj().T @ v.ravel()).reshape(shape)
    x, it, res = solver.cg_normal_equations(D, Dd, eta, 1e-10, 2000)
    ref = np.linalg.solve(Dm, eta.ravel())
    assert np.linalg.norm(x.ravel() - ref) <= 1e-7 * np.linalg.norm(ref) and res < 1e-8 and it < 2000


def test_free_field_closed_form_inverse():
    """Unit links: on a plane wave D_N^m(p) = (1/abar + m/2) + (1/abar - m/2) (M + i sum gamma_mu sin p_mu)/omega, a 4x4
    matrix per momentum; its inverse applied to the spin-colour vector is the solution."""
    dims = (8, 4, 4, 4)
    U = gauge_field(dims, "unit")
    m = -RHO
    qnorm = wilson.norm_bound_Q(m)
    abar, mq = 1.0 / RHO, 0.1
    eps = 0.99 * 0.25 / qnorm ** 2          # free-field floor of Q^2 on this lattice is 0.251
    c = sign.cheb_coeffs(80, eps)
    delta = sign.measure_delta(c, eps, 20001)
    Q = lambda v: wilson.apply_Q(v, U, m)
    DN = lambda v: sign.apply_DN(Q, wilson.apply_gamma5, v, c, eps, qnorm, 1.0 / abar)
    D = lambda v: solver.apply_DNm(DN, v, abar, mq)
    Dd = lambda v: wilson.apply_gamma5(D(wilson.apply_gamma5(v)))
    g, _ = wilson.gamma_matrices()
    n = (2, 1, 3, 0)
    p = np.array([(2 * n[0] + 1) * np.pi / 8] + [2 * np.pi * n[i] / 4 for i in (1, 2, 3)])
    grids = np.meshgrid(*[np.arange(dd) for dd in dims], indexing="ij")
    phase = np.exp(1j * sum(p[i] * grids[i] for i in range(4)))
    rng = np.random.default_rng(4)
    w = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
    b = phase[..., None, None] * w
    Mp = 4 + m - np.cos(p).sum()
    om = np.sqrt(Mp ** 2 + (np.sin(p) ** 2).sum())
    Dp = (1 / abar + mq / 2) * np.eye(4) + (1 / abar - mq / 2) * (Mp * np.eye(4) + 1j * sum(g[mu] * np.sin(p[mu]) for mu in range(4))) / om
    ref = phase[..., None, None] * (np.linalg.inv(Dp) @ w)
    x, it, res = solver.cg_normal_equations(D, Dd, b, 1e-9, 200)
    assert res < 1e-7
    assert np.linalg.norm((x - ref).ravel()) <= (2 * delta / abar / mq + 1e-7) * np.linalg.norm(ref.ravel())


def test_reading_R16_reproduces_the_factor_of_eq_2_12():
    """An error E in sign(Q) changes D_N^m by (1 - abar m/2)(1/abar) gamma5 E: with abar = a/(1+s) and a = 1 this is
    (1 + s - m/2) E, and eq. 2.12 quotes (2/a)(1 + s - a m/2)(kappa_+ + kappa_-) for ||E|| <= 2 (kappa_+ + kappa_-)."""
    s_, mq = 0.6, 0.3
    abar = 1.0 / (1.0 + s_)
    factor = (1.0 - 0.5 * abar * mq) / abar
    assert abs(factor - (1.0 + s_ - 0.5 * mq)) < 1e-15
