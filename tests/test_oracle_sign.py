"""Pins of the sign-function / Neuberger-Dirac oracle (oracle/sign.py): SURVEY.md section 8(c) P7-P11.  CPU only."""
import numpy as np
import pytest

from lattice_inputs import gauge_field, gaussian_spinor
from oracle import sign, wilson


# ------------------------------------------------------------------ P7 scalar polynomial
@pytest.mark.parametrize("n,eps", [(20, 0.05), (60, 0.01), (100, 0.005)])
def test_coefficients_interpolate_at_nodes(n, eps):
    """Chebyshev interpolation: P(y_j) = y_j^{-1/2} exactly at the n+1 nodes (defines the coefficients)."""
    c = sign.cheb_coeffs(n, eps)
    z = np.cos(np.pi * (np.arange(n + 1) + 0.5) / (n + 1))
    y = ((1 - eps) * z + 1 + eps) / 2
    assert np.allclose(sign.eval_P_scalar(c, eps, y) * np.sqrt(y), 1.0, atol=5e-13)


def test_scalar_clenshaw_is_chebval():
    c = sign.cheb_coeffs(50, 0.01)
    y = np.linspace(0.01, 1, 1001)
    ref = np.polynomial.chebyshev.chebval(sign.z_of_y(y, 0.01), c)       # sum_k c_k T_k(z), full c_0
    assert np.allclose(sign.eval_P_scalar(c, 0.01, y), ref, rtol=0, atol=1e-12)


@pytest.mark.parametrize("n,eps,delta_ref", [(100, 0.01, 5.4e-10), (100, 0.005, 2.5e-7), (100, 0.002, 5.9e-5),
                                              (200, 0.002, 5.6e-9), (200, 0.001, 1.3e-6)])
def test_delta_table(n, eps, delta_ref):
    """delta of eq. 2.6 for the interpolation coefficients (values tabulated in SURVEY.md 8(c)-A7), and the
    uniform bound |x P(x^2) - sign x| <= delta on sqrt(eps) <= |x| <= 1."""
    c = sign.cheb_coeffs(n, eps)
    d = sign.measure_delta(c, eps, npts=50001)
    assert 0.8 * delta_ref < d < 1.25 * delta_ref
    x = np.concatenate([-np.geomspace(np.sqrt(eps), 1, 5000), np.geomspace(np.sqrt(eps), 1, 5000)])
    assert np.max(np.abs(x * sign.eval_P_scalar(c, eps, x * x) - np.sign(x))) <= d * (1 + 1e-9) + 1e-15


def test_delta_decays_geometrically():
    """Textbook: the Chebyshev error for y^{-1/2} on [eps,1] decays like ((1-sqrt(eps))/(1+sqrt(eps)))^n."""
    eps = 0.01
    r = (1 - np.sqrt(eps)) / (1 + np.sqrt(eps))
    d40 = sign.measure_delta(sign.cheb_coeffs(40, eps), eps, 20001)
    d80 = sign.measure_delta(sign.cheb_coeffs(80, eps), eps, 20001)
    assert 0.5 * r ** 40 < d80 / d40 < 2.0 * r ** 40


# ------------------------------------------------------------------ P8-P11 on the dense 4^4 operator
def _setup(dense, l=8):
    Qmat, lam, W = dense["Qmat"], dense["lam"], dense["W"]
    dims = dense["dims"]
    shape = dims + (4, 3)
    Q = lambda v: (Qmat @ v.reshape(-1)).reshape(v.shape)
    S_exact = (W * np.sign(lam)) @ W.conj().T
    order = np.argsort(np.abs(lam))
    low = order[:l]
    qnorm = wilson.norm_bound_Q(dense["m"])
    return Q, S_exact, lam, W, low, order, qnorm, shape


def test_dense_matches_operator(dense_4x4_smooth):
    d = dense_4x4_smooth
    psi = gaussian_spinor(d["dims"])
    a = d["Qmat"] @ psi.ravel()
    b = wilson.apply_Q(psi, d["U"], d["m"]).ravel()
    assert np.linalg.norm(a - b) < 1e-13 * np.linalg.norm(b)
    assert np.abs(d["lam"]).max() <= wilson.norm_bound_Q(d["m"])


@pytest.mark.parametrize("n", [40, 60, 80])
def test_polynomial_sign_vs_exact(dense_4x4_smooth, n):
    """P8: || X P_n(X^2) eta - sign(Q) eta || <= delta ||eta|| when Q^2 >= eps ||Q||^2."""
    Q, S, lam, W, low, order, qnorm, shape = _setup(dense_4x4_smooth)
    eps = 0.99 * np.min(lam ** 2) / qnorm ** 2
    c = sign.cheb_coeffs(n, eps)
    delta = sign.measure_delta(c, eps, 50001)
    eta = gaussian_spinor(shape[:4])
    err = np.linalg.norm(sign.sign_poly(Q, eta, c, eps, qnorm).ravel() - S @ eta.ravel())
    assert err <= delta * np.linalg.norm(eta)
    assert err >= 1e-4 * delta * np.linalg.norm(eta)      # and the bound is not vacuous


def test_projected_sign_vs_exact(dense_4x4_smooth):
    """P8 with projection (eq. 2.11): exact eigenvectors in V -> same bound with eps set by the first
    mode outside V (reading R11); S u_k = sign(nu_k) u_k exactly."""
    Q, S, lam, W, low, order, qnorm, shape = _setup(dense_4x4_smooth, l=8)
    V = [W[:, i].reshape(shape) for i in low]
    nu, U = sign.rayleigh_ritz_Q(Q, V)
    assert np.allclose(np.sort(nu), np.sort(lam[low]), atol=1e-12)
    eps = 0.99 * lam[order[8]] ** 2 / qnorm ** 2
    n = 60
    c = sign.cheb_coeffs(n, eps)
    delta = sign.measure_delta(c, eps, 50001)
    eta = gaussian_spinor(shape[:4])
    got = sign.sign_projected(Q, eta, c, eps, qnorm, nu, U)
    assert np.linalg.norm(got.ravel() - S @ eta.ravel()) <= delta * np.linalg.norm(eta)
    for k in range(len(U)):
        su = sign.sign_projected(Q, U[k], c, eps, qnorm, nu, U)
        assert np.linalg.norm((su - np.sign(nu[k]) * U[k]).ravel()) < 1e-12
    assert np.all(sign.residues(Q, nu, U) < 1e-12)


def test_ginsparg_wilson(dense_4x4_smooth):
    """P9: gamma5 D + D gamma5 - (1/c) D gamma5 D = c gamma5 (1 - S^2): zero for the exact sign, bounded by
    c (2 delta + delta^2) ||eta|| for the polynomial; gamma5 D gamma5 = D^dagger."""
    Q, S, lam, W, low, order, qnorm, shape = _setup(dense_4x4_smooth)
    rho = 1.6
    cpre = 1.0 / rho
    g5 = lambda v: wilson.apply_gamma5(v)
    eta = gaussian_spinor(shape[:4])
    # exact
    D = lambda v: cpre * (v + g5((S @ v.ravel()).reshape(shape)))
    gw = g5(D(eta)) + D(g5(eta)) - (1 / cpre) * D(g5(D(eta)))
    assert np.linalg.norm(gw.ravel()) < 1e-12 * np.linalg.norm(eta)
    # polynomial
    eps = 0.99 * np.min(lam ** 2) / qnorm ** 2
    c = sign.cheb_coeffs(60, eps)
    delta = sign.measure_delta(c, eps, 50001)
    Dp = lambda v: sign.apply_DN(Q, g5, v, c, eps, qnorm, cpre)
    gw = g5(Dp(eta)) + Dp(g5(eta)) - (1 / cpre) * Dp(g5(Dp(eta)))
    assert np.linalg.norm(gw.ravel()) <= cpre * (2 * delta + delta ** 2) * np.linalg.norm(eta)
    chi = gaussian_spinor(shape[:4], 77)
    lhs = np.vdot(chi, g5(Dp(g5(eta))))       # <chi, g5 D g5 eta>
    rhs = np.vdot(Dp(chi), eta)               # <D chi, eta> = <chi, D^dagger eta>
    assert abs(lhs - rhs) < 1e-12 * np.linalg.norm(chi) * np.linalg.norm(eta)


def test_operator_count(dense_4x4_smooth):
    """P10: 2n+1 applications of Q per polynomial sign (reading R9)."""
    Q, *_rest, qnorm, shape = _setup(dense_4x4_smooth)
    calls = [0]

    def Qc(v):
        calls[0] += 1
        return Q(v)

    n = 17
    sign.sign_poly(Qc, gaussian_spinor(shape[:4]), sign.cheb_coeffs(n, 0.01), 0.01, qnorm)
    assert calls[0] == 2 * n + 1


def test_vector_clenshaw_equals_spectral(dense_4x4_smooth):
    """The vector recurrence equals the scalar polynomial applied in the eigenbasis: W P(lam^2/qnorm^2) W^dagger eta."""
    Q, S, lam, W, low, order, qnorm, shape = _setup(dense_4x4_smooth)
    eps, n = 0.004, 30
    c = sign.cheb_coeffs(n, eps)
    eta = gaussian_spinor(shape[:4])
    got = sign.clenshaw_P(Q, eta, c, eps, qnorm).ravel()
    p = sign.eval_P_scalar(c, eps, (lam / qnorm) ** 2)
    ref = W @ (p * (W.conj().T @ eta.ravel()))
    assert np.linalg.norm(got - ref) < 1e-12 * np.linalg.norm(ref)


def test_projection_algebra(dense_4x4_smooth):
    """P11: u_k orthonormal, PP^2 = PP, (1-PP) u_k = 0, also for a NON-invariant V (random rotation of
    eigenvectors plus noise), where eq. 2.7 is still well defined."""
    Q, S, lam, W, low, order, qnorm, shape = _setup(dense_4x4_smooth, l=6)
    rng = np.random.default_rng(5)
    from oracle.lowmodes import orthonormalise
    V = orthonormalise([W[:, i].reshape(shape) + 1e-3 * (rng.standard_normal(shape) + 1j * rng.standard_normal(shape))
                        for i in low])
    nu, U = sign.rayleigh_ritz_Q(Q, V)
    G = np.array([[sign.vdot(a, b) for b in U] for a in U])
    assert np.abs(G - np.eye(len(U))).max() < 1e-12
    eta = gaussian_spinor(shape[:4])
    P = lambda v: sum(sign.vdot(u, v) * u for u in U)
    assert np.linalg.norm((P(P(eta)) - P(eta)).ravel()) < 1e-12 * np.linalg.norm(eta)
    # PP Q u_k = nu_k u_k
    for n_k, u in zip(nu, U):
        assert np.linalg.norm((P(Q(u)) - n_k * u).ravel()) < 1e-12


def test_free_field_DN_closed_form():
    """P3 for D_N: on a free-field plane wave sign Q(p) = Q(p)/omega(p), so
    D_N(p) w = c [1 + (M + i sum gamma_mu sin p_mu)/omega] w - holds at any lattice size."""
    dims = (8, 4, 4, 4)
    U = gauge_field(dims, "unit")
    m, cpre = -1.6, 1 / 1.6
    qnorm = wilson.norm_bound_Q(m)
    g, g5m = wilson.gamma_matrices()
    # free-field spectral range of Q^2 over all momenta of this lattice
    lo = np.inf
    for n0 in range(8):
        for n1 in range(4):
            for n2 in range(4):
                for n3 in range(4):
                    p = np.array([(2 * n0 + 1) * np.pi / 8, 2 * np.pi * n1 / 4, 2 * np.pi * n2 / 4, 2 * np.pi * n3 / 4])
                    lo = min(lo, (4 + m - np.cos(p).sum()) ** 2 + (np.sin(p) ** 2).sum())
    eps = 0.99 * lo / qnorm ** 2
    c = sign.cheb_coeffs(100, eps)
    delta = sign.measure_delta(c, eps, 50001)
    Q = lambda v: wilson.apply_Q(v, U, m)
    rng = np.random.default_rng(3)
    w = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
    n = (1, 1, 0, 3)
    p = np.array([(2 * n[0] + 1) * np.pi / 8] + [2 * np.pi * n[i] / 4 for i in (1, 2, 3)])
    grids = np.meshgrid(*[np.arange(d) for d in dims], indexing="ij")
    phase = np.exp(1j * sum(p[i] * grids[i] for i in range(4)))
    psi = phase[..., None, None] * w
    M = 4 + m - np.cos(p).sum()
    om = np.sqrt(M * M + (np.sin(p) ** 2).sum())
    Dp = M * np.eye(4) + 1j * sum(g[mu] * np.sin(p[mu]) for mu in range(4))
    expect = phase[..., None, None] * (cpre * (w + (Dp @ w) / om))
    got = sign.apply_DN(Q, wilson.apply_gamma5, psi, c, eps, qnorm, cpre)
    assert np.linalg.norm((got - expect).ravel()) <= cpre * delta * np.linalg.norm(psi.ravel())


# ------------------------------------------------------------------------------- min-max coefficients (eq. 2.6)
def test_minmax_degree_zero_closed_form():
    """n = 0: minimise max |1 - c0 sqrt(y)| on [eps, 1]: the error is monotone, so it is levelled at the two end points:
    c0 = 2 / (1 + sqrt(eps)), delta = (1 - sqrt(eps)) / (1 + sqrt(eps)) - by hand."""
    for eps in (0.04, 0.25, 0.0025):
        c, delta, E = sign.minmax_coeffs(0, eps)
        r = np.sqrt(eps)
        assert abs(c[0] - 2.0 / (1.0 + r)) < 1e-14 and abs(delta - (1.0 - r) / (1.0 + r)) < 1e-14 and abs(E - delta) < 1e-14


@pytest.mark.parametrize("n,eps", [(8, 0.1), (20, 0.05), (40, 0.01), (100, 0.005), (100, 0.002)])
def test_minmax_equioscillates_and_beats_interpolation(n, eps):
    """Chebyshev's alternation theorem pins the min-max polynomial of eq. 2.6: the error 1 - sqrt(y) P(y) attains +-delta at
    n + 2 points with alternating signs (then P is THE minimiser), de la Vallee-Poussin sandwiches the optimum,
    E <= delta_min <= delta, and delta is below the interpolation polynomial's at the same degree."""
    c, delta, E = sign.minmax_coeffs(n, eps)
    assert E <= delta <= 1.002 * E
    z = -np.cos(np.pi * (np.arange(200 * (n + 2)) + 0.5) / (200 * (n + 2)))
    y = np.concatenate([[eps], ((1 - eps) * z + 1 + eps) / 2, [1.0]])
    e = 1.0 - np.sqrt(y) * sign.eval_P_scalar(c, eps, y)
    assert np.abs(e).max() <= delta * (1 + 1e-9)
    big = np.flatnonzero(np.abs(e) >= 0.995 * delta)
    signs = np.sign(e[big])
    alternations = 1 + int(np.sum(signs[1:] != signs[:-1]))
    assert alternations == n + 2
    ci = sign.cheb_coeffs(n, eps)
    assert delta < 0.75 * sign.measure_delta(ci, eps)
    # the sign-function form of eq. 2.5 obeys the same bound on sqrt(eps) <= |x| <= 1
    x = np.concatenate([-np.geomspace(1.0, np.sqrt(eps), 4001), np.geomspace(np.sqrt(eps), 1.0, 4001)])
    assert np.abs(x * sign.eval_P_scalar(c, eps, x * x) - np.sign(x)).max() <= delta * (1 + 1e-9)


def test_minmax_polynomial_is_a_valid_sign_approximation_on_vectors(dense_4x4_smooth):
    """The coefficient array is an input of the recipe: with the min-max coefficients the polynomial sign function stays
    within ITS (smaller) delta of the exact dense sign - uniformly in eta, which the operator norm on the
    dense spectrum checks."""
    d4 = dense_4x4_smooth
    lam, W, Qmat = d4["lam"], d4["W"], d4["Qmat"]
    shape = tuple(d4["dims"]) + (4, 3)
    Q = lambda v: (Qmat @ v.reshape(-1)).reshape(shape)
    eta = gaussian_spinor(d4["dims"])
    qnorm = 6.4
    eps = 0.99 * (lam ** 2).min() / qnorm ** 2
    S = ((W * np.sign(lam)) @ W.conj().T @ eta.reshape(-1)).reshape(shape)
    n = 40
    errs = {}
    for name, (c, delta) in {"minmax": sign.minmax_coeffs(n, eps)[:2], "interp": (sign.cheb_coeffs(n, eps), None)}.items():
        delta = sign.measure_delta(c, eps) if delta is None else delta
        errs[name] = np.linalg.norm((sign.sign_poly(Q, eta, c, eps, qnorm) - S).ravel()) / np.linalg.norm(eta.ravel())
        assert errs[name] <= delta
        x = lam / qnorm
        assert np.abs(x * sign.eval_P_scalar(c, eps, x * x) - np.sign(x)).max() <= delta      # || X P(X^2) - sign Q || <= delta
