"""Pins of the oracle's error control of the low-mode projectors (section 2.3, eq. 2.8-2.10): closed-form values
of eq. 2.10, kappa = 0 for exact eigenvectors, and the inequality itself checked against the EXACT projector deviation
from the dense 4^4 eigendecomposition for perturbed low-mode spaces of growing error."""
import numpy as np
import pytest

from lattice_inputs import gaussian_spinor
from oracle import lowmodes as olow
from oracle import sign


def test_bound_closed_form_values():
    """eq. 2.10 evaluated by hand: kappa = 0.1 -> 0.1*1.2/(1-0.24) = 0.157894...; kappa = 0 -> 0; the denominator
    vanishes at 2k(1+2k) = 1, i.e. k = (sqrt(5)-1)/4 = 0.30901..."""
    assert abs(olow.projector_bound(0.1) - 0.12 / 0.76) < 1e-15
    assert olow.projector_bound(0.0) == 0.0
    kc = (np.sqrt(5.0) - 1.0) / 4.0
    assert olow.projector_bound(kc - 1e-9) > 1e7 and olow.projector_bound(kc + 1e-9) == float("inf")
    # small kappa: bound = kappa + O(kappa^2)
    assert abs(olow.projector_bound(1e-6) / 1e-6 - 1) < 1e-5


def test_kappa_definition_by_hand():
    nu = np.array([0.5, -0.4, 0.7])
    rho = np.array([0.01, 0.02, 0.03])
    d = np.array([0.1, 0.2, 0.3])
    kp, km = olow.kappa_pm(nu, rho, d)
    assert abs(kp - np.sqrt(0.1 ** 2 + 0.1 ** 2)) < 1e-15 and abs(km - 0.1) < 1e-15
    # d_k by hand: nu_0 = 0.5 > 0 sees the rest {0.9, -0.8} and the projected negative value -0.4 -> 0.4
    dd = olow.distances_d(nu, [0.9, -0.8])
    assert np.allclose(dd, [0.4, 0.4, 0.2])


def test_projector_bound_holds_on_dense_4x4(dense_4x4_smooth):
    d4 = dense_4x4_smooth
    lam, W, Qmat = d4["lam"], d4["W"], d4["Qmat"]
    shape = tuple(d4["dims"]) + (4, 3)
    l = 8
    low = np.argsort(lam * lam)[:l]
    rest = np.delete(lam, low)
    Q = lambda v: (Qmat @ v.reshape(-1)).reshape(shape)
    Ep, Em = W[:, low[lam[low] > 0]], W[:, low[lam[low] < 0]]      # exact eigenvectors of the projected modes

    def deviation(A, B):
        """|| A A^dagger - B B^dagger ||_2 for orthonormal column blocks: sine of the largest principal angle when the
        ranks agree, 1 otherwise."""
        if A.shape[1] != B.shape[1]:
            return 1.0
        if A.shape[1] == 0:
            return 0.0
        sv = np.linalg.svd(B.conj().T @ A, compute_uv=False)
        return float(np.sqrt(max(0.0, 1.0 - sv.min() ** 2)))

    rng = np.random.default_rng(11)
    seen_finite = 0
    for noise in (0.0, 1e-6, 1e-5, 1e-4, 3e-4, 1e-3):
        V = olow.orthonormalise([W[:, i].reshape(shape) + noise * (rng.standard_normal(shape) + 1j * rng.standard_normal(shape))
                                 for i in low])
        nu, U = sign.rayleigh_ritz_Q(Q, V)
        rho = sign.residues(Q, nu, U)
        d = olow.distances_d(nu, rest)
        kp, km = olow.kappa_pm(nu, rho, d)
        Um = np.stack([u.reshape(-1) for u in U], axis=1)
        devp = deviation(Um[:, nu > 0], Ep)
        devm = deviation(Um[:, nu < 0], Em)
        print(noise, kp, km, devp, devm, olow.projector_bound(kp))
        if noise == 0.0:
            assert kp < 1e-10 and km < 1e-10 and devp < 1e-7 and devm < 1e-7
        assert devp <= olow.projector_bound(kp) + 1e-7 and devm <= olow.projector_bound(km) + 1e-7
        seen_finite += np.isfinite(olow.projector_bound(kp))
        # the bound is not vacuous: the deviation is at least a fair fraction of kappa's scale for the noisy spaces
        if noise >= 1e-4 and np.isfinite(olow.projector_bound(kp)):
            assert devp > 0.01 * kp
    assert seen_finite >= 3


# ------------------------------------------------------------------------- dynamic choice of l (R17)
def test_choose_l_hand_made_spectra():
    """The gap rule on spectra written by hand: a cluster straddling a fixed cut is never split when the window allows."""
    a = np.array([0.10, 0.11, 0.30, 0.301, 0.302, 0.50, 0.90])
    assert olow.choose_l(a, 3, 5) == (5, pytest.approx(0.198))          # the cluster 0.300-0.302 stays together
    assert olow.choose_l(a, 2, 4)[0] == 2                                # gap 0.19 below the cluster beats 0.001 inside it
    assert olow.choose_l(a, 3, 4)[0] == 3                                # forced inside the cluster: a tie goes to the smallest l
    assert olow.choose_l(a, 4, 4) == (4, pytest.approx(0.001))           # no freedom: the (small) gap is reported
    b = np.array([0.1, 0.2, 0.3, 0.3001, 0.6, 0.7])
    assert olow.choose_l(b, 3, 4)[0] == 4                                # the pair (0.3, 0.3001) straddles l = 3
    with pytest.raises(AssertionError):
        olow.choose_l(b, 3, 6)                                           # no value beyond the last candidate
    with pytest.raises(AssertionError):
        olow.choose_l(b[::-1], 2, 3)                                     # not sorted


def test_choose_l_is_the_argmax_of_the_gaps_on_the_dense_spectrum(dense_4x4_smooth):
    lam = dense_4x4_smooth["lam"]
    a = np.sort(np.abs(lam))
    for lo, hi in ((4, 12), (8, 24), (1, 40)):
        l, gap = olow.choose_l(a, lo, hi)
        gaps = a[lo:hi + 1] - a[lo - 1:hi]
        assert gap == gaps.max() and l == lo + int(np.argmax(gaps))


def test_gap_rule_lowers_kappa_for_a_perturbed_low_space(dense_4x4_smooth):
    """Why the rule exists: with Ritz vectors of a given (finite) accuracy, cutting at the largest gap of the window gives
    a smaller kappa (eq. 2.9) - hence a smaller bound (2.10) on the projector error - than cutting inside the tightest
    cluster of the same window, and the true projector deviation follows."""
    d4 = dense_4x4_smooth
    lam, W, Qmat = d4["lam"], d4["W"], d4["Qmat"]
    shape = tuple(d4["dims"]) + (4, 3)
    Q = lambda v: (Qmat @ v.reshape(-1)).reshape(shape)
    order = np.argsort(np.abs(lam))
    a = np.abs(lam[order])
    lo, hi, k = 6, 20, 28
    l_gap, gap = olow.choose_l(a, lo, hi)
    gaps = a[lo:hi + 1] - a[lo - 1:hi]
    l_bad = lo + int(np.argmin(gaps))
    assert gaps.min() < 0.2 * gap
    rng = np.random.default_rng(5)
    V = olow.orthonormalise([W[:, i].reshape(shape) + 2e-7 * (rng.standard_normal(shape) + 1j * rng.standard_normal(shape))
                             for i in order[:k]])
    nu, U = sign.rayleigh_ritz_Q(Q, V)
    rho = sign.residues(Q, nu, U)
    o = np.argsort(np.hypot(nu, rho))            # the block is ordered by a_j = ||Q u_j|| (R17)
    nu, U, rho = nu[o], [U[i] for i in o], rho[o]
    ec = olow.error_control(nu, rho, lo, hi)
    assert ec["l"] == l_gap                                              # Ritz values this accurate reproduce the exact choice
    bad = olow.error_control(nu, rho, l_bad, l_bad)
    assert max(ec["kappa"]) < 0.5 * max(bad["kappa"])
    assert np.isfinite(ec["bound"][0]) and np.isfinite(ec["bound"][1])
    # the bound holds at the chosen cut (exact projectors from the dense decomposition)
    Um = np.stack([u.reshape(-1) for u in U[:ec["l"]]], axis=1)
    low = order[:ec["l"]]
    for sgn, i in ((1, 0), (-1, 1)):
        E = W[:, low[sgn * lam[low] > 0]]
        A = Um[:, sgn * nu[:ec["l"]] > 0]
        assert A.shape[1] == E.shape[1]
        sv = np.linalg.svd(E.conj().T @ A, compute_uv=False)
        assert np.sqrt(max(0.0, 1.0 - sv.min() ** 2)) <= ec["bound"][i] + 1e-9
