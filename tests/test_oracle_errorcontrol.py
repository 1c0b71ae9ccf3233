"""Pins of the oracle's error control of the low-mode projectors (section 2.3, eq. 2.8-2.10): closed-form values
of eq. 2.10, kappa = 0 for exact eigenvectors, and the inequality itself checked against the EXACT projector deviation
from the dense 4^4 eigendecomposition for perturbed low-mode spaces of growing error."""
import numpy as np

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
