"""P6: SU(3) compression round trips of the oracle (oracle/su3.py), eq. 2.3."""
import numpy as np
import pytest

from lattice_inputs import haar_su3, smooth_su3, unit_su3
from oracle import su3


def _fields():
    rng = np.random.Generator(np.random.PCG64(99))
    return {"haar": haar_su3(20000, rng), "smooth0.3": smooth_su3(20000, 0.3, rng), "smooth0.25": smooth_su3(20000, 0.25, rng)}


@pytest.mark.parametrize("name", ["haar", "smooth0.3", "smooth0.25"])
def test_recon12(name):
    U = _fields()[name]
    assert np.abs(su3.reconstruct12_cols(su3.compress12_cols(U)) - U).max() < 1e-13     # eq. 2.3 as printed
    assert np.abs(su3.reconstruct12_rows(su3.compress12_rows(U)) - U).max() < 1e-13     # same identity on rows


def test_eq_2_3_by_hand():
    """c = (a x b)^* written out component by component for one matrix."""
    U = haar_su3(1, np.random.Generator(np.random.PCG64(1)))[0]
    a, b, c = U[:, 0], U[:, 1], U[:, 2]
    hand = np.conj(np.array([a[1] * b[2] - a[2] * b[1], a[2] * b[0] - a[0] * b[2], a[0] * b[1] - a[1] * b[0]]))
    assert np.allclose(hand, c, atol=1e-14)


@pytest.mark.parametrize("name", ["haar", "smooth0.3", "smooth0.25"])
def test_recon8(name):
    U = _fields()[name]
    z, th = su3.compress8(U)
    assert z.shape[-1] == 3 and th.shape[-1] == 2          # 3 complex + 2 phases = 8 reals
    R = su3.reconstruct8(z, th)
    N = np.abs(U[:, 0, 1]) ** 2 + np.abs(U[:, 0, 2]) ** 2
    err = np.abs(R - U).reshape(len(U), -1).max(axis=1)
    assert np.all(err * N < 1e-13)                          # error amplified at most ~1/N
    assert err.max() < 1e-10
    assert np.abs(np.einsum("nij,nkj->nik", R, R.conj()) - np.eye(3)).max() < 1e-9
    assert np.abs(np.linalg.det(R) - 1).max() < 1e-9


def test_recon8_singular_on_unit_links():
    assert su3.recon8_min_N(unit_su3(4)) == 0.0
    with np.errstate(all="ignore"):
        z, th = su3.compress8(unit_su3(1))
        assert not np.all(np.isfinite(su3.reconstruct8(z, th)))
