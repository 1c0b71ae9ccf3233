"""Pins of the oracle's index by zero-mode counting: the trace identity index = -1/2 tr sign(Q) that follows
from tr gamma5 = 0 and the Ginsparg-Wilson relation, the index theorem's closed form on constant-flux torus fields
(|index| = sum_a e_a^2 |q01 q23| = 2 |q01 q23| for the Cartan direction diag(1,-1,0), odd under q23 -> -q23), invariance
under a random gauge transformation and a small deformation, index 0 on the topologically trivial synthetic fields, and the
pairing of the non-zero spectra of the two chirality sectors."""
import numpy as np
import pytest

from lattice_inputs import flux_su3, gauge_field, haar_su3
from oracle import index as oindex
from oracle import wilson

DIMS = (4, 4, 2, 2)      # 768 x 768 dense matrices: the flux quanta fit (F = 2 pi / 16 and 2 pi / 4 per plaquette)
M = -1.6


@pytest.fixture(scope="module")
def flux_field():
    U = flux_su3(DIMS, 1, 1)
    return U, wilson.dense_Q(U, M)


def test_trivial_fields_have_index_zero():
    Q = wilson.dense_Q(gauge_field(DIMS, "smooth", eps=0.3), M)
    assert oindex.zero_mode_count(Q) == (0, 0)
    S, lam = oindex.exact_sign(Q)
    assert abs(np.trace(S).real) < 1e-9 and np.sum(lam > 0) == np.sum(lam < 0)


def test_flux_field_index_closed_form_and_trace_identity(flux_field):
    U, Q = flux_field
    npl, nmi = oindex.zero_mode_count(Q, c=1.0 / 1.6)
    S, lam = oindex.exact_sign(Q)
    assert abs(npl - nmi) == 2 and min(npl, nmi) == 0                   # index theorem: 2 |q01 q23|, zero modes of ONE chirality
    assert npl - nmi == round(-0.5 * np.trace(S).real)                  # index = -1/2 tr sign(Q)
    assert npl - nmi == (np.sum(lam < 0) - np.sum(lam > 0)) // 2
    # odd under reversal of one flux, quadratic in the charges, zero without flux in one plane
    assert oindex.index(wilson.dense_Q(flux_su3(DIMS, 1, -1), M)) == -(npl - nmi)
    assert oindex.index(wilson.dense_Q(flux_su3(DIMS, 0, 1), M)) == 0


def test_index_is_gauge_invariant_and_stable_under_deformation(flux_field):
    U, Q = flux_field
    ref = oindex.index(Q)
    rng = np.random.Generator(np.random.PCG64(2010))
    G = haar_su3(int(np.prod(DIMS)), rng).reshape(DIMS + (3, 3))
    Ug = np.empty_like(U)
    for mu in range(4):
        Ug[mu] = np.einsum("...ij,...jk,...lk->...il", G, U[mu], np.roll(G, -1, axis=mu).conj())
    assert oindex.index(wilson.dense_Q(Ug, M)) == ref
    assert oindex.index(wilson.dense_Q(flux_su3(DIMS, 1, 1, noise=0.05), M)) == ref


def test_sector_spectra_pair_up_except_for_the_zero_modes(flux_field):
    U, Q = flux_field
    npl, nmi = oindex.zero_mode_count(Q)
    bp, bm = oindex.sector_spectrum(Q, +1), oindex.sector_spectrum(Q, -1)
    assert np.sum(bp < 1e-9) == npl and np.sum(bm < 1e-9) == nmi
    # D^dagger D has the same non-zero, non-maximal eigenvalues in both sectors (Ginsparg-Wilson pairing)
    mid_p = bp[(bp > 1e-6) & (bp < 2 - 1e-6)]
    mid_m = bm[(bm > 1e-6) & (bm < 2 - 1e-6)]
    assert len(mid_p) == len(mid_m) and np.abs(mid_p - mid_m).max() < 1e-9
    assert bp.min() > -1e-12 and bp.max() < 2 + 1e-12
