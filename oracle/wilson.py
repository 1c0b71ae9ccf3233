"""Oracle (test infrastructure): the massive Wilson-Dirac operator Q = gamma5 D_W, eq. 2.1-2.2.

PAPER.md:L35-42 (section 2.1):

    D_W phi(x) = (4+m) phi(x) - 1/2 sum_{mu=+-0..+-3} U_mu(x) (1 - gamma_mu) phi(x + a mu^),   Q = gamma5 D_W   (2.1)
    U_{-mu}(x) = U_mu(x - a mu^)^{-1},   gamma_{-mu} = -gamma_mu                                               (2.2)

Readings: a = 1; mu = 0 is time (extent dims[0]); time boundary condition is a
sign `bc_time` (+1 periodic, -1 antiperiodic) carried by every hop that crosses the x0 = T-1 <-> 0 seam;
space is periodic; chiral gamma basis (R2); U acts on colour, gamma on spin.

Array conventions: psi[x0,x1,x2,x3,spin,colour], U[mu,x0,x1,x2,x3,row,col], complex128.
"""
import numpy as np

_s1 = np.array([[0, 1], [1, 0]], dtype=np.complex128)
_s2 = np.array([[0, -1j], [1j, 0]], dtype=np.complex128)
_s3 = np.array([[1, 0], [0, -1]], dtype=np.complex128)
_z2 = np.zeros((2, 2), dtype=np.complex128)
_i2 = np.eye(2, dtype=np.complex128)


def gamma_matrices():
    """(gamma_0..gamma_3, gamma_5) in the chiral basis of DESIGN.md reading R2 (the paper is silent on the
    basis; BASELINE.json config 0 says 'chiral gamma basis'):
        gamma_0 = [[0,-1],[-1,0]],  gamma_k = [[0,-i sigma_k],[i sigma_k,0]],  gamma_5 = gamma_0 gamma_1 gamma_2 gamma_3.
    """
    g0 = np.block([[_z2, -_i2], [-_i2, _z2]])
    gk = [np.block([[_z2, -1j * s], [1j * s, _z2]]) for s in (_s1, _s2, _s3)]
    g = [g0] + gk
    g5 = g[0] @ g[1] @ g[2] @ g[3]
    return g, g5


def apply_DW(psi, U, m, bc_time=-1):
    """D_W psi by eq. 2.1 with the +-mu sum split by eq. 2.2 (U^{-1} = U^dagger for SU(3)):

        D_W psi(x) = (4+m) psi(x) - 1/2 sum_{mu=0}^{3} [ U_mu(x) (1-gamma_mu) psi(x+mu^)
                                                        + U_mu(x-mu^)^dagger (1+gamma_mu) psi(x-mu^) ]
    """
    g, _ = gamma_matrices()
    one = np.eye(4, dtype=np.complex128)
    out = (4.0 + m) * psi
    for mu in range(4):
        fwd = np.roll(psi, -1, axis=mu)          # fwd[x] = psi[x + mu^]
        bwd = np.roll(psi, +1, axis=mu)          # bwd[x] = psi[x - mu^]
        Ub = np.roll(U[mu], +1, axis=mu)         # Ub[x]  = U_mu(x - mu^)
        if mu == 0 and bc_time != 1:
            fwd[-1] *= bc_time                   # hop from x0 = T-1 to x0 = 0 crosses the seam
            bwd[0] *= bc_time                    # hop from x0 = 0 to x0 = T-1 crosses the seam
        out -= 0.5 * np.einsum("...ab,st,...tb->...sa", U[mu], one - g[mu], fwd)
        out -= 0.5 * np.einsum("...ba,st,...tb->...sa", Ub.conj(), one + g[mu], bwd)
    return out


def apply_gamma5(psi):
    _, g5 = gamma_matrices()
    return np.einsum("st,...tb->...sb", g5, psi)


def apply_Q(psi, U, m, bc_time=-1):
    """Q psi = gamma5 D_W psi (eq. 2.1)."""
    return apply_gamma5(apply_DW(psi, U, m, bc_time))


def apply_Q_literal(psi, U, m, bc_time=-1):
    """Eq. 2.1 read literally, site by site, as a sum over the eight signed directions +-0..+-3 with
    eq. 2.2 used verbatim: U_{-mu}(x) = inverse(U_mu(x - mu^)) (numpy.linalg.inv, not the dagger) and
    gamma_{-mu} = -gamma_mu.  Pure Python loops: tiny lattices only.  Serves as the brute-force pin of
    the vectorised `apply_Q` (tests/test_oracle_wilson.py)."""
    g, g5 = gamma_matrices()
    one = np.eye(4, dtype=np.complex128)
    dims = psi.shape[:4]
    out = np.zeros_like(psi)
    for x in np.ndindex(*dims):
        acc = (4.0 + m) * psi[x]
        for mu in range(4):
            for sgn in (+1, -1):
                y = list(x)
                y[mu] += sgn
                phase = 1.0
                if y[mu] >= dims[mu] or y[mu] < 0:
                    y[mu] %= dims[mu]
                    if mu == 0:
                        phase = bc_time
                y = tuple(y)
                if sgn > 0:
                    link = U[(mu,) + x]
                    gam = g[mu]
                else:
                    link = np.linalg.inv(U[(mu,) + y])   # U_{-mu}(x) = U_mu(x - mu^)^{-1}
                    gam = -g[mu]                          # gamma_{-mu} = -gamma_mu
                acc = acc - 0.5 * phase * ((one - gam) @ psi[y] @ link.T)
        out[x] = g5 @ acc
    return out


def dense_Q(U, m, bc_time=-1):
    """The matrix of Q on the whole lattice (N = 12 V rows), built column by column by applying the
    operator to unit vectors; index order = C order of psi[x0,x1,x2,x3,spin,colour].  4^4 -> 3072 x 3072
    (BASELINE.json north_star: 'dense 3072x3072 eigendecomposition')."""
    dims = U.shape[1:5]
    n = int(np.prod(dims)) * 12
    mat = np.empty((n, n), dtype=np.complex128)
    e = np.zeros(n, dtype=np.complex128)
    for j in range(n):
        e[j] = 1.0
        mat[:, j] = apply_Q(e.reshape(dims + (4, 3)), U, m, bc_time).reshape(n)
        e[j] = 0.0
    return mat


def norm_bound_Q(m):
    """||Q|| <= |4+m| + 4 (reading R6: each pair 1/2[(1-g)T + (1+g)T^dagger] with T the unitary
    covariant shift is unitary, so the hopping term has norm <= 4)."""
    return abs(4.0 + m) + 4.0
