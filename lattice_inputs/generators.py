"""Random SU(3) fields and Gaussian spinors (numpy, PCG64, fixed seeds)."""
import numpy as np

SEED_GAUGE = 1010      # gauge fields
SEED_SOURCE = 5636     # source spinors
SEED_TRANSFORM = 2010  # random gauge transformations (tests)


def _rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


def _complex_gaussian(rng, shape):
    """Re, Im ~ N(0,1); drawn in C order with (re, im) as the last axis."""
    a = rng.standard_normal(tuple(shape) + (2,))
    return a[..., 0] + 1j * a[..., 1]


def haar_su3(n, rng):
    """n Haar-distributed SU(3) matrices: complex Gaussian 3x3 -> QR -> fix the column phases with
    diag(R)/|diag(R)| -> remove the determinant phase (principal cube root). BASELINE.json config 0/2."""
    out = np.empty((n, 3, 3), dtype=np.complex128)
    step = 1 << 20
    for lo in range(0, n, step):
        hi = min(n, lo + step)
        a = _complex_gaussian(rng, (hi - lo, 3, 3))
        q, r = np.linalg.qr(a)
        d = np.einsum("nii->ni", r)
        q = q * (d / np.abs(d))[:, None, :]
        det = np.linalg.det(q)
        out[lo:hi] = q * (det ** (-1.0 / 3.0))[:, None, None]
    return out


def smooth_su3(n, eps, rng):
    """n 'smooth-ish' SU(3) matrices U = exp(i eps H), H = traceless Hermitian part of a complex
    Gaussian 3x3 (via eigh). BASELINE.json configs 1/3/4."""
    out = np.empty((n, 3, 3), dtype=np.complex128)
    step = 1 << 20
    eye = np.eye(3)
    for lo in range(0, n, step):
        hi = min(n, lo + step)
        a = _complex_gaussian(rng, (hi - lo, 3, 3))
        h = 0.5 * (a + a.conj().transpose(0, 2, 1))
        h = h - (np.einsum("nii->n", h) / 3.0)[:, None, None] * eye
        w, v = np.linalg.eigh(h)
        out[lo:hi] = np.einsum("nij,nj,nkj->nik", v, np.exp(1j * eps * w), v.conj())
    return out


def unit_su3(n):
    out = np.zeros((n, 3, 3), dtype=np.complex128)
    out[:, 0, 0] = out[:, 1, 1] = out[:, 2, 2] = 1.0
    return out


def gauge_field(dims, kind, seed=SEED_GAUGE, eps=0.3):
    """U[mu, x0, x1, x2, x3, row, col]; kind in {'haar', 'smooth', 'unit'}."""
    dims = tuple(int(d) for d in dims)
    n = 4 * int(np.prod(dims))
    if kind == "haar":
        u = haar_su3(n, _rng(seed))
    elif kind == "smooth":
        u = smooth_su3(n, eps, _rng(seed))
    elif kind == "unit":
        u = unit_su3(n)
    else:
        raise ValueError(f"unknown gauge field kind {kind!r}")
    return u.reshape((4,) + dims + (3, 3))


def flux_su3(dims, q01, q23, noise=0.0, seed=SEED_GAUGE):
    """A topologically non-trivial SU(3) field for the index tests: constant abelian field strength on the 4-torus in the
    Cartan direction T = diag(1, -1, 0), with q01 flux quanta through the (x0, x1) planes and q23 through the (x2, x3)
    planes (F = 2 pi q / (L_a L_b) per plaquette; the transition functions sit on the last links of x0 and x2), times an
    optional random rotation exp(i noise H) of every link that removes the degeneracies of the purely diagonal field.
    Input recipe only: diagonal phases and a matrix exponential, no operator of the method."""
    dims = tuple(int(d) for d in dims)
    L0, L1, L2, L3 = dims
    t = np.array([1.0, -1.0, 0.0])
    x = np.indices(dims)
    f01 = 2.0 * np.pi * q01 / (L0 * L1)
    f23 = 2.0 * np.pi * q23 / (L2 * L3)
    phases = [np.where(x[0] == L0 - 1, -f01 * L0 * x[1], 0.0), f01 * x[0],
              np.where(x[2] == L2 - 1, -f23 * L2 * x[3], 0.0), f23 * x[2]]
    u = np.zeros((4,) + dims + (3, 3), dtype=np.complex128)
    for mu in range(4):
        for a in range(3):
            u[mu, ..., a, a] = np.exp(1j * phases[mu] * t[a])
    if noise:
        r = smooth_su3(4 * int(np.prod(dims)), noise, _rng(seed)).reshape(u.shape)
        u = np.einsum("...ij,...jk->...ik", r, u)
    return u


def gaussian_spinor(dims, seed=SEED_SOURCE):
    """psi[x0, x1, x2, x3, spin, colour], Re/Im ~ N(0,1)."""
    dims = tuple(int(d) for d in dims)
    return _complex_gaussian(_rng(seed), dims + (4, 3))


def parse_lattice(name):
    """'16^3x32' (spatial L, time T as the paper and BASELINE.json quote lattices) -> dims (T, L, L, L)."""
    s, t = name.lower().replace(" ", "").split("x")
    l, p = s.split("^")
    if p != "3":
        raise ValueError(name)
    return (int(t), int(l), int(l), int(l))


def lattice_name(dims):
    t, l1, l2, l3 = dims
    return f"{l1}^3x{t}" if l1 == l2 == l3 else "x".join(str(d) for d in dims)
