"""Host-side checks of the C-ABI boundary that need no GPU: the library loads, exports every symbol that
include/nd_b200.h declares, the binding covers exactly those symbols, the two host utilities (nd_cheb_coeffs, nd_heev)
agree with independent computations, and the product fails loudly (never falls back) without a CUDA device."""
import ctypes
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "nd_b200.h")


def declared_symbols():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"ND_API\s+[\w\s\*]+?\b(nd_\w+)\s*\(", text)))


def test_header_declares_the_boundary_calls():
    names = declared_symbols()
    for must in ("nd_create", "nd_set_gauge", "nd_apply_Q", "nd_apply_Q2", "nd_apply_DN", "nd_apply_sign", "nd_axpy",
                 "nd_dot", "nd_norm2", "nd_block_dot", "nd_block_axpy", "nd_lowmodes_compute", "nd_pack_spinor"):
        assert must in names


def test_library_exports_every_declared_symbol():
    import paper_1010_5636_b200 as nd

    lib = nd.load_library()
    raw = ctypes.CDLL(nd.LIB_PATH)
    for name in declared_symbols():
        assert hasattr(raw, name), f"{name} declared in nd_b200.h but not exported"
    assert sorted(nd.SIGNATURES) == declared_symbols()
    assert lib is nd.load_library()


def test_only_declared_symbols_are_exported():
    import paper_1010_5636_b200 as nd

    out = subprocess.run(["nm", "-D", "--defined-only", nd.LIB_PATH], capture_output=True, text=True, check=True).stdout
    exported = sorted(l.split()[-1] for l in out.splitlines() if " T " in l and l.split()[-1].startswith("nd_"))
    assert exported == declared_symbols()


def test_cheb_coeffs_matches_independent_fit():
    """nd_cheb_coeffs (library, long double DCT) vs numpy's Chebyshev interpolation of y^{-1/2} on [eps, 1] and the
    delta table of SURVEY.md 8(c)-A7."""
    import paper_1010_5636_b200 as nd
    from numpy.polynomial import chebyshev as C

    for n, eps, dref in ((100, 0.01, 5.4e-10), (100, 0.002, 5.9e-5), (200, 0.002, 5.6e-9)):
        c, delta = nd.cheb_coeffs(n, eps)
        ref = C.chebinterpolate(lambda z: 1.0 / np.sqrt(((1 - eps) * z + 1 + eps) / 2), n)
        assert np.abs(c - ref).max() < 1e-12 * np.abs(ref).max()
        assert abs(delta / dref - 1) < 0.05
    assert nd.load_library().nd_cheb_coeffs(5, 1.5, None, None) == -1


def test_heev_matches_lapack():
    import paper_1010_5636_b200 as nd

    rng = np.random.default_rng(3)
    for k in (1, 2, 7, 28, 64):
        a = rng.standard_normal((k, k)) + 1j * rng.standard_normal((k, k))
        a = a + a.conj().T
        w, z = nd.heev(a)
        assert np.abs(w - np.linalg.eigvalsh(a)).max() < 1e-12 * max(1.0, np.abs(a).max() * k)
        assert np.abs(z.conj().T @ z - np.eye(k)).max() < 1e-12
        assert np.abs(a @ z - z * w).max() < 1e-11 * max(1.0, np.abs(a).max() * k)
    # degenerate spectrum and an already diagonal matrix
    w, z = nd.heev(np.diag([2.0, 1.0, 1.0, 2.0, -3.0]).astype(np.complex128))
    assert np.allclose(w, [-3, 1, 1, 2, 2]) and np.abs(z.conj().T @ z - np.eye(5)).max() < 1e-15


def test_no_cpu_fallback_without_a_device():
    """Without a CUDA device nd_create must fail with ND_ERR_CUDA and Context() must raise."""
    import torch

    import paper_1010_5636_b200 as nd

    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    lib = nd.load_library()
    h = ctypes.c_void_p()
    dims = (ctypes.c_int * 4)(4, 4, 4, 4)
    assert lib.nd_create(ctypes.byref(h), dims, 64, 12, -1, 0, None) == -5 and not h.value
    with pytest.raises(nd.NDError):
        nd.Context((4, 4, 4, 4))
    # null / bad arguments are reported, not crashed on
    assert lib.nd_create(None, dims, 64, 12, -1, 0, None) == -1
    assert lib.nd_create(ctypes.byref(h), dims, 16, 12, -1, 0, None) == -1
    assert lib.nd_apply_Q(None, None, None, 0.0) == -1
    assert lib.nd_last_error(None) == b"null context"


def test_product_never_imports_the_oracle():
    """The CUDA path and the oracle share no code: nothing under paper_1010_5636_b200/ mentions oracle/, and
    importing the package does not pull the oracle in."""
    pkg = os.path.join(ROOT, "paper_1010_5636_b200")
    for dirpath, _, files in os.walk(pkg):
        if os.path.basename(dirpath) in ("build", "__pycache__"):
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert "wilson_ref" not in text, f
    code = "import sys; import paper_1010_5636_b200; assert not any(m == 'oracle' or m.startswith('oracle.') for m in sys.modules)"
    subprocess.run([sys.executable, "-c", code], cwd=ROOT, check=True)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_1010_5636_b200" not in text.replace("`paper_1010_5636_b200/`", ""), f


def test_projector_error_matches_oracle():
    """nd_projector_error (library, eq. 2.9-2.10) vs the oracle's independent functions on random inputs, and the
    hand-evaluated value of eq. 2.10 at kappa = 0.1."""
    import paper_1010_5636_b200 as nd
    from oracle import lowmodes as olow

    rng = np.random.default_rng(9)
    for l, nrest in ((1, 0), (6, 5), (20, 12)):
        nu = rng.uniform(0.3, 0.6, l) * rng.choice([-1.0, 1.0], l)
        rho = rng.uniform(1e-4, 2e-2, l)
        rest = rng.uniform(0.7, 1.5, nrest) * rng.choice([-1.0, 1.0], nrest)
        if l == 1:
            rest = np.array([0.9])
        kappa, bound, d = nd.projector_error(nu, rho, rest)
        dref = olow.distances_d(nu, rest)
        kp, km = olow.kappa_pm(nu, rho, dref)
        assert np.allclose(d, dref, rtol=1e-14) and abs(kappa[0] - kp) <= 1e-14 and abs(kappa[1] - km) <= 1e-14
        for i, k in enumerate((kp, km)):
            ref = olow.projector_bound(k)
            assert (np.isinf(ref) and np.isinf(bound[i])) or abs(bound[i] - ref) <= 1e-13 * max(1.0, ref)
    kappa, bound, _ = nd.projector_error([1.0], [0.1], [2.0])
    assert abs(kappa[0] - 0.1) < 1e-16 and abs(bound[0] - 0.12 / 0.76) < 1e-15 and kappa[1] == 0 and bound[1] == 0
    assert np.isinf(nd.projector_error([1.0], [0.5], [2.0])[1][0])


def test_choose_l_matches_oracle():
    """nd_choose_l (library, R17) vs the oracle's independent gap rule on hand-made and random spectra."""
    import paper_1010_5636_b200 as nd
    from oracle import lowmodes as olow

    a = np.array([0.10, 0.11, 0.30, 0.301, 0.302, 0.50, 0.90])
    for lo, hi in ((3, 5), (2, 4), (3, 4), (4, 4), (1, 6)):
        l, gap = nd.choose_l(a, lo, hi)
        lo_, gap_ = olow.choose_l(a, lo, hi)
        assert l == lo_ and abs(gap - gap_) < 1e-15
    rng = np.random.default_rng(3)
    for _ in range(50):
        k = int(rng.integers(3, 80))
        a = np.sort(rng.random(k))
        lo = int(rng.integers(1, k - 1))
        hi = int(rng.integers(lo, k - 1))
        assert nd.choose_l(a, lo, hi)[0] == olow.choose_l(a, lo, hi)[0]
    for bad in ((a[::-1], 1, 2), (a, 0, 2), (a, 3, 2), (a, 1, len(a))):
        with pytest.raises(nd.NDError):
            nd.choose_l(*bad)


@pytest.mark.parametrize("n,eps", [(0, 0.04), (12, 0.1), (40, 0.01), (100, 0.005)])
def test_minmax_coeffs_match_oracle(n, eps):
    """nd_minmax_coeffs (library, Remez in C++) vs oracle.sign.minmax_coeffs (numpy): the min-max polynomial is unique, so two
    independent implementations must give the same polynomial and the same delta; closed form at n = 0."""
    import paper_1010_5636_b200 as nd
    from oracle import sign as osign

    c, delta, lev = nd.minmax_coeffs(n, eps)
    co, do, Eo = osign.minmax_coeffs(n, eps)
    assert lev <= delta <= 1.002 * lev and abs(delta - do) <= 3e-3 * do
    y = np.geomspace(eps, 1.0, 5001)
    assert np.abs(np.sqrt(y) * (osign.eval_P_scalar(c, eps, y) - osign.eval_P_scalar(co, eps, y))).max() <= 5e-3 * delta
    assert osign.measure_delta(c, eps) <= delta * (1 + 1e-6)          # the library's delta is what its coefficients deliver
    if n == 0:
        r = np.sqrt(eps)
        assert abs(c[0] - 2 / (1 + r)) < 1e-14 and abs(delta - (1 - r) / (1 + r)) < 1e-14
    else:
        ci, di = nd.cheb_coeffs(n, eps)
        assert delta < 0.75 * di


def test_header_is_plain_c_and_links_from_c(tmp_path):
    """The boundary is a C ABI: include/nd_b200.h compiles as strict C99 (no C++-isms, no torch types), a plain-C program links
    against libnd_b200.so, and without a CUDA device nd_create fails with ND_ERR_CUDA and a NULL context instead of crashing
    (there is no CPU fallback).  On a GPU box the same program creates and destroys a context."""
    import shutil
    import subprocess

    import paper_1010_5636_b200 as nd

    if shutil.which("gcc") is None:
        pytest.skip("no gcc")
    nd.load_library()
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    src = tmp_path / "abi_smoke.c"
    src.write_text(
        '#include <stdio.h>\n#include "nd_b200.h"\n'
        "int main(void) {\n"
        "    nd_ctx* ctx = (nd_ctx*)0;\n"
        "    const int dims[4] = {4, 4, 4, 4};\n"
        "    double c[9], delta = 0.0;\n"
        "    int rc = nd_cheb_coeffs(8, 0.1, c, &delta);          /* host utility: works without a GPU */\n"
        "    if (rc != ND_OK || !(delta > 0.0 && delta < 1.0)) return 3;\n"
        "    rc = nd_create(&ctx, dims, 64, 12, -1, 0, (void*)0);\n"
        '    printf("%d %d %lld\\n", rc, ctx != (nd_ctx*)0, rc == ND_OK ? nd_volume(ctx) : -1LL);\n'
        "    if (rc == ND_OK) return nd_destroy(ctx) == ND_OK ? 0 : 4;\n"
        "    return (rc == ND_ERR_CUDA && ctx == (nd_ctx*)0) ? 0 : 5;\n"
        "}\n")
    exe = tmp_path / "abi_smoke"
    libdir = os.path.dirname(nd.LIB_PATH)
    subprocess.run(["gcc", "-std=c99", "-pedantic", "-Wall", "-Wextra", "-Werror", "-I", os.path.join(root, "include"), str(src), "-o", str(exe),
                    "-L", libdir, "-lnd_b200", "-Wl,-rpath," + libdir], check=True, capture_output=True, text=True)
    r = subprocess.run([str(exe)], capture_output=True, text=True, timeout=120)
    assert r.returncode == 0, (r.returncode, r.stdout, r.stderr)
    rc, have_ctx, vol = (int(x) for x in r.stdout.split())
    assert (rc, have_ctx, vol) in ((0, 1, 256), (-5, 0, -1))
