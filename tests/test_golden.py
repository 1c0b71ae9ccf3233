"""tests/golden/delta_table.txt (written by tests/golden/make_delta_table.py from the oracle alone): delta of eq. 2.6
 for interpolation and min-max coefficients.  Checked here: the oracle still reproduces it, the library's host
utilities nd_cheb_coeffs / nd_minmax_coeffs (no GPU) agree with it, and the rows SURVEY.md 8(c)-A7 quotes from its own
independent check agree to the two digits quoted there."""
import os

import numpy as np
import pytest

from oracle import sign as osign

HERE = os.path.dirname(os.path.abspath(__file__))
SURVEY_A7 = {(100, 0.01): 5.4e-10, (100, 0.005): 2.5e-7, (100, 0.002): 5.9e-5, (200, 0.002): 5.6e-9, (200, 0.001): 1.3e-6}


def rows():
    out = []
    with open(os.path.join(HERE, "golden", "delta_table.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            n, eps, kind, delta = line.split()
            out.append((int(n), float(eps), kind, float(delta)))
    return out


def test_table_has_the_survey_rows():
    got = {(n, eps): d for n, eps, kind, d in rows() if kind == "interpolation"}
    for key, want in SURVEY_A7.items():
        assert abs(got[key] - want) <= 0.05 * want, (key, got[key], want)


@pytest.mark.parametrize("n,eps,kind,delta", rows())
def test_oracle_and_library_reproduce_the_table(n, eps, kind, delta):
    import paper_1010_5636_b200 as nd

    if kind == "interpolation":
        c = osign.cheb_coeffs(n, eps)
        assert abs(osign.measure_delta(c, eps) - delta) <= 1e-5 * delta
        c_lib, d_lib = nd.cheb_coeffs(n, eps)
        assert np.abs(np.asarray(c_lib) - c).max() <= 1e-12 * np.abs(c).max()
        assert abs(d_lib - delta) <= 2e-3 * delta + 3e-13          # two independent grids for the maximum
    else:
        c, d_or, levelled = osign.minmax_coeffs(n, eps)
        assert abs(d_or - delta) <= 1e-5 * delta and levelled <= d_or <= 1.002 * levelled
        c_lib, d_lib, lev_lib = nd.minmax_coeffs(n, eps)
        assert abs(d_lib - delta) <= 5e-3 * delta
        interp = [d for nn, ee, k, d in rows() if (nn, ee, k) == (n, eps, "interpolation")][0]
        assert delta < 0.7 * interp                                 # the min-max polynomial is the better one at equal degree
