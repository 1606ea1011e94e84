"""qcd_inv_sqrt_coeffs is host-only code behind the C ABI, so its parity against the oracle
(oracle/rational.py, mpmath at 50 digits) runs without a GPU.  Tolerances: the library works in plain
double precision from a closed form; measured agreement is ~2e-13 relative for n <= 30, the bar is
1e-11 (an error of that size changes r(x) by 1e-11 relative, below every delta used here)."""
import ctypes

import numpy as np
import pytest

import paper_1710_09178_b200 as q
from paper_1710_09178_b200 import binding, build
from oracle import rational as R

CASES = [(1, 0.5, 40.5), (2, 1.0, 9.0), (5, 0.01, 9.0), (10, 2.5e-5, 8.5), (12, 1.25e-5, 8.5),
         (16, 2.5e-5, 8.5), (24, 5e-5, 34.0)]


@pytest.fixture(scope="module", autouse=True)
def _built():
    build.build()


@pytest.mark.parametrize("n,xmin,xmax", CASES)
def test_coefficients_match_the_oracle(n, xmin, xmax):
    c0, c, d, delta = q.inv_sqrt_coeffs(n, xmin, xmax)
    z = R.zolotarev_inv_sqrt(n, xmin, xmax)
    assert abs(c0 / z["c0"] - 1) <= 1e-11
    assert np.abs(c / z["c"] - 1).max() <= 1e-11
    assert np.abs(d / z["d"] - 1).max() <= 1e-11
    assert abs(delta - z["delta"]) <= 1e-6 * z["delta"] + 2e-15
    assert (np.diff(d) > 0).all() and (d > 0).all() and (c > 0).all()


@pytest.mark.parametrize("n,xmin,xmax", [(8, 1e-4, 8.5), (16, 2.5e-5, 8.5)])
def test_library_coefficients_meet_their_own_delta(n, xmin, xmax):
    """Independent of the oracle's coefficients: evaluate the LIBRARY's r(x) in 50 digits on a fine
    grid; the relative error must stay within the delta the library reports."""
    c0, c, d, delta = q.inv_sqrt_coeffs(n, xmin, xmax)
    x = xmin * (xmax / xmin) ** (np.arange(3001) / 3000.0)
    err = R.relative_error_curve(c0, c, d, x)
    assert np.abs(err).max() <= delta * (1 + 1e-6) + 1e-13
    assert np.abs(err).max() >= 0.999 * delta


def test_bad_arguments():
    lib = q.load_library()
    buf = (ctypes.c_double * 8)()
    p = ctypes.cast(buf, ctypes.c_void_p)
    for n, lo, hi in ((0, 1.0, 2.0), (65, 1.0, 2.0), (4, 0.0, 2.0), (4, 2.0, 2.0), (4, 3.0, 2.0), (4, -1.0, 2.0),
                      (4, 1.0, float("inf")), (4, float("nan"), 2.0)):
        assert lib.qcd_inv_sqrt_coeffs(n, lo, hi, p, p, p, None) == binding.QCD_EINVAL
    assert lib.qcd_inv_sqrt_coeffs(2, 1.0, 2.0, None, p, p, None) == binding.QCD_EINVAL
    with pytest.raises(q.QcdError, match="QCD_EINVAL"):
        q.inv_sqrt_coeffs(3, 5.0, 1.0)
    assert lib.qcd_inv_sqrt(None, 0, None, 4, 1.0, 2.0, 1e-10, 10, None, None, None, None) == binding.QCD_EINVAL
