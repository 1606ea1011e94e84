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


def test_wide_interval_with_the_maximum_number_of_poles_stays_finite():
    """The product of the n numerator factors of a residue grows like (xmax/xmin)^(n/2): 1e448 for
    n = 64 on [1e-12, 100].  The library pairs numerator and denominator factors, so every coefficient
    stays finite and agrees with the 50-digit oracle."""
    n, xmin, xmax = 64, 1e-12, 100.0
    c0, c, d, delta = q.inv_sqrt_coeffs(n, xmin, xmax)
    z = R.zolotarev_inv_sqrt(n, xmin, xmax)
    assert np.isfinite(c).all() and np.isfinite(d).all() and np.isfinite(c0)
    assert abs(c0 / z["c0"] - 1) <= 1e-8
    assert np.abs(c / z["c"] - 1).max() <= 1e-8 and np.abs(d / z["d"] - 1).max() <= 1e-8


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


# ------------------------------------------------------------------ qcd_pow_coeffs (any exponent; x^(1/4))

from fractions import Fraction  # noqa: E402

POW_CASES = [(1, 4, 6, 1e-3, 7.0), (1, 4, 10, 2.5e-5, 8.5), (-1, 4, 9, 1e-4, 8.5), (1, 2, 8, 1e-4, 8.5),
             (3, 4, 5, 1e-2, 9.0), (-1, 3, 7, 1e-3, 8.5)]


@pytest.mark.parametrize("num,den,n,xmin,xmax", POW_CASES)
def test_pow_coefficients_match_the_oracle(num, den, n, xmin, xmax):
    """Library: Remez in binary128 (csrc/remez.cu).  Oracle: Remez in 50 digits with mpmath.  Both
    stop when the extrema are level to ~1e-11 relative, which moves a coefficient by far less than
    the 1e-9 asked here."""
    c0, c, d, delta = q.pow_coeffs(num, den, n, xmin, xmax)
    z = R.minimax_pow(Fraction(num, den), n, xmin, xmax)
    assert abs(c0 / z["c0"] - 1) <= 1e-9
    assert np.abs(c / z["c"] - 1).max() <= 1e-9 and np.abs(d / z["d"] - 1).max() <= 1e-9
    assert abs(delta / z["delta"] - 1) <= 1e-6
    assert (np.diff(d) > 0).all() and (d > 0).all() and (np.sign(c) == -np.sign(num)).all()


def test_pow_library_meets_its_own_delta_and_the_papers_figure():
    """x^(1/4) on [5e-5, 34] with 24 terms 'has an error of < 1e-12 throughout the
    approximation range'.  The library's fit, evaluated in 50 digits, must say the same."""
    c0, c, d, delta = q.pow_coeffs(1, 4, 24, 5e-5, 34.0)
    assert 1e-14 < delta < 1e-12
    x = 5e-5 * (34.0 / 5e-5) ** (np.arange(1501) / 1500.0)
    err = R.relative_error_curve_pow(0.25, c0, c, d, x)
    assert np.abs(err).max() <= delta * (1 + 1e-6) + 3e-15       # + rounding of 49 coefficients to double
    assert np.abs(err).max() >= 0.99 * delta
    # 'about 30 coefficients to achieve an error below 1e-11' at xmin < (2 m a)^2 = 1.6e-5
    assert q.pow_coeffs(1, 4, 30, 1.6e-5, 34.0)[3] < 1e-11


def _extrema(err):
    """indices of the local extrema of |err| (end points included)"""
    a = np.abs(err)
    idx = [i for i in range(len(a))
           if (i == 0 or a[i] >= a[i - 1]) and (i == len(a) - 1 or a[i] > a[i + 1])]
    return [i for i in idx if a[i] > 0.5 * a.max()]


@pytest.mark.parametrize("num,den,n,xmin,xmax", [(1, 4, 10, 2.5e-5, 8.5), (-1, 3, 7, 1e-3, 8.5),
                                                  (-1, 2, 8, 1e-4, 8.5), (1, 4, 6, 1e-3, 7.0)])
def test_library_fits_satisfy_chebyshevs_criterion(num, den, n, xmin, xmax):
    """Independent of the oracle's Remez (which uses the same algorithm as csrc/remez.cu): a type-(n,n)
    rational function whose relative error reaches +-delta with alternating sign at 2n+2 points of
    [xmin, xmax], end points included, IS the minimax approximation (it is unique).  The LIBRARY's
    coefficients are evaluated in 50 digits (evaluation only) and checked for exactly that: the count,
    the alternation, the level, the end points."""
    c0, c, d, delta = q.pow_coeffs(num, den, n, xmin, xmax)
    x = xmin * (xmax / xmin) ** (np.arange(6001) / 6000.0)
    err = R.relative_error_curve_pow(num / den, c0, c, d, x)
    ext = _extrema(err)
    assert len(ext) == 2 * n + 2 and ext[0] == 0 and ext[-1] == len(x) - 1
    signs = np.sign(err[ext])
    assert (signs[1:] * signs[:-1] < 0).all()
    assert np.abs(np.abs(err[ext]) / delta - 1).max() < 2e-4
    assert abs(np.abs(err).max() / delta - 1) < 1e-6


def test_pow_minus_one_half_is_the_closed_form():
    a = q.pow_coeffs(-1, 2, 12, 2.5e-5, 8.5)
    b = q.inv_sqrt_coeffs(12, 2.5e-5, 8.5)
    assert a[0] == b[0] and np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])
    # and -2/4 is the same exponent
    assert q.pow_coeffs(-2, 4, 12, 2.5e-5, 8.5)[0] == b[0]


def test_pow_bad_arguments_and_over_resolution():
    for num, den, n, lo, hi in ((0, 4, 4, 1.0, 2.0), (1, 0, 4, 1.0, 2.0), (4, 4, 4, 1.0, 2.0), (-5, 4, 4, 1.0, 2.0),
                                (1, 4, 0, 1.0, 2.0), (1, 4, 65, 1.0, 2.0), (1, 4, 4, 2.0, 1.0), (1, 4, 4, 0.0, 1.0)):
        with pytest.raises(q.QcdError, match="QCD_EINVAL"):
            q.pow_coeffs(num, den, n, lo, hi)
    with pytest.raises(q.QcdError, match="QCD_ENOTCONV"):       # delta would be ~1e-40: nothing to level
        q.pow_coeffs(1, 4, 40, 0.1, 8.5)


def _golden_cases():
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "rational_coefficients.txt")
    cases, cur = [], None
    for line in open(path):
        f = line.split()
        if not f or f[0].startswith("#"):
            continue
        if f[0] == "case":
            cur = dict(num=int(f[1]), den=int(f[2]), n=int(f[3]), xmin=float(f[4]), xmax=float(f[5]),
                       delta=float(f[6]), c0=float(f[7]), c=[], d=[])
            cases.append(cur)
        else:
            cur["c"].append(float(f[1]))
            cur["d"].append(float(f[2]))
    return cases


def test_library_against_the_stored_oracle_coefficients():
    """tests/golden/rational_coefficients.txt is written by the oracle alone; the library must
    reproduce every stored coefficient (and the oracle must still produce them: a regression pin)."""
    cases = _golden_cases()
    assert len(cases) == 4
    for g in cases:
        c0, c, d, delta = q.pow_coeffs(g["num"], g["den"], g["n"], g["xmin"], g["xmax"])
        assert abs(c0 / g["c0"] - 1) <= 1e-9 and abs(delta / g["delta"] - 1) <= 1e-6
        assert np.abs(c / np.array(g["c"]) - 1).max() <= 1e-9
        assert np.abs(d / np.array(g["d"]) - 1).max() <= 1e-9
    g = cases[0]
    z = R.zolotarev_inv_sqrt(g["n"], g["xmin"], g["xmax"])
    assert z["c0"] == g["c0"] and np.array_equal(z["c"], g["c"]) and np.array_equal(z["d"], g["d"])
