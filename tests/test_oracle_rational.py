"""Pins for oracle/rational.py: the minimax (Zolotarev) approximation of x^(-1/2) in the
partial-fraction form of eq. 8 (appendix :288-304).  None of the pins re-uses the
oracle's formula: they are Chebyshev's equioscillation criterion, a closed form derived by hand for
one pole, statements the paper makes about its own approximation, and `eigh` on a dense operator."""
import numpy as np
import pytest

import lattice_inputs as li
import oracle
from oracle import rational as R
from helpers import c as cplx, dense_from_operator


def _extrema(err):
    """indices of the local extrema of |err| (end points included)"""
    a = np.abs(err)
    idx = [i for i in range(len(a))
           if (i == 0 or a[i] >= a[i - 1]) and (i == len(a) - 1 or a[i] > a[i + 1])]
    return [i for i in idx if a[i] > 0.5 * a.max()]


@pytest.mark.parametrize("n,xmin,xmax", [(3, 1.0, 50.0), (6, 1e-3, 7.0), (10, 2.5e-5, 8.5)])
def test_equioscillation_2n_plus_2_points(n, xmin, xmax):
    """Chebyshev: a type-(n,n) rational function whose relative error reaches +-delta with
    alternating sign at 2n+2 points of [xmin, xmax] is THE minimax approximation."""
    z = R.zolotarev_inv_sqrt(n, xmin, xmax)
    x = xmin * (xmax / xmin) ** (np.arange(6001) / 6000.0)
    err = R.relative_error_curve(z["c0"], z["c"], z["d"], x)
    ext = _extrema(err)
    assert len(ext) == 2 * n + 2
    signs = np.sign(err[ext])
    assert (signs[1:] * signs[:-1] < 0).all()
    # equal magnitude (grid resolution limits the interior ones to ~1e-5 relative)
    assert np.abs(np.abs(err[ext]) / z["delta"] - 1).max() < 2e-4
    assert abs(np.abs(err).max() / z["delta"] - 1) < 1e-6
    # both end points are extrema
    assert ext[0] == 0 and ext[-1] == len(x) - 1
    # shifts of a multishift CG must be non-negative, residues of x^(-1/2) are positive
    assert (z["d"] > 0).all() and (z["c"] > 0).all() and z["c0"] > 0
    assert (np.diff(z["d"]) > 0).all()


def test_type_n_minus_1_n_has_2n_plus_1_points():
    n, xmin, xmax = 5, 0.01, 9.0
    z = R.zolotarev_inv_sqrt(n, xmin, xmax, with_c0=False)
    assert z["c0"] == 0.0
    x = xmin * (xmax / xmin) ** (np.arange(6001) / 6000.0)
    err = R.relative_error_curve(z["c0"], z["c"], z["d"], x)
    ext = _extrema(err)
    assert len(ext) == 2 * n + 1
    assert (np.sign(err[ext])[1:] * np.sign(err[ext])[:-1] < 0).all()


def test_one_pole_closed_form():
    """n = 1 without c_0: r = c/(x + d).  sqrt(x) c/(x+d) peaks at x = d and must take equal values
    at both ends, 1/(1+d) = sqrt(b)/(b+d) => d = sqrt(b) (on [1, b]); balancing the peak
    c/(2 b^(1/4)) against the end value c/(1+sqrt(b)) around 1 gives c and delta."""
    xmin, xmax = 0.5, 40.5
    b = xmax / xmin
    z = R.zolotarev_inv_sqrt(1, xmin, xmax, with_c0=False)
    hi, lo = 1 / (2 * b ** 0.25), 1 / (1 + np.sqrt(b))
    c_unit = 2 / (hi + lo)                       # on [1, b]
    assert z["d"][0] == pytest.approx(np.sqrt(b) * xmin, rel=1e-14)
    assert z["c"][0] == pytest.approx(c_unit * np.sqrt(xmin), rel=1e-13)
    assert z["delta"] == pytest.approx((hi - lo) / (hi + lo), rel=1e-12)


def test_paper_keeping_c0_halves_the_error():
    """'keeping coeff0 halved the error of the approximation without increasing the
    number of shifts required in the conjugate gradient'."""
    for n, xmin, xmax in ((8, 1e-4, 8.5), (12, 1.25e-5, 8.5), (20, 5e-5, 34.0)):
        with_c0 = R.zolotarev_inv_sqrt(n, xmin, xmax, with_c0=True)["delta"]
        without = R.zolotarev_inv_sqrt(n, xmin, xmax, with_c0=False)["delta"]
        assert 0.4 < with_c0 / without < 0.6


def test_paper_orders_of_magnitude():
    """The paper quotes, for its own (exponent 1/4 and -1/2) minimax fits: 24 terms on [5e-5, 34]
    reach < 1e-12 (appendix) and 'about 30 coefficients' reach < 1e-11 at the lightest
    mass ma = 0.002, i.e. xmin < (2ma)^2 = 1.6e-5.  The x^(-1/2) minimax error
    must be consistent with both."""
    assert R.zolotarev_inv_sqrt(24, 5e-5, 34.0)["delta"] < 1e-12
    assert R.zolotarev_inv_sqrt(30, 1.6e-5, 34.0)["delta"] < 1e-11
    # and it must NOT be reachable with far fewer terms (a wrong, too optimistic delta would pass above)
    assert R.zolotarev_inv_sqrt(12, 5e-5, 34.0)["delta"] > 1e-8


def test_r_squared_times_x_is_one():
    z = R.zolotarev_inv_sqrt(14, 1e-5, 8.5)
    x = np.logspace(-5, np.log10(8.5), 997)
    r = R.eval_eq8(z["c0"], z["c"], z["d"], x)
    assert np.abs(r * r * x - 1).max() <= 2.1 * z["delta"]


def test_eq8_on_a_dense_operator():
    """(M^dag M)^(-1/2) phi = Q diag(lambda^(-1/2)) Q^dag phi on the 4^4 lattice of config 1, against
    c_0 phi + sum_k c_k (M^dag M + d_k)^(-1) phi with the oracle's own multishift solve."""
    cfg, links, b, _, _ = li.make_config_inputs(1)
    lat = oracle.Lattice(cfg.dims, links)
    nh = lat.volume // 2
    a = dense_from_operator(lambda v: lat.mdagm(cfg.mass, 0, v), nh)
    lam, qmat = np.linalg.eigh(a)
    assert lam.min() >= cfg.mass ** 2 - 1e-12
    xmin, xmax = 0.9 * lam.min(), 1.1 * lam.max()
    z = R.zolotarev_inv_sqrt(10, xmin, xmax)
    phi = cplx(b).reshape(-1)
    exact = qmat @ ((qmat.conj().T @ phi) / np.sqrt(lam))
    sol = lat.solve_exact(cfg.mass, 0, b, z["d"], z["c"], 1e-12)
    got = z["c0"] * phi + cplx(sol["y"]).reshape(-1)
    err = np.linalg.norm(got - exact) / np.linalg.norm(exact)
    assert err <= 1.05 * z["delta"] + 1e-12
    # and the same through the eigen-decomposition (eq. 8 as a scalar identity)
    r = np.asarray(R.eval_eq8(z["c0"], z["c"], z["d"], lam), dtype=float)
    assert np.abs(r * np.sqrt(lam) - 1).max() <= 1.0001 * z["delta"]


# ------------------------------------------------------------------ any exponent (x^(1/4))

from fractions import Fraction  # noqa: E402


@pytest.mark.parametrize("alpha,n,xmin,xmax", [(Fraction(1, 4), 6, 1e-3, 7.0), (Fraction(-1, 4), 5, 1e-2, 9.0),
                                               (Fraction(1, 4), 10, 2.5e-5, 8.5)])
def test_minimax_pow_equioscillates(alpha, n, xmin, xmax):
    """Chebyshev's criterion again: 2n+2 alternating extrema of equal size of r(x)/x^alpha - 1."""
    z = R.minimax_pow(alpha, n, xmin, xmax)
    x = xmin * (xmax / xmin) ** (np.arange(6001) / 6000.0)
    err = R.relative_error_curve_pow(float(alpha), z["c0"], z["c"], z["d"], x)
    ext = _extrema(err)
    assert len(ext) == 2 * n + 2 and ext[0] == 0 and ext[-1] == len(x) - 1
    signs = np.sign(err[ext])
    assert (signs[1:] * signs[:-1] < 0).all()
    assert np.abs(np.abs(err[ext]) / z["delta"] - 1).max() < 2e-4
    assert abs(np.abs(err).max() / z["delta"] - 1) < 1e-6
    assert (z["d"] > 0).all() and (np.diff(z["d"]) > 0).all()
    # x^alpha with alpha > 0 grows: negative residues; alpha < 0: positive (Stieltjes function)
    assert (z["c"] * np.sign(float(alpha)) < 0).all() and z["c0"] > 0


def test_minimax_pow_reproduces_the_closed_form_at_minus_one_half():
    """The general routine run at alpha = -1/2 must land on Zolotarev's solution (pinned above)."""
    z = R.minimax_pow(Fraction(-1, 2), 7, 3e-4, 8.5)
    zz = R.zolotarev_inv_sqrt(7, 3e-4, 8.5)
    assert abs(z["c0"] / zz["c0"] - 1) < 1e-13 and abs(z["delta"] / zz["delta"] - 1) < 1e-9
    assert np.abs(z["c"] / zz["c"] - 1).max() < 1e-13 and np.abs(z["d"] / zz["d"] - 1).max() < 1e-13


def test_paper_degree_24_fourth_root_is_below_1e_12():
    """The one number the paper prints about its coefficients (appendix): for ma =
    0.005, xmin = 5e-5, xmax = 34 and 24 terms the x^(1/4) fit 'has an error of < 1e-12 throughout the
    approximation range'.  A minimax error above that would contradict the paper; one far below it
    would mean the oracle is not solving the paper's problem."""
    z = R.minimax_pow(Fraction(1, 4), 24, 5e-5, 34.0, steps=3)
    assert 1e-14 < z["delta"] < 1e-12


def test_minimax_pow_fourth_power_and_inverse():
    z = R.minimax_pow(Fraction(1, 4), 9, 1e-4, 8.5)
    x = np.logspace(-4, np.log10(8.5), 499)
    r = R.eval_eq8(z["c0"], z["c"], z["d"], x)
    assert np.abs(r ** 4 / x - 1).max() <= 4.1 * z["delta"]
    zi = R.minimax_pow(Fraction(-1, 4), 9, 1e-4, 8.5)        # x^(1/4) x^(-1/4) = 1
    ri = R.eval_eq8(zi["c0"], zi["c"], zi["d"], x)
    assert np.abs(r * ri - 1).max() <= 1.01 * (z["delta"] + zi["delta"])
    assert z["delta"] < 1e-5 and zi["delta"] < 1e-5


def test_fourth_root_on_a_dense_operator():
    """(M^dag M)^(1/4) phi through eigh against eq. 8 with the oracle's multishift solves."""
    cfg, links, b, _, _ = li.make_config_inputs(1)
    lat = oracle.Lattice(cfg.dims, links)
    a = dense_from_operator(lambda v: lat.mdagm(cfg.mass, 0, v), lat.volume // 2)
    lam, qmat = np.linalg.eigh(a)
    z = R.minimax_pow(Fraction(1, 4), 10, 0.9 * lam.min(), 1.1 * lam.max())
    phi = cplx(b).reshape(-1)
    exact = qmat @ ((qmat.conj().T @ phi) * lam ** 0.25)
    sol = lat.solve_exact(cfg.mass, 0, b, z["d"], z["c"], 1e-12)
    got = z["c0"] * phi + cplx(sol["y"]).reshape(-1)
    assert np.linalg.norm(got - exact) / np.linalg.norm(exact) <= 1.05 * z["delta"] + 1e-12
