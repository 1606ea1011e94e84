"""CPU oracle, part 2 (TEST INFRASTRUCTURE, not the product): the rational approximation of
(M^dag M)^(-1/2) in the partial-fraction form of eq. 8,

    x^(-1/2)  ~=  r(x) = c_0 + sum_{k=1..n} c_k / (x + d_k),      xmin <= x <= xmax

"There are known algorithms to compute c_k and d_k and we use the MiniMax approximation function
of Mathematica": the paper asks for the MINIMAX rational function of type (n, n) in
the relative error, |1 - sqrt(x) r(x)| <= delta on [xmin, xmax].  For the inverse square root that
minimax problem has a closed-form solution (Zolotarev, 1877), which is what this module writes
out, slowly, in 50-digit arithmetic with mpmath (a library routine for K and sn):

    with b = xmax/xmin, kappa'^2 = 1 - 1/b, K' = K(kappa'), N = 2n+1 (type (n,n)) or 2n (type (n-1,n)):
        a_l = sn^2(l K'/N; kappa') / (1 - sn^2(l K'/N; kappa')),        l = 1 .. N-1
        r(x) = D/sqrt(xmin) * prod_l (x/xmin + a_{2l}) / prod_l (x/xmin + a_{2l-1})
    and D is fixed by max(1 - sqrt(x) r) = -min(1 - sqrt(x) r), found here by brute force on a grid.

Nothing here is taken on trust: tests/test_oracle_rational.py pins the result with Chebyshev's
equioscillation theorem (a type-(n,n) rational function whose weighted error attains +-delta with
alternating sign at 2n+2 points IS the minimax solution, whatever formula produced it), with the
paper's own remark that keeping c_0 halves the error at the same number of shifts,
with r(x)^2 x = 1 +- 2 delta, and with eq. 8 evaluated on a dense (M^dag M)_ee through `eigh`.
The product's own coefficient routine (csrc/zolotarev.cu, double precision, its own AGM for sn)
shares no code with this file.

The exponent 1/4 of the heat-bath step (appendix :288-304) has no closed form and no
coefficients are printed in the paper; it is out of scope.
"""
from __future__ import annotations

import mpmath as mp
import numpy as np

DPS = 50


def _a_coefficients(n: int, b, with_c0: bool):
    m = 1 - mp.mpf(1) / b                      # kappa'^2
    kp = mp.ellipk(m)                          # K'
    big_n = 2 * n + 1 if with_c0 else 2 * n
    a = [None]                                 # a[l], l = 1 .. N-1
    for l in range(1, big_n):
        s2 = mp.ellipfun("sn", l * kp / big_n, m=m) ** 2
        a.append(s2 / (1 - s2))
    den = [a[2 * l - 1] for l in range(1, n + 1)]
    num = [a[2 * l] for l in range(1, (n if with_c0 else n - 1) + 1)]
    return num, den


def _product_form(num, den, x):
    v = mp.mpf(1)
    for t in num:
        v *= x + t
    for t in den:
        v /= x + t
    return v


def zolotarev_inv_sqrt(n: int, xmin: float, xmax: float, with_c0: bool = True, grid: int = 4000):
    """Minimax (relative error) rational approximation of x^(-1/2) on [xmin, xmax] with n poles,
    as eq. 8: returns dict(c0, c[n], d[n], delta) of Python floats / numpy arrays, d ascending.
    with_c0=False gives the type (n-1, n) function (c0 = 0) of PAPER.md:304."""
    with mp.workdps(DPS):
        xmin_, xmax_ = mp.mpf(xmin), mp.mpf(xmax)
        if not (n >= 1 and 0 < xmin_ < xmax_):
            raise ValueError("need n >= 1 and 0 < xmin < xmax")
        b = xmax_ / xmin_
        num, den = _a_coefficients(n, b, with_c0)
        # D by brute force: f(x) = sqrt(x) prod/prod oscillates between fmin and fmax on [1, b];
        # the error 1 - D f is balanced when D = 2 / (fmax + fmin).  The extrema are located on a
        # geometric grid and refined by golden-section search between the neighbouring grid points.
        def f(x):
            return mp.sqrt(x) * _product_form(num, den, x)

        pts = [mp.power(b, mp.mpf(i) / grid) for i in range(grid + 1)]
        val = [f(x) for x in pts]
        fmax, fmin = max(val), min(val)
        for target, sign in ((fmax, 1), (fmin, -1)):
            i = val.index(target)
            lo, hi = pts[max(i - 1, 0)], pts[min(i + 1, grid)]
            best = _golden(lambda x: sign * f(x), lo, hi)
            if sign > 0:
                fmax = max(fmax, best)
            else:
                fmin = min(fmin, -best)
        big_d = 2 / (fmax + fmin)
        delta = (fmax - fmin) / (fmax + fmin)
        # partial fractions of D prod(y + num)/prod(y + den) in y = x/xmin, then back to x
        c0 = big_d if with_c0 else mp.mpf(0)
        res = []
        for k in range(n):
            v = big_d
            for t in num:
                v *= t - den[k]
            for j in range(n):
                if j != k:
                    v /= den[j] - den[k]
            res.append(v)
        s = mp.sqrt(xmin_)
        out = dict(c0=float(c0 / s), c=np.array([float(v * s) for v in res]),
                   d=np.array([float(t * xmin_) for t in den]), delta=float(delta))
    order = np.argsort(out["d"])
    out["c"], out["d"] = out["c"][order], out["d"][order]
    return out


def _golden(g, lo, hi, iters: int = 80):
    """max of a unimodal g on [lo, hi] (golden-section search in the current mp precision)."""
    phi = (mp.sqrt(5) - 1) / 2
    a, b = lo, hi
    c, d = b - phi * (b - a), a + phi * (b - a)
    gc, gd = g(c), g(d)
    for _ in range(iters):
        if gc > gd:
            b, d, gd = d, c, gc
            c = b - phi * (b - a)
            gc = g(c)
        else:
            a, c, gc = c, d, gd
            d = a + phi * (b - a)
            gd = g(d)
    return max(gc, gd)


def eval_eq8(c0: float, c, d, x):
    """r(x) = c0 + sum_k c_k / (x + d_k)  (eq. 8) for numpy x, in long double."""
    x = np.asarray(x, dtype=np.longdouble)
    r = np.full(x.shape, np.longdouble(c0))
    for ck, dk in zip(c, d):
        r = r + np.longdouble(ck) / (x + np.longdouble(dk))
    return r


def relative_error_curve(c0: float, c, d, x):
    """1 - sqrt(x) r(x) at the points x, evaluated with mpmath (50 digits) from the float
    coefficients: what a user of the coefficients actually gets."""
    out = []
    with mp.workdps(DPS):
        for xv in x:
            xv = mp.mpf(float(xv))
            r = mp.mpf(float(c0))
            for ck, dk in zip(c, d):
                r += mp.mpf(float(ck)) / (xv + mp.mpf(float(dk)))
            out.append(float(1 - mp.sqrt(xv) * r))
    return np.array(out)
