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

The exponent 1/4 of the heat-bath step (appendix :288-304) has no closed form; the
second half of this file finds its minimax approximation with a Remez exchange iteration.
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


# ---------------------------------------------------------------------------------------------
# Any exponent: x^alpha, -1 < alpha < 1, alpha != 0 -- in particular the paper's b = 4, alpha = 1/4
# (heat bath, appendix :288-304: "rational approximation to the function x^(1/4)").
# No closed form exists; the paper calls Mathematica's MiniMax at 80 digits.  The oracle runs the
# Remez exchange algorithm, in 50 digits, directly on the eq. 8 parameters (c_0, c_k, d_k):
#   repeat:  (1) solve the 2n+2 equations  r(x_i)/f(x_i) - 1 = (-1)^i E  for (c_0, c_k, d_k, E) by
#                Newton's method with the analytic Jacobian (d_k = exp(u_k) keeps the poles negative);
#            (2) move every reference point x_i to the nearest local extremum of r/f - 1
#   until the 2n+2 extrema have equal magnitude (Chebyshev: that IS the minimax solution).
# Newton needs a start inside its basin.  x^(+1/2) has a closed form too -- if r(y) ~ y^(-1/2) with
# relative error oscillating in [1-delta, 1+delta], then 1/r(y) ~ y^(1/2) oscillates in
# [1/(1+delta), 1/(1-delta)] at the same 2n+2 points -- so the iteration starts from the Zolotarev
# data at alpha = +-1/2 (same sign as the target) and walks alpha to the target in a few steps.
# Pins: tests/test_oracle_rational.py (equioscillation; alpha = -1/2 against the closed form; the
# error level the paper prints for degree 24; eigh on a dense operator).

def _start_half(n, xmin, xmax, sign):
    """Exact eq. 8 data (c0, c, d, references) of the minimax approximation of x^(sign/2)."""
    b = xmax / xmin
    m = 1 - 1 / b
    kp = mp.ellipk(m)
    big_n = 2 * n + 1
    num, den = _a_coefficients(n, b, True)
    xs = [xmin / mp.ellipfun("dn", j * kp / big_n, m=m) ** 2 for j in range(big_n + 1)]
    poles, zeros = (den, num) if sign < 0 else (num, den)   # of r (sign<0) or of 1/r (sign>0)
    res = []
    for k in range(n):
        v = mp.mpf(1)
        for t in zeros:
            v *= t - poles[k]
        for j in range(n):
            if j != k:
                v /= poles[j] - poles[k]
        res.append(v)
    s = mp.sqrt(xmin) if sign > 0 else 1 / mp.sqrt(xmin)   # overall constant: Newton levels it
    return s, [s * v * xmin for v in res], [t * xmin for t in poles], xs


def _remez_eq8(alpha, c0, c, d, xs, xmin, xmax, spread_tol):
    n = len(c)
    f = lambda x: mp.power(x, alpha)                        # noqa: E731
    u = [mp.log(t) for t in d]
    big_e = mp.mpf(0)
    newton_tol = mp.mpf(10) ** (-(mp.mp.dps - 10))
    for _ in range(15):
        for _ in range(15):                                  # (1) Newton on the levelled equations
            dd = [mp.e ** uk for uk in u]
            size = 2 * n + 2
            jac, g = mp.matrix(size, size), mp.matrix(size, 1)
            for i, x in enumerate(xs):
                fx, sgn = f(x), (-1) ** i
                g[i] = (c0 + sum(ck / (x + dk) for ck, dk in zip(c, dd))) / fx - 1 - sgn * big_e
                jac[i, 0] = 1 / fx
                for k in range(n):
                    jac[i, 1 + k] = 1 / ((x + dd[k]) * fx)
                    jac[i, 1 + n + k] = -c[k] * dd[k] / ((x + dd[k]) ** 2 * fx)
                jac[i, 2 * n + 1] = -sgn
            if max(abs(g[i]) for i in range(size)) < newton_tol:
                break
            step = mp.lu_solve(jac, -g)
            lam = mp.mpf(1)
            biggest = max(abs(step[1 + n + k]) for k in range(n))
            if biggest > mp.mpf("0.5"):                      # never move a pole by more than e^0.5
                lam = mp.mpf("0.5") / biggest
            c0 += lam * step[0]
            for k in range(n):
                c[k] += lam * step[1 + k]
                u[k] += lam * step[1 + n + k]
            big_e += lam * step[2 * n + 1]
        dd = [mp.e ** uk for uk in u]
        err = lambda x: (c0 + sum(ck / (x + dk) for ck, dk in zip(c, dd))) / f(x) - 1   # noqa: E731
        lx = [mp.log(x) for x in xs]                         # (2) exchange, in log x
        new = []
        for i in range(len(xs)):
            lo = lx[0] if i == 0 else (lx[i - 1] + lx[i]) / 2
            hi = lx[-1] if i == len(xs) - 1 else (lx[i] + lx[i + 1]) / 2
            sg = 1 if err(xs[i]) > 0 else -1
            grid = 24
            vals = [sg * err(mp.e ** (lo + (hi - lo) * j / grid)) for j in range(grid + 1)]
            j = vals.index(max(vals))
            a = lo + (hi - lo) * max(j - 1, 0) / grid
            b = lo + (hi - lo) * min(j + 1, grid) / grid
            best_l = _golden_arg(lambda l: sg * err(mp.e ** l), a, b)
            new.append(mp.e ** best_l)
        new[0], new[-1] = xmin, xmax
        mags = [abs(err(x)) for x in new]
        xs = new
        if (max(mags) - min(mags)) / max(mags) < spread_tol:
            break
    return c0, c, dd, xs, max(mags)


def _golden_arg(g, lo, hi, iters: int = 50):
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
    return c if gc > gd else d


def minimax_pow(alpha, n: int, xmin: float, xmax: float, steps: int = 6):
    """Minimax (relative error) approximation of x^alpha on [xmin, xmax] in the form of eq. 8,
    c0 + sum_k c[k]/(x + d[k]) with n poles; -1 < alpha < 1, alpha != 0 (a Fraction, float or
    mpf).  Returns dict(c0, c[n], d[n], delta), d ascending."""
    with mp.workdps(DPS):
        al = mp.mpf(alpha.numerator) / alpha.denominator if hasattr(alpha, "numerator") else mp.mpf(alpha)
        if not (n >= 1 and 0 < xmin < xmax and -1 < al < 1 and al != 0):
            raise ValueError("need n >= 1, 0 < xmin < xmax, -1 < alpha < 1, alpha != 0")
        xmin_, xmax_ = mp.mpf(xmin), mp.mpf(xmax)
        sign = 1 if al > 0 else -1
        c0, c, d, xs = _start_half(n, xmin_, xmax_, sign)
        half = mp.mpf(sign) / 2
        tol = mp.mpf(10) ** (-14)
        for j in range(steps + 1):
            a_j = half + (al - half) * j / steps
            c0, c, d, xs, delta = _remez_eq8(a_j, c0, list(c), list(d), xs, xmin_, xmax_, tol)
        out = dict(c0=float(c0), c=np.array([float(v) for v in c]), d=np.array([float(v) for v in d]),
                   delta=float(delta))
    order = np.argsort(out["d"])
    out["c"], out["d"] = out["c"][order], out["d"][order]
    return out


def relative_error_curve_pow(alpha: float, c0: float, c, d, x):
    """r(x)/x^alpha - 1 at the points x, evaluated with mpmath from the float coefficients."""
    out = []
    with mp.workdps(DPS):
        for xv in x:
            xv = mp.mpf(float(xv))
            r = mp.mpf(float(c0))
            for ck, dk in zip(c, d):
                r += mp.mpf(float(ck)) / (xv + mp.mpf(float(dk)))
            out.append(float(r / mp.power(xv, mp.mpf(alpha)) - 1))
    return np.array(out)
