// zolotarev.cu -- SURVEY 8(f) NEXT-2, host code only: coefficients of the rational approximation
//     x^(-1/2) ~= c_0 + sum_{k<n} c_k / (x + d_k)        on [xmin, xmax]            (eq. 8)
// The paper obtains them from Mathematica's MiniMax (appendix :288-304) in 80-digit
// arithmetic and prints none.  For the exponent -1/2 the minimax problem (relative error, type
// (n,n)) has Zolotarev's closed-form solution in Jacobi elliptic functions, which is well
// conditioned in plain double precision when written in terms of the COMPLEMENTARY parameter
// 1/b = xmin/xmax (never 1 - small):
//     a_l = sn^2(l K'/N; k') / cn^2(l K'/N; k'),  k'^2 = 1 - 1/b,  N = 2n+1,  l = 1..2n
//     r(y) = D prod_{l=1..n} (y + a_{2l}) / prod_{l=1..n} (y + a_{2l-1}),   y = x/xmin
// The relative error 1 - sqrt(y) r(y) equioscillates at y_j = 1/dn^2(j K'/N; k'), j = 0..N, so D
// and delta follow from the values at y_0 = 1 and y_1 alone.  Everything here is this file's own:
// the AGM evaluation of sn/cn/dn, the reflection a_l a_{N-l} = b for the large coefficients, the
// partial fractions.  The oracle (oracle/rational.py) computes the same object with mpmath in 50
// digits and a brute-force search for D, and is pinned by the equioscillation theorem.
#include <cmath>

#include "internal.cuh"

namespace qcd {

namespace {

// Arithmetic-geometric-mean ladder for parameter m = 1 - mc (Abramowitz & Stegun 16.4, 17.6).
struct Agm {
    double a[40], c[40];
    int n;
    explicit Agm(double mc)
    {
        double a0 = 1.0, b0 = std::sqrt(mc);
        a[0] = a0;
        c[0] = std::sqrt(1.0 - mc);
        n = 0;
        while (n < 38) {
            const double an = 0.5 * (a0 + b0), bn = std::sqrt(a0 * b0), cn = 0.5 * (a0 - b0);
            ++n;
            a[n] = an;
            c[n] = cn;
            a0 = an;
            b0 = bn;
            if (std::fabs(cn) <= 1e-17 * an) break;
        }
    }
    double K() const { return M_PI / (2.0 * a[n]); }
    // amplitude phi_0 (sn = sin, cn = cos) and phi_1 (dn = cos phi_0 / cos(phi_1 - phi_0))
    void amplitude(double u, double &phi0, double &phi1) const
    {
        double phi = std::ldexp(a[n] * u, n);
        phi1 = phi;
        for (int i = n; i >= 1; --i) {
            if (i == 1) phi1 = phi;
            phi = 0.5 * (phi + std::asin(c[i] / a[i] * std::sin(phi)));
        }
        phi0 = phi;
    }
};

}  // namespace

// The raw Zolotarev data for b = xmax/xmin and N = 2n+1, in the scaled variable y = x/xmin:
//   a[l], l = 1..2n (a[0] unused):  a_l = sn^2/cn^2 (l K'/N)      -- poles (odd l) and zeros (even l) of r
//   ref[j], j = 0..N:               y_j = 1/dn^2(j K'/N)          -- the 2n+2 equioscillation points
// Returns 0, or 1 for bad arguments.
int zolotarev_data(int n, double xmin, double xmax, double *a, double *ref)
{
    if (n < 1 || n > kMaxShifts || !(xmin > 0.0) || !(xmax > xmin) || !std::isfinite(xmax)) return 1;
    const double b = xmax / xmin;
    const Agm agm(1.0 / b);
    const double Kp = agm.K();
    const int N = 2 * n + 1;
    for (int l = 1; l <= n; ++l) {
        double p0, p1;
        agm.amplitude(l * Kp / N, p0, p1);
        const double t = std::tan(p0);
        a[l] = t * t;
        if (ref) {
            const double dn = std::cos(p0) / std::cos(p1 - p0);
            ref[l] = 1.0 / (dn * dn);
        }
    }
    for (int l = n + 1; l <= 2 * n; ++l) {
        a[l] = b / a[N - l];                            // sn(K'-u) = cn(u)/dn(u)
        if (ref) ref[l] = b / ref[N - l];               // dn(K'-u) = k/dn(u), k^2 = 1/b
    }
    if (ref) { ref[0] = 1.0; ref[N] = b; }
    return 0;
}

// Returns 0, 1 for bad arguments, 2 if a coefficient is not finite.  c and d hold n doubles each, d ascending.
int zolotarev_inv_sqrt(int n, double xmin, double xmax, double *c0, double *c, double *d, double *delta)
{
    double a[2 * kMaxShifts + 2], ref[2 * kMaxShifts + 2];
    if (zolotarev_data(n, xmin, xmax, a, ref) != 0) return 1;
    // den_k = a_{2k-1}, num_k = a_{2k}, k = 1..n
    auto f = [&](double y) {                            // sqrt(y) prod (y+num)/(y+den)
        double v = std::sqrt(y);
        for (int k = 1; k <= n; ++k) v *= (y + a[2 * k]) / (y + a[2 * k - 1]);
        return v;
    };
    const double f0 = f(1.0), f1 = f(ref[1]);
    const double D = 2.0 / (f0 + f1);
    if (delta) *delta = std::fabs(f0 - f1) / (f0 + f1);
    // partial fractions in y, then x = xmin y:  1/sqrt(x) = r(y)/sqrt(xmin)
    const double s = std::sqrt(xmin);
    *c0 = D / s;
    for (int k = 1; k <= n; ++k) {
        const double dk = a[2 * k - 1];
        // numerator and denominator factors taken in pairs: the interlacing a_1 < a_2 < ... keeps every
        // ratio and every partial product bounded (by xmax/xmin), where the product of all n numerator
        // factors alone grows like (xmax/xmin)^(n/2) and overflows for large n on wide intervals
        double v = D * (a[2 * k] - dk);
        for (int l = 1; l <= n; ++l)
            if (l != k) v *= (a[2 * l] - dk) / (a[2 * l - 1] - dk);
        c[k - 1] = v * s;
        d[k - 1] = dk * xmin;
    }
    if (!std::isfinite(*c0)) return 2;
    for (int k = 0; k < n; ++k)
        if (!std::isfinite(c[k]) || !std::isfinite(d[k]) || !(d[k] > 0.0)) return 2;
    return 0;
}

}  // namespace qcd
