// remez.cu -- SURVEY 8(f) NEXT-2, host code only: minimax coefficients of
//     x^alpha ~= c_0 + sum_{k<n} c_k / (x + d_k)      on [xmin, xmax],  -1 < alpha < 1, alpha != 0
// in the relative error -- the paper's eq. 8 for b = 4 (alpha = 1/4, heat bath) and b = -2
// (PAPER.md:131-133), which it takes from Mathematica's MiniMax at 80 digits (appendix :288-304).
//
// Remez exchange directly on the eq. 8 parameters, in IEEE binary128 (__float128, 33 digits: the
// pole/residue Jacobian is far better conditioned than polynomial coefficients, plain double is not
// enough beyond n ~ 12):
//   (1) Newton on the 2n+2 equations r(x_i)/x_i^alpha - 1 = (-1)^i E in (c_0, c_k, log d_k, E);
//   (2) every reference x_i moves to the nearest local extremum of r/x^alpha - 1 (search in log x);
// until the 2n+2 extrema agree to 1e-11 relative.  Newton starts from a closed form: alpha = -1/2 is
// Zolotarev's solution (zolotarev.cu) and alpha = +1/2 is its reciprocal -- if sqrt(y) r(y) oscillates
// in [1-delta, 1+delta] then 1/(sqrt(y) r(y)) oscillates in [1/(1+delta), 1/(1-delta)] at the same
// points -- and alpha is walked from +-1/2 to the target in kSteps steps, each started from the last.
#include <quadmath.h>

#include <cmath>
#include <memory>
#include <new>

#include "internal.cuh"

namespace qcd {

int zolotarev_inv_sqrt(int n, double xmin, double xmax, double *c0, double *c, double *d, double *delta);

namespace {

typedef __float128 q;
constexpr int kMaxM = 2 * kMaxShifts + 2;
constexpr int kSteps = 6;

struct Fit {
    int n;
    q alpha;
    q c0, c[kMaxShifts], u[kMaxShifts];      // u_k = log d_k
    q xs[kMaxM];                             // 2n+2 references, ascending
    q E;

    q r_over_f(q x) const
    {
        q v = c0;
        for (int k = 0; k < n; ++k) v += c[k] / (x + expq(u[k]));
        return v * expq(-alpha * logq(x));
    }
    q err(q x) const { return r_over_f(x) - 1; }
};

// The closed-form start, in binary128 (zolotarev.cu's double version is accurate to ~1e-13, which is
// not inside Newton's basin once delta itself is ~1e-14).  Same construction: AGM ladder in the
// complementary parameter 1/b, amplitudes phi_0, phi_1, a_l = tan^2 phi_0, y_l = 1/dn^2, reflection for
// the upper half.  a[1..2n], ref[0..2n+1], both in y = x/xmin.
void zolotarev_data_q(int n, q b, q *a, q *ref)
{
    q la[48], lc[48];
    int m = 0;
    q a0 = 1, b0 = sqrtq(1 / b);
    la[0] = 1;
    lc[0] = sqrtq(1 - 1 / b);
    while (m < 46) {
        const q an = (a0 + b0) / 2, bn = sqrtq(a0 * b0), cn = (a0 - b0) / 2;
        ++m;
        la[m] = an;
        lc[m] = cn;
        a0 = an;
        b0 = bn;
        if (fabsq(cn) <= (q)1e-34 * an) break;
    }
    const q Kp = 4 * atanq((q)1) / (2 * la[m]);   // pi / (2 a_m)
    const int N = 2 * n + 1;
    for (int l = 1; l <= n; ++l) {
        q phi = ldexpq(la[m] * (l * Kp / N), m), phi1 = phi;
        for (int i = m; i >= 1; --i) {
            if (i == 1) phi1 = phi;
            phi = (phi + asinq(lc[i] / la[i] * sinq(phi))) / 2;
        }
        const q t = tanq(phi), dn = cosq(phi) / cosq(phi1 - phi);
        a[l] = t * t;
        ref[l] = 1 / (dn * dn);
    }
    for (int l = n + 1; l <= 2 * n; ++l) {
        a[l] = b / a[N - l];
        ref[l] = b / ref[N - l];
    }
    ref[0] = 1;
    ref[N] = b;
}

// Solve A z = rhs in place (Gaussian elimination, partial pivoting); false if singular.
bool solve(int m, q (*A)[kMaxM], q *rhs)
{
    for (int col = 0; col < m; ++col) {
        int piv = col;
        for (int i = col + 1; i < m; ++i)
            if (fabsq(A[i][col]) > fabsq(A[piv][col])) piv = i;
        if (A[piv][col] == 0) return false;
        if (piv != col) {
            for (int j = 0; j < m; ++j) { q t = A[col][j]; A[col][j] = A[piv][j]; A[piv][j] = t; }
            q t = rhs[col]; rhs[col] = rhs[piv]; rhs[piv] = t;
        }
        for (int i = col + 1; i < m; ++i) {
            const q f = A[i][col] / A[col][col];
            if (f == 0) continue;
            for (int j = col; j < m; ++j) A[i][j] -= f * A[col][j];
            rhs[i] -= f * rhs[col];
        }
    }
    for (int i = m - 1; i >= 0; --i) {
        q s = rhs[i];
        for (int j = i + 1; j < m; ++j) s -= A[i][j] * rhs[j];
        rhs[i] = s / A[i][i];
    }
    return true;
}

// (1) level the error on the current references; false if Newton breaks down
bool newton(Fit &F, q (*J)[kMaxM])
{
    const int n = F.n, m = 2 * n + 2;
    q g[kMaxM];
    for (int it = 0; it < 25; ++it) {
        q worst = 0;
        for (int i = 0; i < m; ++i) {
            const q x = F.xs[i], inv_f = expq(-F.alpha * logq(x)), sgn = (i & 1) ? -1 : 1;
            q val = F.c0;
            J[i][0] = inv_f;
            for (int k = 0; k < n; ++k) {
                const q dk = expq(F.u[k]), t = 1 / (x + dk);
                val += F.c[k] * t;
                J[i][1 + k] = t * inv_f;
                J[i][1 + n + k] = -F.c[k] * dk * t * t * inv_f;
            }
            J[i][2 * n + 1] = -sgn;
            g[i] = -(val * inv_f - 1 - sgn * F.E);
            if (fabsq(g[i]) > worst) worst = fabsq(g[i]);
        }
        if (!(worst == worst)) return false;
        if (worst < (q)1e-30) return true;           // binary128 rounding in the residuals is ~1e-32
        if (!solve(m, J, g)) return false;
        q big = 0;
        for (int k = 0; k < n; ++k)
            if (fabsq(g[1 + n + k]) > big) big = fabsq(g[1 + n + k]);
        const q lam = big > (q)0.5 ? (q)0.5 / big : 1;          // never move a pole by more than e^(1/2)
        F.c0 += lam * g[0];
        for (int k = 0; k < n; ++k) { F.c[k] += lam * g[1 + k]; F.u[k] += lam * g[1 + n + k]; }
        F.E += lam * g[2 * n + 1];
    }
    return true;     // not fully converged: the exchange loop decides whether the fit is good enough
}

// (2) exchange; returns the relative spread of the new extrema and their largest magnitude
q exchange(Fit &F, q xmin, q xmax, q &largest)
{
    const int m = 2 * F.n + 2;
    q lx[kMaxM], nx[kMaxM];
    for (int i = 0; i < m; ++i) lx[i] = logq(F.xs[i]);
    const q phi = (sqrtq((q)5.0) - 1) / 2;
    for (int i = 0; i < m; ++i) {
        const q lo = i == 0 ? lx[0] : (lx[i - 1] + lx[i]) / 2;
        const q hi = i == m - 1 ? lx[m - 1] : (lx[i] + lx[i + 1]) / 2;
        const q sg = F.err(F.xs[i]) > 0 ? 1 : -1;
        constexpr int grid = 16;
        int jb = 0;
        q best = -(q)1e300;
        for (int j = 0; j <= grid; ++j) {
            const q v = sg * F.err(expq(lo + (hi - lo) * j / grid));
            if (v > best) { best = v; jb = j; }
        }
        q a = lo + (hi - lo) * (jb > 0 ? jb - 1 : 0) / grid, b = lo + (hi - lo) * (jb < grid ? jb + 1 : grid) / grid;
        q c = b - phi * (b - a), d = a + phi * (b - a);
        q gc = sg * F.err(expq(c)), gd = sg * F.err(expq(d));
        for (int it = 0; it < 70; ++it) {                   // golden section: (b-a) shrinks by 0.618^70
            if (gc > gd) { b = d; d = c; gd = gc; c = b - phi * (b - a); gc = sg * F.err(expq(c)); }
            else { a = c; c = d; gc = gd; d = a + phi * (b - a); gd = sg * F.err(expq(d)); }
        }
        nx[i] = expq(gc > gd ? c : d);
    }
    nx[0] = xmin;
    nx[m - 1] = xmax;
    q mn = (q)1e300;
    largest = 0;
    for (int i = 0; i < m; ++i) {
        F.xs[i] = nx[i];
        const q e = fabsq(F.err(nx[i]));
        if (e > largest) largest = e;
        if (e < mn) mn = e;
    }
    return (largest - mn) / largest;
}

}  // namespace

// alpha = num/den.  Returns 0 ok, 1 bad arguments, 2 did not converge.  d ascending.
int remez_pow(int num, int den, int n, double xmin, double xmax, double *c0, double *c, double *d,
              double *delta)
{
    if (den == 0 || num == 0 || n < 1 || n > kMaxShifts || !(xmin > 0.0) || !(xmax > xmin) ||
        !std::isfinite(xmax))
        return 1;
    const q target = (q)num / (q)den;
    if (!(fabsq(target) < 1)) return 1;
    q a[kMaxM], ref[kMaxM];
    zolotarev_data_q(n, (q)xmax / (q)xmin, a, ref);
    {   // over-resolved: when even the closed form at alpha = -1/2 is at the rounding level of the double
        // coefficients, the exchange has nothing left to level (and would take a minute to say so)
        double zc0, zc[kMaxShifts], zd[kMaxShifts], zdelta = 0.0;
        if (zolotarev_inv_sqrt(n, xmin, xmax, &zc0, zc, zd, &zdelta) != 0) return 1;
        if (zdelta < 2e-15) return 2;
    }
    std::unique_ptr<q[][kMaxM]> Jbuf(new (std::nothrow) q[kMaxM][kMaxM]);   // 270 KB: not on the stack
    if (!Jbuf) return 2;
    q(*J)[kMaxM] = Jbuf.get();
    Fit F;
    F.n = n;
    F.E = 0;
    const int sign = target > 0 ? 1 : -1;
    // closed-form start in x = xmin y: poles/zeros of r (alpha = -1/2) or of 1/r (alpha = +1/2)
    for (int k = 0; k < n; ++k) {
        const q pole = sign < 0 ? a[2 * k + 1] : a[2 * k + 2];
        q v = 1;
        for (int l = 0; l < n; ++l) v *= (sign < 0 ? a[2 * l + 2] : a[2 * l + 1]) - pole;
        for (int j = 0; j < n; ++j)
            if (j != k) v /= (sign < 0 ? a[2 * j + 1] : a[2 * j + 2]) - pole;
        const q s = sign > 0 ? sqrtq((q)xmin) : 1 / sqrtq((q)xmin);
        F.c[k] = s * v * (q)xmin;
        F.u[k] = logq(pole * (q)xmin);
        F.c0 = s;
    }
    for (int j = 0; j <= 2 * n + 1; ++j) F.xs[j] = ref[j] * (q)xmin;
    F.xs[0] = xmin;
    F.xs[2 * n + 1] = xmax;
    const q half = (q)sign / 2;
    q largest = 0;
    for (int step = 0; step <= kSteps; ++step) {
        F.alpha = half + (target - half) * step / kSteps;
        bool ok = false;
        for (int outer = 0; outer < 20; ++outer) {
            if (!newton(F, J)) return 2;
            if (exchange(F, xmin, xmax, largest) < (q)1e-11) { ok = true; break; }
            // the error is already far below what the double coefficients returned can express:
            // levelling it further is noise in binary128
            if (largest < (q)1e-19) { ok = true; break; }
        }
        if (!ok) return 2;
    }
    *c0 = (double)F.c0;
    for (int k = 0; k < n; ++k) { c[k] = (double)F.c[k]; d[k] = (double)expq(F.u[k]); }
    for (int i = 1; i < n; ++i)                       // poles stay ordered in practice; make sure
        for (int j = i; j > 0 && d[j] < d[j - 1]; --j) {
            double t = d[j]; d[j] = d[j - 1]; d[j - 1] = t;
            t = c[j]; c[j] = c[j - 1]; c[j - 1] = t;
        }
    if (delta) *delta = (double)largest;
    return 0;
}

}  // namespace qcd
