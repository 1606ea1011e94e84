/*
 * staggered_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct fp64 implementation of what the hot path of
 * arXiv:1710.09178 (Gupta & Majumdar) computes, written from the paper's
 * definitions, for checking the CUDA library against.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may call it.  It shares NO code with paper_1710_09178_b200/ (no header, no
 * index helper, no constant): the two are independent restatements.
 *
 * What is computed, and the passage each function follows
 * -------------------------------------------------------
 *   orc_D_full      (D psi)(x) on the whole lattice.  PAPER.md:106 (M_ik: forward
 *                   hop U_{i,mu} delta_{i,k-mu}, backward hop -U^dag_{i-mu,mu}
 *                   delta_{i,k+mu}), in the 1/2-normalised form of BASELINE.json
 *                   north_star (M = m + D), with the staggered
 *                   phases eta_mu(x) the paper "absorbed into the U's"
 *                   (convention SURVEY.md C4) and antiperiodic
 *                   time boundary (north_star) written out.
 *   orc_dslash      D_oe / D_eo: D restricted to one input parity and the other
 *                   output parity.  PAPER.md:110-112 (block form), parity =
 *                   (x+y+z+t) mod 2 (Fig. 2).
 *   orc_mdagm       (M^dag M)_pp = m^2 - D_{p,q} D_{q,p}.  PAPER.md:114-119.
 *   orc_cg          textbook single-system conjugate gradient.
 *   orc_multishift_cg   the shifted CG of PAPER.md:136 ([5] Jegerlehner, [6]
 *                   Clark-Kennedy); the paper prints no recurrences, so the
 *                   standard CG-M construction of SURVEY.md 8(c.2) is followed
 *                   line by line, same symbols.  Evaluates the partial-fraction
 *                   sum of eq. 8: y = sum_k c_k x_k.
 *   orc_polish      defect correction of each x_k down to the fp64 floor so the
 *                   result can stand for the exact solution.
 *
 * Layouts (canonical exchange layout, the same buffers the CUDA library gets):
 *   site address l = ((t*Nz + z)*Ny + y)*Nx + x           (PAPER.md:43, 0-based)
 *   links   double[V][4][3][3][2]  U_mu(l)[row][col] (re,im)   72 V doubles
 *   full vector   double[V][3][2]                              6 V doubles
 *   parity vector double[V/2][3][2]: sites of that parity in increasing l
 *
 * Pins (tests/test_oracle_*.py): free-field spectrum m^2 + sum sin^2 p_mu on
 * antiperiodic momenta, plane waves, anti-hermiticity, gauge covariance,
 * hand-derived matrix elements (tests/golden/), D_ee = D_oo = 0, dense
 * numpy.linalg.solve on 2^4 and 4^4, eq. 8 via eigh, multishift vs
 * single-shift CG.  Nothing here is "parity unpinned".
 *
 * Reductions are accumulated in long double.
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double _Complex cplx;

typedef struct orc_lattice {
    int N[4];            /* Nx, Ny, Nz, Nt */
    long V;              /* number of sites */
    const cplx *U;       /* borrowed: U[(l*4+mu)*9 + row*3 + col] */
    signed char *par;    /* par[l] = (x+y+z+t) mod 2 */
    long *half;          /* half[l] = rank of l among the sites of its parity */
    cplx *full_a;        /* scratch: one full-lattice vector */
    cplx *half_a;        /* scratch: one parity vector */
} orc_lattice;

int orc_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

static long site_address(const int N[4], int x, int y, int z, int t)
{
    return (((long)t * N[2] + z) * N[1] + y) * N[0] + x;
}

static void site_coords(const int N[4], long l, int c[4])
{
    c[0] = (int)(l % N[0]); l /= N[0];
    c[1] = (int)(l % N[1]); l /= N[1];
    c[2] = (int)(l % N[2]); l /= N[2];
    c[3] = (int)l;
}

orc_lattice *orc_create(const int dims[4], const double *links)
{
    orc_lattice *L = (orc_lattice *)calloc(1, sizeof *L);
    if (!L) return NULL;
    for (int i = 0; i < 4; i++) L->N[i] = dims[i];
    L->V = (long)dims[0] * dims[1] * dims[2] * dims[3];
    L->U = (const cplx *)links;
    L->par = (signed char *)malloc((size_t)L->V);
    L->half = (long *)malloc((size_t)L->V * sizeof(long));
    L->full_a = (cplx *)malloc((size_t)L->V * 3 * sizeof(cplx));
    L->half_a = (cplx *)malloc((size_t)(L->V / 2) * 3 * sizeof(cplx));
    if (!L->par || !L->half || !L->full_a || !L->half_a) return NULL;
    long count[2] = {0, 0};
    for (long l = 0; l < L->V; l++) {
        int c[4];
        site_coords(L->N, l, c);
        int p = (c[0] + c[1] + c[2] + c[3]) & 1;
        L->par[l] = (signed char)p;
        L->half[l] = count[p]++;
    }
    return L;
}

void orc_destroy(orc_lattice *L)
{
    if (!L) return;
    free(L->par); free(L->half); free(L->full_a); free(L->half_a);
    free(L);
}

/* eta_mu(x) = (-1)^(sum_{nu<mu} x_nu), mu order x,y,z,t */
static double eta_phase(int mu, const int c[4])
{
    int s = 0;
    for (int nu = 0; nu < mu; nu++) s += c[nu];
    return (s & 1) ? -1.0 : 1.0;
}

/*
 * (D psi)(x) = 1/2 sum_mu eta_mu(x) [ s+ U_mu(x) psi(x+mu) - s- U_mu(x-mu)^dag psi(x-mu) ]
 * s+ = -1 on a hop across t = Nt-1 -> 0, s- = -1 on a hop across t = 0 -> Nt-1
 * (antiperiodic in t), periodic in x, y, z.   PAPER.md:106; SURVEY.md 8(c.1).
 * Extents of 2: x+mu and x-mu coincide; both terms are still added (C8).
 */
static void site_D(const orc_lattice *L, const cplx *psi, long l, cplx out[3])
{
    int c[4];
    site_coords(L->N, l, c);
    out[0] = out[1] = out[2] = 0.0;
    for (int mu = 0; mu < 4; mu++) {
        int cp[4] = {c[0], c[1], c[2], c[3]};
        int cm[4] = {c[0], c[1], c[2], c[3]};
        cp[mu] = (c[mu] + 1) % L->N[mu];
        cm[mu] = (c[mu] - 1 + L->N[mu]) % L->N[mu];
        long lp = site_address(L->N, cp[0], cp[1], cp[2], cp[3]);
        long lm = site_address(L->N, cm[0], cm[1], cm[2], cm[3]);
        double splus = (mu == 3 && c[3] == L->N[3] - 1) ? -1.0 : 1.0;
        double sminus = (mu == 3 && c[3] == 0) ? -1.0 : 1.0;
        double eta = eta_phase(mu, c);
        const cplx *Ux = L->U + (l * 4 + mu) * 9;    /* U_mu(x)      */
        const cplx *Um = L->U + (lm * 4 + mu) * 9;   /* U_mu(x - mu) */
        for (int a = 0; a < 3; a++) {
            cplx fwd = 0.0, bwd = 0.0;
            for (int b = 0; b < 3; b++) {
                fwd += Ux[a * 3 + b] * psi[lp * 3 + b];
                bwd += conj(Um[b * 3 + a]) * psi[lm * 3 + b];
            }
            out[a] += 0.5 * eta * (splus * fwd - sminus * bwd);
        }
    }
}

/* D on the whole lattice: full vector -> full vector. */
void orc_D_full(orc_lattice *L, const double *psi_, double *out_)
{
    const cplx *psi = (const cplx *)psi_;
    cplx *out = (cplx *)out_;
#pragma omp parallel for schedule(static)
    for (long l = 0; l < L->V; l++) site_D(L, psi, l, out + l * 3);
}

/*
 * D_{out_parity, other}: input lives on the sites of parity 1-out_parity, output on
 * the sites of out_parity (D_oe = even in -> odd out).
 * Written as the definition: embed the input in a full-lattice vector that is zero
 * on the other parity, apply D, keep the sites of out_parity.
 */
static void dslash_into(orc_lattice *L, int out_parity, const cplx *in, cplx *out, cplx *full)
{
#pragma omp parallel for schedule(static)
    for (long l = 0; l < L->V; l++) {
        if (L->par[l] != out_parity)
            for (int a = 0; a < 3; a++) full[l * 3 + a] = in[L->half[l] * 3 + a];
        else
            for (int a = 0; a < 3; a++) full[l * 3 + a] = 0.0;
    }
#pragma omp parallel for schedule(static)
    for (long l = 0; l < L->V; l++)
        if (L->par[l] == out_parity) site_D(L, full, l, out + L->half[l] * 3);
}

void orc_dslash(orc_lattice *L, int out_parity, const double *in, double *out)
{
    dslash_into(L, out_parity, (const cplx *)in, (cplx *)out, L->full_a);
}

/* (M^dag M)_pp in = m^2 in - D_{p,q} D_{q,p} in     (C3) */
static void mdagm_into(orc_lattice *L, double mass, int parity, const cplx *in, cplx *out)
{
    long n = (L->V / 2) * 3;
    dslash_into(L, 1 - parity, in, L->half_a, L->full_a);
    dslash_into(L, parity, L->half_a, out, L->full_a);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < n; i++) out[i] = mass * mass * in[i] - out[i];
}

void orc_mdagm(orc_lattice *L, double mass, int parity, const double *in, double *out)
{
    mdagm_into(L, mass, parity, (const cplx *)in, (cplx *)out);
}

/* <a,b> = sum conj(a) b ; only the real part is ever needed */
static double re_dot(long n, const cplx *a, const cplx *b)
{
    long double s = 0.0L;
#pragma omp parallel for schedule(static) reduction(+ : s)
    for (long i = 0; i < n; i++)
        s += (long double)creal(a[i]) * creal(b[i]) + (long double)cimag(a[i]) * cimag(b[i]);
    return (double)s;
}

/* ||b - (A + sigma) x|| / ||b||, recomputed from scratch (not a recursion value) */
static double true_residual(orc_lattice *L, double mass, int parity, double sigma,
                            const cplx *b, const cplx *x, cplx *work, cplx *rout)
{
    long n = (L->V / 2) * 3;
    mdagm_into(L, mass, parity, x, work);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < n; i++) work[i] = b[i] - (work[i] + sigma * x[i]);
    if (rout) memcpy(rout, work, (size_t)n * sizeof(cplx));
    return sqrt(re_dot(n, work, work) / re_dot(n, b, b));
}

/*
 * Textbook CG for (A + sigma) x = b, A = (M^dag M)_pp, starting from the x passed
 * in.  Stops when the recursion residual satisfies ||r|| <= tol ||b||.
 * Returns 0 if converged, 1 if max_iter was hit.
 */
int orc_cg(orc_lattice *L, double mass, int parity, double sigma, const double *b_,
           double *x_, double tol, int max_iter, int *iterations, double *true_res)
{
    long n = (L->V / 2) * 3;
    const cplx *b = (const cplx *)b_;
    cplx *x = (cplx *)x_;
    cplx *r = (cplx *)malloc((size_t)n * sizeof(cplx));
    cplx *p = (cplx *)malloc((size_t)n * sizeof(cplx));
    cplx *q = (cplx *)malloc((size_t)n * sizeof(cplx));
    double rho_b = re_dot(n, b, b);
    true_residual(L, mass, parity, sigma, b, x, q, r); /* r = b - (A+sigma) x */
    memcpy(p, r, (size_t)n * sizeof(cplx));
    double rho = re_dot(n, r, r);
    int it = 0, status = 1;
    if (sqrt(rho / rho_b) <= tol) status = 0;
    while (status && it < max_iter) {
        mdagm_into(L, mass, parity, p, q);
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; i++) q[i] += sigma * p[i];
        double alpha = rho / re_dot(n, p, q);
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; i++) { x[i] += alpha * p[i]; r[i] -= alpha * q[i]; }
        double rho_new = re_dot(n, r, r);
        double beta = rho_new / rho;
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; i++) p[i] = r[i] + beta * p[i];
        rho = rho_new;
        it++;
        if (sqrt(rho / rho_b) <= tol) status = 0;
    }
    if (iterations) *iterations = it;
    if (true_res) *true_res = true_residual(L, mass, parity, sigma, b, x, q, NULL);
    free(r); free(p); free(q);
    return status;
}

/*
 * Multishift CG, SURVEY.md 8(c.2) line by line.  A = (M^dag M)_pp, shifts sigma_k >= 0.
 * Internally sorted so sigma_0 is the smallest (base system, C12); outputs are in the
 * caller's order.  x: nshift parity vectors (may be NULL), y = sum_k residues[k] x_k
 * (may be NULL), true_res[k] recomputed (C10).  freeze_factor = f of C13 (0.1).
 * Returns 0 if converged, 1 if max_iter was hit.
 */
int orc_multishift_cg(orc_lattice *L, double mass, int parity, const double *b_, int nshift,
                      const double *shifts, const double *residues, double tol, int max_iter,
                      double freeze_factor, double *x_out, double *y_out, int *iterations,
                      double *true_res)
{
    long n = (L->V / 2) * 3;
    const cplx *b = (const cplx *)b_;
    int N = nshift;
    int *order = (int *)malloc((size_t)N * sizeof(int));   /* order[k] = caller index of k-th smallest */
    for (int k = 0; k < N; k++) order[k] = k;
    for (int i = 1; i < N; i++)                              /* insertion sort, stable */
        for (int j = i; j > 0 && shifts[order[j]] < shifts[order[j - 1]]; j--) {
            int tmp = order[j]; order[j] = order[j - 1]; order[j - 1] = tmp;
        }
    double *sigma = (double *)malloc((size_t)N * sizeof(double));
    for (int k = 0; k < N; k++) sigma[k] = shifts[order[k]];

    cplx **x = (cplx **)malloc((size_t)N * sizeof(cplx *));
    cplx **p = (cplx **)malloc((size_t)N * sizeof(cplx *));
    for (int k = 0; k < N; k++) {
        x[k] = (cplx *)calloc((size_t)n, sizeof(cplx));      /* x_k = 0 (C11) */
        p[k] = (cplx *)malloc((size_t)n * sizeof(cplx));
        memcpy(p[k], b, (size_t)n * sizeof(cplx));           /* p_k = b */
    }
    cplx *r = (cplx *)malloc((size_t)n * sizeof(cplx));
    cplx *q = (cplx *)malloc((size_t)n * sizeof(cplx));
    memcpy(r, b, (size_t)n * sizeof(cplx));                  /* r = b */
    double rho = re_dot(n, r, r), rho_b = rho;
    double *zeta = (double *)malloc((size_t)N * sizeof(double));
    double *zeta_old = (double *)malloc((size_t)N * sizeof(double));
    double *zeta_new = (double *)malloc((size_t)N * sizeof(double));
    double *alpha_k = (double *)malloc((size_t)N * sizeof(double));
    int *active = (int *)malloc((size_t)N * sizeof(int));
    for (int k = 0; k < N; k++) { zeta[k] = zeta_old[k] = 1.0; active[k] = 1; }
    double alpha_old = 1.0, beta_old = 0.0;

    int it = 0, status = 1;
    if (rho_b == 0.0) status = 0;
    while (status && it < max_iter) {
        /* q = A p_0 + sigma_0 p_0 */
        mdagm_into(L, mass, parity, p[0], q);
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; i++) q[i] += sigma[0] * p[0][i];
        double alpha = rho / re_dot(n, p[0], q);
        for (int k = 0; k < N; k++) {
            if (!active[k]) continue;
            double delta = sigma[k] - sigma[0];
            zeta_new[k] = zeta[k] * zeta_old[k] * alpha_old /
                          (alpha * beta_old * (zeta_old[k] - zeta[k]) +
                           zeta_old[k] * alpha_old * (1.0 + delta * alpha));
            alpha_k[k] = alpha * zeta_new[k] / zeta[k];
        }
        for (int k = 0; k < N; k++) {
            if (!active[k]) continue;
            cplx *xk = x[k], *pk = p[k];
            double ak = alpha_k[k];
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; i++) xk[i] += ak * pk[i];
        }
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; i++) r[i] -= alpha * q[i];
        double rho_new = re_dot(n, r, r);
        double beta = rho_new / rho;
        for (int k = 0; k < N; k++) {
            if (!active[k]) continue;
            double ratio = zeta_new[k] / zeta[k];
            double bk = beta * ratio * ratio, zk = zeta_new[k];
            cplx *pk = p[k];
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; i++) pk[i] = zk * r[i] + bk * pk[i];
        }
        for (int k = 0; k < N; k++) {
            if (!active[k]) continue;
            zeta_old[k] = zeta[k];
            zeta[k] = zeta_new[k];
        }
        alpha_old = alpha; beta_old = beta; rho = rho_new;
        it++;
        for (int k = 1; k < N; k++)                           /* never freeze the base (C13) */
            if (active[k] && fabs(zeta[k]) * sqrt(rho) <= freeze_factor * tol * sqrt(rho_b))
                active[k] = 0;
        if (sqrt(rho / rho_b) <= tol) status = 0;
    }
    if (iterations) *iterations = it;

    if (y_out) {
        cplx *y = (cplx *)y_out;
        memset(y, 0, (size_t)n * sizeof(cplx));
        for (int k = 0; k < N; k++) {                         /* eq. 8: sum_k c_k x_k */
            double ck = residues[order[k]];
            cplx *xk = x[k];
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; i++) y[i] += ck * xk[i];
        }
    }
    for (int k = 0; k < N; k++) {
        if (true_res)
            true_res[order[k]] = true_residual(L, mass, parity, sigma[k], b, x[k], q, NULL);
        if (x_out) memcpy((cplx *)x_out + (long)order[k] * n, x[k], (size_t)n * sizeof(cplx));
    }
    for (int k = 0; k < N; k++) { free(x[k]); free(p[k]); }
    free(x); free(p); free(r); free(q); free(order); free(sigma);
    free(zeta); free(zeta_old); free(zeta_new); free(alpha_k); free(active);
    return status;
}

/*
 * Polish x (one shift) to the fp64 floor by defect correction:
 *   r = b - (A+sigma) x (recomputed);  solve (A+sigma) e = r by CG;  x += e;
 * repeated until the true residual stops decreasing by at least a factor 2.
 * Returns the final true relative residual.
 */
double orc_polish(orc_lattice *L, double mass, int parity, double sigma, const double *b_,
                  double *x_, int max_rounds, int max_iter)
{
    long n = (L->V / 2) * 3;
    const cplx *b = (const cplx *)b_;
    cplx *x = (cplx *)x_;
    cplx *r = (cplx *)malloc((size_t)n * sizeof(cplx));
    cplx *e = (cplx *)malloc((size_t)n * sizeof(cplx));
    cplx *w = (cplx *)malloc((size_t)n * sizeof(cplx));
    cplx *xtry = (cplx *)malloc((size_t)n * sizeof(cplx));
    double res = true_residual(L, mass, parity, sigma, b, x, w, r);
    for (int round = 0; round < max_rounds && res > 0.0; round++) {
        memset(e, 0, (size_t)n * sizeof(cplx));
        int its;
        orc_cg(L, mass, parity, sigma, (const double *)r, (double *)e, 1e-8, max_iter, &its, NULL);
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; i++) xtry[i] = x[i] + e[i];
        double res_try = true_residual(L, mass, parity, sigma, b, xtry, w, e);
        if (res_try < res) {
            int big_step = res_try < 0.5 * res;
            memcpy(x, xtry, (size_t)n * sizeof(cplx));
            memcpy(r, e, (size_t)n * sizeof(cplx));
            res = res_try;
            if (!big_step) break;
        } else {
            break;
        }
    }
    free(r); free(e); free(w); free(xtry);
    return res;
}
