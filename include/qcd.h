/*
 * qcd.h -- C ABI of the B200-native staggered-fermion hot path of arXiv:1710.09178
 * (Gupta & Majumdar): the even-odd staggered Dirac operator D_oe / D_eo, the
 * single-parity normal operator (M^dag M)_pp = m^2 - D_pq D_qp, and the multishift
 * conjugate gradient that evaluates the partial-fraction sum of the rational
 * approximation (eq. 8).  Citations are PAPER.md:<line>; "SURVEY C<n>" names a
 * reading of the paper listed in SURVEY.md 8(c) and DESIGN.md.
 *
 * Conventions
 * -----------
 *  Lattice     sites x = (x,y,z,t), 0 <= x_mu < N_mu, all N_mu even and >= 2.
 *              canonical address l = ((t*Nz + z)*Ny + y)*Nx + x        (PAPER.md:43, 0-based)
 *              parity(x) = (x+y+z+t) mod 2, QCD_EVEN = 0                (Fig. 2; C2)
 *  Operator    (D psi)(x) = 1/2 sum_mu eta_mu(x) [ s+ U_mu(x) psi(x+mu) - s- U_mu(x-mu)^dag psi(x-mu) ]
 *              (PAPER.md:106 in the M = m + D normalisation, C1), eta_0 = 1, eta_1 = (-1)^x,
 *              eta_2 = (-1)^(x+y), eta_3 = (-1)^(x+y+z) (C4); periodic in x,y,z, antiperiodic
 *              in t: s+ = -1 on the hop t = Nt-1 -> 0, s- = -1 on the hop t = 0 -> Nt-1 (C5).
 *  Canonical layouts (what callers exchange; fp64, little-endian, (re,im) pairs):
 *              links          double[V][4][3][3][2] = U_mu(l)[row][col]     72 V doubles
 *              parity vector  double[V/2][3][2], the sites of ONE parity in increasing l
 *                             (a full colour vector is 6 V doubles)
 *  Internal layout            the library's own parity-split, site-fastest SoA ("ap(V,3)",
 *              PAPER.md:210): an internal vector is 6*(V/2) doubles, opaque to the caller;
 *              qcd_pack / qcd_unpack convert.
 *  Alignment   EVERY device buffer passed to the library (canonical links and vectors, internal
 *              vectors, d_x, d_y) must be 16-byte aligned -- they are accessed with 16-byte loads
 *              and stores -- and input and output ranges must not overlap; either violation
 *              returns QCD_EINVAL before anything is launched.
 *  Pointers    d_* = DEVICE memory owned by the caller (e.g. torch.empty(...).data_ptr());
 *              h_* = HOST memory owned by the caller.  The library owns only its handle, its
 *              reordered gauge copy and its workspace, all released by qcd_destroy.
 *              No pointer is retained after a call returns.
 *  Streams     all work is enqueued on the context's stream.  qcd_dslash, qcd_mdagm, qcd_pack,
 *              qcd_unpack, qcd_load_gauge return WITHOUT synchronising.  Calls that return host
 *              scalars or fill host buffers (qcd_multishift_cg, *_host) synchronise the stream
 *              before returning.
 *  Errors      every call returns a qcd_status; nothing aborts or throws across the ABI.
 *              qcd_last_error() gives the text of the last failure on that context (or of the
 *              last failed qcd_create when ctx == NULL).
 *  No CPU fallback: without an sm_100 CUDA device qcd_create returns QCD_ECUDA.
 */
#ifndef QCD_H
#define QCD_H

#ifdef __cplusplus
extern "C" {
#endif

#define QCD_API __attribute__((visibility("default")))

typedef struct qcd_ctx qcd_ctx; /* opaque; owned by the library */

typedef enum {
    QCD_OK = 0,
    QCD_EINVAL = 1,   /* bad argument: odd or < 2 extent, NULL pointer, negative shift, nshift < 1 or
                         > QCD_MAX_SHIFTS, tol <= 0, bad parity, overlapping in/out ranges, a device
                         pointer that is not 16-byte aligned */
    QCD_ENOMEM = 2,   /* device or host allocation failed */
    QCD_ECUDA = 3,    /* CUDA error, or no sm_100 device */
    QCD_ENOTCONV = 4, /* max_iter reached; outputs are still written and true_res filled */
    QCD_ESTATE = 5    /* operator used before qcd_load_gauge */
} qcd_status;

enum { QCD_EVEN = 0, QCD_ODD = 1 };
enum { QCD_MAX_SHIFTS = 64 };

/* Library version string, e.g. "qcd_b200 0.1 (sm_100a)". */
QCD_API const char *qcd_version(void);

/* Create a context for an Nx x Ny x Nz x Nt lattice (dims = {Nx,Ny,Nz,Nt}) and quark mass m.
 * cuda_stream: a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream) or NULL for the
 * default stream.  Uses the calling thread's current CUDA device. */
QCD_API qcd_status qcd_create(const int dims[4], double mass, void *cuda_stream, qcd_ctx **out);
QCD_API qcd_status qcd_destroy(qcd_ctx *ctx);
QCD_API qcd_status qcd_set_mass(qcd_ctx *ctx, double mass);
QCD_API qcd_status qcd_set_stream(qcd_ctx *ctx, void *cuda_stream);

/* Execution options.  PDL, CG_GRAPH and CG_BATCH leave every result bit-identical.
 *   QCD_OPT_PDL       (default 1) launch every kernel with programmatic dependent launch, so that its
 *                     index arithmetic overlaps the tail of its predecessor in the stream or graph.
 *   QCD_OPT_CG_GRAPH  (default 1) how qcd_multishift_cg enqueues its iterations.  0: four kernel launches
 *                     per iteration from the host.  1: one captured CUDA graph per batch of iterations.
 *                     2: ONE graph for the whole solve, a WHILE conditional node whose body is one
 *                     iteration and whose condition the device-side stop test sets: no early-exit
 *                     launches after convergence, no host polling.  Measured on B200 it is no faster
 *                     than 1 (7.93 vs 7.84 ms at 32^3x8, 5.69 vs 5.31 ms at 4^4): the loop node costs
 *                     about 1 us per iteration and breaks the PDL chain between iterations.
 *   QCD_OPT_CG_BATCH  (default 8) iterations per batch (per body of the device-side loop: QCD_OPT_CG_DEFER
 *                     iterations); the host reads the device's convergence flag
 *                     once per batch, one batch late, so up to 2 batches of early-exit kernels follow
 *                     convergence.  1 <= value <= 1024.
 *   QCD_OPT_CG_DEFER  (default 8) deferred shift updates.  Inside the iteration only p_0 of the base system
 *                     is needed (the next M^dag M acts on it); x_k and p_k of the shifts k >= 1 are
 *                     needed at the end.  With value m > 1 the per-iteration update touches the base
 *                     shift only, the last m residuals are kept in a ring, and every m iterations ONE
 *                     pass applies the m stored updates to x_k, p_k of all other shifts: those vectors
 *                     move once per m iterations instead of once per iteration (96 V/m bytes per shift
 *                     and iteration instead of 96 V).  Every element sees the same operations in the
 *                     same order: results are bit-identical to value 1 (update every iteration).
 *                     1 <= value <= 8.  The y-only form defers in the same way (y and the p_k of the shifts
 *                     k >= 1 once per m iterations; y then agrees with value 1 to rounding, the sum being
 *                     taken in another order).  Not used by single-shift solves.
 *   QCD_OPT_CG_FUSE   (default 1) 1: the r-update and the base-shift update of an iteration run as ONE cooperative
 *                     kernel with a grid-wide barrier between them (needs QCD_OPT_CG_DEFER > 1, not used
 *                     by QCD_OPT_CG_GRAPH = 2); 0: two kernels, the second
 *                     waiting for the first's last block.  Bit-identical results.
 *   QCD_OPT_TGROUP    (default 0 = chosen by the library) order in which the Dslash CTAs walk the
 *                     lattice: groups of this many 128-site chunks of a t-slice are processed for all t
 *                     before the next group starts, so +-t neighbours are reused out of L2.  Dslash and
 *                     M^dag M stay bit-identical; CG results change at rounding level only (the
 *                     <p,Ap> partial sums are added in CTA order).  Values above the chunks per slice
 *                     mean plain lexicographic order.
 *   QCD_OPT_L2_PERSIST_MB (default 0 = off) applies at the NEXT qcd_load_gauge: Dslash launches carry
 *                     an L2 access-policy window that keeps this many MB of the gauge field in the
 *                     persisting set-aside of L2 (capped by the device limits; the limit is device-
 *                     wide).  Helps back-to-back applies on lattices slightly larger than L2, hurts the
 *                     CG when the set-aside takes L2 away from its vectors.  Bit-identical results.
 *   QCD_OPT_Y_ONLY    (default 0) qcd_inv_sqrt and qcd_apply_pow need only y = c0 phi + sum c_k x_k, so with
 *                     1 the shifted solutions x_k are never formed: the iteration accumulates
 *                     y += c_k alpha_k p_k directly, which halves the traffic of the per-shift update
 *                     and skips the residual pass.  y agrees with the default path to rounding.
 *                     true_res[] then holds the recursion's ESTIMATES |zeta_k| sqrt(rho)/||b|| (the
 *                     freezing threshold 0.1 tol for shifts frozen early), not recomputed residuals.
 *                     qcd_multishift_cg is not affected.
 *   QCD_OPT_LINK_ROWS (default 3) how the NEXT qcd_load_gauge stores the links.  3: all nine entries
 *                     (576 V bytes, "72V double precision words").  2: two-row storage
 *                     (384 V bytes): "one often stores and moves only two rows ... of the (3 x 3)
 *                     complex link matrix and recovers the third by orthogonalization";
 *                     the stencil rebuilds row_2 = conj(row_0 x row_1) in registers.  REQUIRES links in
 *                     SU(3) (unitary, det = 1): qcd_load_gauge then checks every third row against
 *                     conj(row_0 x row_1) (tolerance 1e-10 per component), SYNCHRONISES to read the
 *                     verdict and returns QCD_EINVAL (no field loaded) if a link fails.  Results differ
 *                     from the 3-row path at rounding level only (relative 1e-15).
 *   QCD_OPT_DSLASH_KERNEL  which Dslash kernel every entry point uses.  0: links loaded straight into
 *                     registers (thread per site, LDG.128).  1: links staged through shared memory by
 *                     the bulk-copy engine (cp.async.bulk behind an mbarrier ring, a producer warp per
 *                     CTA).  Bit-identical results.
 *   QCD_OPT_DSLASH_PERSIST (default 0) with kernel 1: 0 launches one CTA per 128-site tile; n > 0
 *                     launches a persistent grid of n CTAs per SM that walk the tiles round-robin.
 *                     Dslash and M^dag M stay bit-identical; CG results change at rounding level only
 *                     (the <p,Ap> partial sums are added per CTA).
 *   QCD_OPT_SWEEP_ALTERNATE  (default 1) 1: Dslash launches whose OUTPUT parity is even walk the lattice in
 *                     descending order, the others in ascending order, and the last
 *                     QCD_OPT_SWEEP_KEEP_MB of link data of every sweep are left in L2 with the ordinary
 *                     priority while the rest streams (evict-first).  D_oe and D_eo read the same links,
 *                     and inside M^dag M and the CG they alternate, so every apply starts on the links
 *                     its predecessor touched last.  0: one direction, all links streaming (the better
 *                     setting for an isolated apply behind a cold L2).  Dslash and M^dag M stay
 *                     bit-identical.
 *   QCD_OPT_SWEEP_KEEP_MB (default 48) see above; 0 <= value <= 4096.
 *   QCD_OPT_MIXED     (default 0) SURVEY 8(f) NEXT-3, the mixed-precision variant the paper sets aside
 *                     (PAPER.md:168).  With 1, the NEXT qcd_load_gauge also stores an fp32 copy of the
 *                     three-row links (+288 V bytes), and qcd_multishift_cg becomes: (1) the fp64
 *                     multishift CG down to 10^-QCD_OPT_MIXED_SWITCH_EXP only; (2) every shift on its
 *                     own by defect correction -- residual with the fp64 operator, inner single-shift CG
 *                     on the fp32-link operator (fp64 arithmetic and vectors, half the link bytes),
 *                     x_k += e -- until the recomputed fp64 residual is <= tol.  Same results within
 *                     the same tolerances; `iterations` counts stage 1 plus all inner iterations.
 *                     qcd_inv_sqrt / qcd_apply_pow keep the fp64 solver.
 *   QCD_OPT_MIXED_SWITCH_EXP (default 5) the loose tolerance of stage 1 is 10^-value, 1 <= value <= 15.
 *   QCD_OPT_OPERATOR_LINKS32 (default 0) with 1, qcd_dslash and qcd_mdagm apply the operator built on
 *                     the fp32 copy of the links (QCD_ESTATE unless the field was loaded with
 *                     QCD_OPT_MIXED = 1): the inner operator of the mixed solver on its own.
 * Returns QCD_EINVAL for an unknown option or a value out of range. */
enum { QCD_OPT_PDL = 0, QCD_OPT_CG_GRAPH = 1, QCD_OPT_CG_BATCH = 2, QCD_OPT_LINK_ROWS = 3, QCD_OPT_TGROUP = 4,
       QCD_OPT_L2_PERSIST_MB = 5, QCD_OPT_Y_ONLY = 6, QCD_OPT_DSLASH_KERNEL = 7, QCD_OPT_DSLASH_PERSIST = 8,
       QCD_OPT_MIXED = 9, QCD_OPT_MIXED_SWITCH_EXP = 10, QCD_OPT_OPERATOR_LINKS32 = 11,
       QCD_OPT_SWEEP_ALTERNATE = 12, QCD_OPT_CG_DEFER = 13, QCD_OPT_SWEEP_KEEP_MB = 14, QCD_OPT_CG_FUSE = 15 };
QCD_API qcd_status qcd_set_option(qcd_ctx *ctx, int option, long value);

/* Size in doubles of one internal parity vector: 6 * V/2. */
QCD_API long qcd_vector_doubles(const qcd_ctx *ctx);

/* a1: ingest the gauge field.  d_links_canonical: 72*V doubles, canonical layout.
 * Builds the library's parity-split site-fastest copy with 1/2, eta_mu(x) and the antiperiodic
 * sign folded into the stored links ("certain phases have been absorbed into the U's",
 * PAPER.md:104).  The caller's buffer is not retained. */
QCD_API qcd_status qcd_load_gauge(qcd_ctx *ctx, const double *d_links_canonical);
QCD_API qcd_status qcd_load_gauge_host(qcd_ctx *ctx, const double *h_links_canonical);

/* Canonical one-parity vector (6*V/2 doubles) <-> internal vector.  in/out must not alias. */
QCD_API qcd_status qcd_pack(qcd_ctx *ctx, int parity, const double *d_canonical, double *d_internal);
QCD_API qcd_status qcd_unpack(qcd_ctx *ctx, int parity, const double *d_internal, double *d_canonical);

/* a2/a3: d_out[out_parity] = D_{out_parity, other} d_in[other]  (C6):
 * out_parity = QCD_ODD is D_oe (even in, odd out), QCD_EVEN is D_eo.  Internal layout; d_in and
 * d_out must not alias. */
QCD_API qcd_status qcd_dslash(qcd_ctx *ctx, int out_parity, const double *d_in, double *d_out);

/* The same stencil restricted to the t-slices t0 <= t < t0 + nt of the output (all other sites of d_out are
 * left untouched), optionally fused with d_out = coeff * d_src - (D d_in) (d_src on out_parity, may be NULL).
 * This is the building block of a t-slab decomposition (PAPER.md:146-148 slices along z; SURVEY 8(f)
 * NEXT-4): a rank holds its slab plus one halo slice on either side as a lattice of its own and computes
 * the interior slices only (paper_1710_09178_b200/slab.py).  QCD_EINVAL unless 0 <= t0, nt >= 1,
 * t0 + nt <= Nt.  Does not synchronise. */
QCD_API qcd_status qcd_dslash_range(qcd_ctx *ctx, int out_parity, const double *d_in, double *d_out,
                                    int t0, int nt, const double *d_src, double coeff);

/* Slab (distributed) mode, SURVEY 8(f) NEXT-4 (slabs with halos, a face
 * exchange before every D, two reduced scalars per CG iteration).  With enable != 0 the context's lattice
 * is ONE RANK'S t-slab held with one halo slice on either side (extents Nx, Ny, Nz, nt_owned + 2; see
 * paper_1710_09178_b200/slab.py for the index maps, the parity flip and the seam carried by the links).
 * From then on
 *   qcd_dslash, qcd_mdagm      call halo(user, d_in, stream) first -- the caller fills the two halo t-slices
 *                              of that internal vector, WHICH IS THEREFORE WRITTEN -- and compute the owned
 *                              slices 1 .. Nt-2 only; the halo slices of the output are left untouched;
 *   qcd_multishift_cg          additionally calls allreduce(user, d_buf, count, stream) wherever an inner
 *                              product leaves the rank (||b||^2, <p_0,q> and ||r||^2 once per iteration,
 *                              the residual norms at the end): an in-place SUM over the ranks of `count`
 *                              doubles in DEVICE memory.  The halo slices of d_b are ignored (taken as
 *                              zero); those of d_x and d_y hold no result.  Every rank
 *                              runs the same iteration on replicated scalars, so all ranks make the same
 *                              calls in the same order.  No CUDA graphs, no PDL in this mode.
 * Both callbacks must be ordered on `stream` (they may synchronise it).  QCD_OPT_MIXED and the y-only form
 * are not available in slab mode.  halo, allreduce: see the typedefs. */
typedef void (*qcd_halo_fn)(void *user, double *d_vec, void *cuda_stream);
typedef void (*qcd_allreduce_fn)(void *user, double *d_buf, int count, void *cuda_stream);
QCD_API qcd_status qcd_set_slab(qcd_ctx *ctx, int enable, qcd_halo_fn halo, qcd_allreduce_fn allreduce, void *user);

/* a4: d_out = m^2 d_in - D_{p,q} D_{q,p} d_in on `parity` p  (C3).
 * Internal layout; d_in and d_out must not alias. */
QCD_API qcd_status qcd_mdagm(qcd_ctx *ctx, int parity, const double *d_in, double *d_out);

/* a5/a6: multishift CG (refs [5],[6]; recurrences SURVEY 8(c.2)).  Solves
 * (M^dag M + shifts[k]) x_k = d_b on `parity` for k < nshift, x_k = 0 initial guess (C11), until the
 * base (smallest-shift) system's recursion residual satisfies ||r|| <= tol ||b|| (C10); converged
 * shifts are frozen at 0.1 tol (C13).  Shifts need not be sorted (C12).
 *   d_b        internal vector (source)
 *   shifts     host, nshift values >= 0;   residues: host, nshift values (c_k of eq. 8)
 *   d_x        nshift internal vectors, contiguous, caller's shift order; may be NULL
 *   d_y        internal vector, y = sum_k residues[k] x_k (eq. 8 without c_0, C14); may be NULL
 *              d_b, d_x and d_y must not overlap one another (QCD_EINVAL)
 *   iterations host int;  true_res: host, nshift doubles, ||b - (M^dag M + sigma_k) x_k|| / ||b||
 *              recomputed from x_k (not the recursion value).
 * Returns QCD_OK, or QCD_ENOTCONV if max_iter iterations did not reach tol. Synchronises. */
QCD_API qcd_status qcd_multishift_cg(qcd_ctx *ctx, int parity, const double *d_b, int nshift,
                             const double *shifts, const double *residues, double tol,
                             int max_iter, double *d_x, double *d_y, int *iterations,
                             double *true_res);

/* the paper's "step 2", (M^dag M)^(-1/2) phi, through the rational
 * approximation of eq. 8:  x^(-1/2) ~= c_0 + sum_{k<n} c_k / (x + d_k).
 *
 * qcd_inv_sqrt_coeffs: HOST ONLY, needs no context and no GPU.  Writes the minimax (relative error)
 * approximation of type (n, n) on [xmin, xmax] -- what the paper takes from Mathematica's MiniMax
 * (appendix :288-304), computed here from Zolotarev's closed form in double precision:
 *   c0       host, 1 double;   coef, shift: host, n doubles each (c_k > 0; d_k > 0, ascending)
 *   delta    host, may be NULL: max over [xmin, xmax] of |1 - sqrt(x) r(x)| (formed in double
 *            precision from two function values: not resolved below ~1e-15)
 * The caller chooses xmin < lambda_min(M^dag M) (>= m^2 in this normalisation) and
 * xmax > lambda_max (m^2 + 4 for unit links, about 7 for random SU(3), never above m^2 + 16; the
 * paper keeps xmax = 34 in its normalisation, which is 8.5 here).  QCD_EINVAL unless
 * 1 <= n <= QCD_MAX_SHIFTS and 0 < xmin < xmax; QCD_ENOTCONV if a coefficient is not finite.
 *
 * qcd_inv_sqrt: d_out = c_0 d_phi + sum_k c_k (M^dag M + d_k)^(-1) d_phi on `parity` with those
 * coefficients, by ONE multishift CG (n shifts) and a fused combine.  Arguments as
 * qcd_multishift_cg; true_res has n entries (shift order ascending); d_out must not alias d_phi.
 * The result differs from (M^dag M)^(-1/2) phi by at most delta (approximation) + O(tol) (solver)
 * in relative 2-norm, provided the spectrum lies in [xmin, xmax].  Synchronises. */
QCD_API qcd_status qcd_inv_sqrt_coeffs(int n, double xmin, double xmax, double *c0, double *coef,
                                       double *shift, double *delta);
QCD_API qcd_status qcd_inv_sqrt(qcd_ctx *ctx, int parity, const double *d_phi, int n, double xmin,
                                double xmax, double tol, int max_iter, double *d_out,
                                int *iterations, double *true_res, double *delta);

/* The general exponent of eq. 8, (M^dag M)^(1/b): alpha = num/den with
 * 0 < |alpha| < 1, in particular the heat-bath power alpha = 1/4 (b = 4, appendix :288-304).
 *
 * qcd_pow_coeffs: HOST ONLY.  Minimax (relative error, type (n, n)) approximation
 *   x^alpha ~= c0 + sum_{k<n} coef[k] / (x + shift[k])  on [xmin, xmax]; shift ascending and > 0; coef < 0
 * for alpha > 0, > 0 for alpha < 0.  alpha = -1/2 is the closed form of qcd_inv_sqrt_coeffs; any other
 * exponent runs a Remez exchange iteration in binary128 arithmetic started from that closed form
 * (about 0.1-1 s).  delta (may be NULL): max |r(x)/x^alpha - 1|.  QCD_EINVAL for bad arguments,
 * QCD_ENOTCONV if the iteration does not converge (n too large for the interval: delta would be
 * below ~1e-15).
 *
 * qcd_apply_pow: d_out = c0 d_phi + sum_k coef[k] (M^dag M + shift[k])^(-1) d_phi, as qcd_inv_sqrt. */
QCD_API qcd_status qcd_pow_coeffs(int num, int den, int n, double xmin, double xmax, double *c0,
                                  double *coef, double *shift, double *delta);
QCD_API qcd_status qcd_apply_pow(qcd_ctx *ctx, int parity, const double *d_phi, int num, int den, int n,
                                 double xmin, double xmax, double tol, int max_iter, double *d_out,
                                 int *iterations, double *true_res, double *delta);

/* Host-buffer forms (canonical layout on the host; H2D copy, pack, compute, unpack, D2H copy and a
 * stream synchronise all happen inside the call).  h_x: nshift canonical parity vectors or NULL;
 * h_y: one canonical parity vector or NULL. */
QCD_API qcd_status qcd_dslash_host(qcd_ctx *ctx, int out_parity, const double *h_in, double *h_out);
QCD_API qcd_status qcd_mdagm_host(qcd_ctx *ctx, int parity, const double *h_in, double *h_out);
QCD_API qcd_status qcd_multishift_cg_host(qcd_ctx *ctx, int parity, const double *h_b, int nshift,
                                  const double *shifts, const double *residues, double tol,
                                  int max_iter, double *h_x, double *h_y, int *iterations,
                                  double *true_res);

/* Number of kernels this context has launched so far (for bench.py's gpu_launches claim). */
QCD_API long qcd_launch_count(const qcd_ctx *ctx);

/* Text of the last error on ctx (ctx == NULL: of the last failed qcd_create). Never NULL. */
QCD_API const char *qcd_last_error(const qcd_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* QCD_H */
