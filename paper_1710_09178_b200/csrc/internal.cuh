// internal.cuh -- shared declarations of the CUDA library (not part of the ABI).
//
// Internal HBM layout:
//   parity vector  double2 v[3][Vh]               colour-major planes, site-fastest ("ap(V,3)")
//   links          double2 W[2][4][9][Vh]         [parity of the link's base site][mu][row*3+col][h]
//                  W_mu(x) = 1/2 eta_mu(x) s+_mu(x) U_mu(x)   (phases absorbed)
//   links, 2-row   double2 W[2][4][6][Vh]         rows 0 and 1 of the plain U_mu(x);
//                  the third row, eta, the seam sign and the 1/2 are applied inside the stencil
//   half index     h = ((t*Nz + z)*Ny + y)*(Nx/2) + x/2   == canonical address l >> 1
// so that (D psi)(x) = sum_mu [ W_mu(x) psi(x+mu) - W_mu(x-mu)^dag psi(x-mu) ].
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/qcd.h"

namespace qcd {

constexpr int kMaxShifts = QCD_MAX_SHIFTS;
constexpr int kMaxDefer = 8;   // iterations whose updates of the shifts k >= 1 can be applied in one pass (blas.cu)

// n / d for 0 <= n < 2^31 with one mulhi (d fixed at context creation).
struct FastDiv {
    uint32_t d, magic, shift;
    __host__ void init(uint32_t div)
    {
        d = div;
        shift = 0;
        while ((1u << shift) < div) ++shift;
        magic = (uint32_t)(((uint64_t(1) << 32) * ((uint64_t(1) << shift) - div)) / div + 1);
    }
    __device__ __forceinline__ void divmod(uint32_t n, uint32_t &q, uint32_t &r) const
    {
        q = (__umulhi(n, magic) + n) >> shift;
        r = n - q * d;
    }
};

struct Geom {
    int Nx, Ny, Nz, Nt, Nxh;
    int Vh;          // sites of one parity
    int sy, sz, st;  // half-index strides of +y, +z, +t
    FastDiv dxh, dy, dz;
    int t0, nt_run;  // t-slices t0 <= t < t0 + nt_run are computed by a Dslash launch (default: all)
    int chunks;      // Dslash CTAs per t-slice
    int tgroup;      // chunks per group of the Dslash CTA order (dslash.cu), 1 <= tgroup <= chunks
};

// Device-resident scalars of the multishift CG; no host round trip per iteration.
struct CgState {
    double rho, rho_b, pAp, alpha, beta, alpha_old, beta_old;
    double tol, freeze, sigma0;
    double sigma[kMaxShifts];     // sorted ascending, sigma[0] = base
    double zeta[kMaxShifts], zeta_old[kMaxShifts], zeta_new[kMaxShifts];
    double coef_a[kMaxShifts], coef_z[kMaxShifts], coef_b[kMaxShifts];  // x_k += a p_k ; p_k = z r + b p_k
    long long xoff[kMaxShifts];   // element (double2) offset of x_k in the x buffer
    int list[kMaxShifts];         // compacted indices of the shifts updated this iteration
    int nlist;
    int active[kMaxShifts];
    int nshift, iter, max_iter;
    int done;                     // set by the r-update of the converging iteration
    int done_prev;                // set one (dead) iteration later: gates the shift update
    unsigned counter;             // last-block-done ticket
    double scratch;               // generic reduction result (norms for true residuals)
    double red[2];                // slab mode: <p_0,q> and ||r'||^2, summed over the rank, then over the ranks
    int not_su3;                  // set by the two-row gauge ingest (layout.cu)
    double cy[kMaxShifts];        // y-only mode: residues c_k of eq. 8 in sorted-shift order
    // deferred shift updates (blas.cu): the coefficients of the last `defer` iterations, slot (n - 1) % defer
    // for iteration n = 1, 2, ..., written by the last block of that iteration's r-update
    int defer;                    // 1 <= defer <= kMaxDefer; also the number of slots of the residual ring
    int enq;                      // iterations enqueued so far, dead ones included (r-update, CTA 0)
    double hist_a[kMaxDefer][kMaxShifts], hist_z[kMaxDefer][kMaxShifts], hist_b[kMaxDefer][kMaxShifts];
    int hist_on[kMaxDefer][kMaxShifts];   // shift k took part in the iteration of this slot
};

// ---- programmatic dependent launch (PDL) ----
// Every kernel of the library is launched with cudaLaunchAttributeProgrammaticStreamSerialization
// (unless switched off by QCD_OPT_PDL): it may become resident while its predecessor in the stream
// (or graph) is still draining, runs its index arithmetic, and blocks in pdl_wait() until the
// predecessor has completed and its writes are visible.  Rules kept by every kernel: nothing written
// and nothing produced by an earlier kernel read before pdl_wait(); pdl_launch_dependents() only
// after pdl_wait(), so completion is transitive along the chain.  One deliberate use of the window:
// the Dslash requests its first two link matrices BEFORE pdl_wait() -- the gauge field is constant
// between qcd_load_gauge calls, and the first Dslash after a load is launched without PDL (api.cu).
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents()
{
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}

// apw != nullptr: the launch carries an L2 access-policy window (persisting lines for part of the
// gauge field, see api.cu); as a launch attribute it is recorded in captured graph nodes too.
template <class... KArgs, class... Args>
inline cudaError_t launch_kernel_apw(void (*kernel)(KArgs...), int grid, int block, cudaStream_t s,
                                     bool pdl, const cudaAccessPolicyWindow *apw, Args... args)
{
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3((unsigned)block);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = s;
    cudaLaunchAttribute attr[2];
    unsigned n = 0;
    if (pdl) {
        attr[n].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[n].val.programmaticStreamSerializationAllowed = 1;
        ++n;
    }
    if (apw != nullptr) {
        attr[n].id = cudaLaunchAttributeAccessPolicyWindow;
        attr[n].val.accessPolicyWindow = *apw;
        ++n;
    }
    cfg.attrs = attr;
    cfg.numAttrs = n;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

template <class... KArgs, class... Args>
inline cudaError_t launch_kernel(void (*kernel)(KArgs...), int grid, int block, cudaStream_t s,
                                 bool pdl, Args... args)
{
    return launch_kernel_apw(kernel, grid, block, s, pdl, nullptr, args...);
}
#endif

// ---- launchers (each enqueues on `s` and returns the number of kernels launched) ----
struct Launch {
    cudaStream_t s;
    bool pdl;
    const cudaAccessPolicyWindow *apw = nullptr;   // only the Dslash launches use it
};

// not_su3 (device int, zeroed by the caller): set to 1 by the two-row ingest when a link is not in SU(3)
int launch_ingest_links(const Geom &g, const double *links_canon, double2 *W, int link_rows, int *not_su3,
                        Launch L);
// fp32 copy of the three-row internal links: W32[2][4][9][Vh] = (float) 1/2 eta s+ U  (NEXT-3)
int launch_ingest_links32(const Geom &g, const double *links_canon, float2 *W32, Launch L);
// out = b - q, *result = ||out||^2 (one ticketed reduction)
int launch_residual(long n2, const double2 *b, const double2 *q, double2 *out, double *partial, unsigned *counter,
                    double *result, int Vh, int halo, Launch L);   // halo as in launch_cg_init
// sites h0 <= h < h1 only (h1 < 0: all)
int launch_pack(const Geom &g, const double *canon, double2 *internal, Launch L, int h0 = 0, int h1 = -1);
int launch_unpack(const Geom &g, const double2 *internal, double *canon, Launch L, int h0 = 0, int h1 = -1);

struct DslashParams {
    const double2 *W;
    const float2 *W32;         // fp32 copy of the three-row links (same layout), used when links32 != 0
    int links32;
    int link_rows;             // 3: W[2][4][9][Vh] with signs folded in; 2: W[2][4][6][Vh] plain rows 0,1
    const double2 *in;
    double2 *out;
    int out_parity;
    int reverse;               // 1: the CTAs walk the tiles in descending order (QCD_OPT_SWEEP_ALTERNATE)
    int keep_tiles;            // tiles at the end of the sweep whose links stay in L2 with the ordinary priority
                               // (all others are loaded evict-first)
    // optional fused epilogue: out = coeff * src - D in     (src on out_parity); src == nullptr: out = D in
    const double2 *src;
    double coeff;              // used when coeff_from_state == 0
    int coeff_from_state;      // 1: coeff = mass2 + st->sigma0 read on device
    double mass2;
    // optional fused <src,out>: one partial sum per CTA in partial[blockIdx] (the CG's r-update adds them)
    int dot_mode;              // 0 none, 1 on
    double *partial;
    CgState *st;               // also the early-exit flag when non-null
};
int launch_dslash(const Geom &g, const DslashParams &p, Launch L);
// dslash_bulk.cu: the same operator with the links staged through shared memory by cp.async.bulk;
// ctas_per_sm > 0: persistent grid of that many CTAs per SM, 0: one CTA per 128-site tile
int launch_dslash_bulk(const Geom &g, const DslashParams &p, int ctas_per_sm, Launch L);
int dslash_bulk_grid_blocks(const Geom &g, int ctas_per_sm);
int dslash_grid_blocks(const Geom &g);
int dslash_chunks(const Geom &g);

// D applied to up to kMultiRhs vectors in one pass over the links (dslash_multi.cu).
//   b == nullptr:  out_j = D in_j
//   b != nullptr:  *result[j] = || b - (coeff[j] src_j - D in_j) ||^2, nothing stored
// vector j lives at base + off[j] (double2 elements).  partial must hold kMultiRhs * grid doubles.
constexpr int kMultiRhs = 4;
struct DslashMultiParams {
    const double2 *W;
    int link_rows, out_parity, nrhs;
    int reverse, keep_tiles;   // as in DslashParams
    const double2 *in;
    long long in_off[kMultiRhs];
    double2 *out;
    long long out_off[kMultiRhs];
    const double2 *src;
    long long src_off[kMultiRhs];
    double coeff[kMultiRhs];
    const double2 *b;
    double *partial;
    unsigned *counter;
    double *result[kMultiRhs];
};
int launch_dslash_multi(const Geom &g, const DslashMultiParams &p, Launch L);

// BLAS-1 (n2 = 3*Vh double2 elements per vector)
int blas_grid_blocks(long n2);
// halo > 0 (slab mode): the first and the last `halo` sites of every colour plane (Vh sites) are taken as zero
int launch_cg_init(long n2, const double2 *b, double2 *r, double2 *p, long pstride, int nshift,
                   double *partial, CgState *st, int Vh, int halo, Launch L);
// loop_handle != 0: the kernel is a node of a WHILE conditional graph and sets its condition
// The residual lives in a ring of st->defer vectors (stride n2): r after iteration n is slot (n - 1) % defer,
// the initial residual b is slot defer - 1.
// pap_partial[0 .. npap): the per-CTA partial sums of <p_0,q> the preceding Dslash wrote
int launch_cg_update_r(long n2, double2 *ring, const double2 *q, const double *pap_partial, int npap,
                       double *partial, CgState *st, unsigned long long loop_handle, Launch L);
// r-update and base-shift update in one cooperative kernel (QCD_OPT_CG_FUSE); returns 0 without launching if
// the grid cannot be co-resident
int launch_cg_update_r_base(long n2, double2 *ring, const double2 *q, const double *pap_partial, int npap,
                            double *partial, double2 *x, double2 *p, CgState *st, int y_only, Launch L);
// y-only form: y += sum_k c_k alpha_k p_k ; p_k = zeta_k r + beta_k p_k   (no x_k are kept)
int launch_cg_update_shifts_y(long n2, const double2 *ring, double2 *y, double2 *p, long pstride,
                              CgState *st, int base_only, Launch L);
int launch_cg_flush_shifts_y(long n2, const double2 *ring, double2 *y, double2 *p, long pstride,
                             const CgState *st, int window, Launch L);
// x_k += alpha_k p_k ; p_k = zeta_k r + beta_k p_k for the shifts of this iteration; base_only: shift 0 alone
int launch_cg_update_shifts(long n2, const double2 *ring, double2 *x, double2 *p, long pstride,
                            CgState *st, int base_only, Launch L);
// the deferred updates of the shifts k >= 1 for the last `window` enqueued iterations, in one pass
int launch_cg_flush_shifts(long n2, const double2 *ring, double2 *x, double2 *p, long pstride,
                           const CgState *st, int window, Launch L);
// ---- slab (distributed) mode: the reductions leave the rank between the kernels (api.cu) ----
// split != 0: the r-update's last block stores the rank's ||r'||^2 in st->red[1] and leaves the scalar step
// to launch_cg_scalars (after the all-reduce)
int launch_cg_update_r_split(long n2, double2 *ring, const double2 *q, const double *pap, double *partial,
                             CgState *st, Launch L);
int launch_sum_partials(const double *partial, int n, double *out, Launch L);   // *out = sum partial[0..n)
int launch_cg_scalars(CgState *st, Launch L);        // alpha_k/zeta, beta, freeze, stop from st->red[0..1]
int launch_cg_after_init(CgState *st, Launch L);     // rho_b = rho (all-reduced), done = (rho == 0)

// y = c0 b + sum_k residues[k] x_k  (b == nullptr: no c0 term)
int launch_combine(long n2, const double2 *x, const long long *xoff_host, const double *residues,
                   int nshift, double c0, const double2 *b, double2 *y, Launch L);

// y += c0 b in place (the c_0 term of eq. 8 on the y-only path)
int launch_add_c0(long n2, double c0, const double2 *b, double2 *y, Launch L);

// host only (zolotarev.cu): minimax x^(-1/2) ~= c0 + sum_k c[k]/(x + d[k]) on [xmin, xmax]; 0 = ok
int zolotarev_inv_sqrt(int n, double xmin, double xmax, double *c0, double *c, double *d, double *delta);
// host only (remez.cu): minimax x^(num/den) ~= c0 + sum_k c[k]/(x + d[k]); 0 ok, 1 bad arguments, 2 not converged
int remez_pow(int num, int den, int n, double xmin, double xmax, double *c0, double *c, double *d,
              double *delta);

}  // namespace qcd
