// dslash.cu -- a2/a3/a4 of SURVEY 8(a): the even-odd staggered Dirac operator
//   out(x) = sum_mu [ W_mu(x) in(x+mu) - W_mu(x-mu)^dag in(x-mu) ],  x of parity out_parity
// (PAPER.md:106 with 1/2, eta and the t-seam sign folded into W, see layout.cu), optionally fused
// with out = coeff*src - (.) (the m^2 term of M^dag M) and with per-CTA partial sums
// of Re<src,out>, from which the CG's r-update forms alpha.
//
// HBM-bound stencil: 8 links (1152 B) + 48 B out per site, neighbour vectors mostly from L2/L1;
// 570 flop / 1248 B = 0.46 flop/B, so no tensor cores (BASELINE.json north_star).  One thread per
// output site, site-fastest planes: every load/store of a warp is a contiguous run of 16-byte
// elements (LDG.128/STG.128).
#include "cg_scalars.cuh"
#include "dslash_site.cuh"
#include "reduce.cuh"

namespace qcd {

namespace {

constexpr int kBlock = kDslashBlock;
#ifndef QCD_DSLASH3_MINB
#define QCD_DSLASH3_MINB 4   // 128 registers: 24.4 / 120.5 / 393 us; unbounded (60 regs) 26.0 / 129 / 404; 1 (254 regs) 25.7 / 120.2 / 394
#endif
// link matrices requested before griddepcontrol.wait, in hop order +0, -0, +1, -1, ...
#ifndef QCD_DSLASH_PREFETCH
#define QCD_DSLASH_PREFETCH 2   // measured at 32^3x8: 0 -> 24.6 us, 1 -> 23.6, 2 -> 23.0, 3 (spills) -> 25.5
#endif
// minimum resident CTAs per SM asked of ptxas for the two-row kernel (caps its registers)
#ifndef QCD_DSLASH2_MINB
#define QCD_DSLASH2_MINB 4   // measured on B200 (32^3x8 / 48^3x12 / 64^3x16): 4 -> 16.8 / 83.4 / 274 us; 7 -> 17.1 / 88.6 / 276; 1 -> 18.9 / - / 296
#endif

// ROWS == 3: W holds 1/2 eta s+ U (all nine entries, signs folded in at ingest).
// ROWS == 2: W holds rows 0 and 1 of the plain U; eta_mu(x), the t-seam sign and the 1/2 are applied
//            here.  All of them depend on the OUTPUT site only: eta_mu does not depend on x_mu, and
//            the seam sign of the backward hop is s-_mu(x).
// WT = double2: the links as stored (p.W).  WT = float2: the fp32 copy p.W32 (NEXT-3, inner operator of
// the mixed-precision solver, three rows only); every entry is widened on load, the arithmetic is fp64.
template <bool XPAY, bool DOT, int ROWS, class WT = double2>
__global__ void __launch_bounds__(kBlock, ROWS == 2 ? QCD_DSLASH2_MINB : QCD_DSLASH3_MINB)
dslash_kernel(const Geom g, const DslashParams p)
{
    constexpr int NW = 3 * ROWS;
    const int Vh = g.Vh;
    const WT *__restrict__ const W = sizeof(WT) == sizeof(float2) ? reinterpret_cast<const WT *>(p.W32)
                                                                 : reinterpret_cast<const WT *>(p.W);
    Site site;
    locate_tile<ROWS == 2>(g, p.out_parity, p.reverse ? gridDim.x - 1 - blockIdx.x : blockIdx.x, threadIdx.x, site);
    // the last keep_tiles CTAs of the sweep leave their links in L2 with the ordinary priority (the next
    // apply, walking the other way, starts there); the others stream (evict-first): api.cu, decide_sweep
    const uint64_t pol = l2_policy(blockIdx.x + (unsigned)p.keep_tiles >= gridDim.x);
#define QCD_LOAD_LINK(w, u) load_link_hint<ROWS>(w, Vh, u, pol)
    const bool valid = site.valid;
    const uint32_t h = site.h;
    const int par = p.out_parity;
    const int *hp = site.hp, *hm = site.hm, *nf = site.nf, *nb = site.nb;
    double dot = 0.0;
    // The gauge links are constant between qcd_load_gauge calls (and the first Dslash after a load is
    // launched without PDL, api.cu), so the links of the first hops may be requested BEFORE waiting for
    // the preceding kernel: they stream in while that kernel drains.
    constexpr int NPF = QCD_DSLASH_PREFETCH;       // hops 0 .. NPF-1 in the order (+0, -0, +1, -1, ...)
    double2 pre[NPF > 0 ? NPF : 1][9];
    auto request_links = [&]() {
#pragma unroll
        for (int k = 0; k < NPF; ++k) {
            const int mu = k >> 1;
            if (k & 1) QCD_LOAD_LINK(W + ((long)((1 - par) * 4 + mu) * NW) * Vh + hm[mu], pre[k]);
            else QCD_LOAD_LINK(W + ((long)(par * 4 + mu) * NW) * Vh + h, pre[k]);
        }
    };
    // Inside the CG, `done` was last written two or more kernels back (r-update), which has completed
    // by the time this kernel may start: a dead iteration is recognised early and requests nothing.
    // (Only a hint: after a cg_init for a zero source it may still read 0; the check after the wait decides.)
    const bool early = valid && !(p.st != nullptr && *(volatile const int *)&p.st->done);
    if (early) request_links();
    // everything above is index arithmetic and constant data; from here on data of the preceding kernel is read
    pdl_wait();
    pdl_launch_dependents();
    if (p.st != nullptr && p.st->done) return;   // CG already converged: dead iteration
    if (valid && !early) request_links();
    if (valid) {
        const double2 *__restrict__ in = p.in;
        double2 acc[3];
        acc[0] = acc[1] = acc[2] = make_double2(0.0, 0.0);
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) {
            {   // forward hop: + W_mu(x) in(x+mu), link based at x (parity par)
                const WT *__restrict__ w = W + ((long)(par * 4 + mu) * NW) * Vh + h;
                double2 u[9], v[3];
                if (2 * mu < NPF) {
#pragma unroll
                    for (int i = 0; i < 9; ++i) u[i] = pre[2 * mu < NPF ? 2 * mu : 0][i];
                } else {
                    QCD_LOAD_LINK(w, u);
                }
#pragma unroll
                for (int c = 0; c < 3; ++c) v[c] = __ldg(in + (long)c * Vh + hp[mu]);
                if (ROWS == 2) {
#pragma unroll
                    for (int c = 0; c < 3; ++c) v[c] = make_double2(flip(v[c].x, nf[mu]), flip(v[c].y, nf[mu]));
                }
#pragma unroll
                for (int a = 0; a < 3; ++a)
#pragma unroll
                    for (int b = 0; b < 3; ++b) cmad(acc[a], u[a * 3 + b], v[b]);
            }
            {   // backward hop: - W_mu(x-mu)^dag in(x-mu), link based at x-mu (parity 1-par)
                const WT *__restrict__ w = W + ((long)((1 - par) * 4 + mu) * NW) * Vh + hm[mu];
                double2 u[9], v[3];
                if (2 * mu + 1 < NPF) {
#pragma unroll
                    for (int i = 0; i < 9; ++i) u[i] = pre[2 * mu + 1 < NPF ? 2 * mu + 1 : 0][i];
                } else {
                    QCD_LOAD_LINK(w, u);
                }
#pragma unroll
                for (int c = 0; c < 3; ++c) v[c] = __ldg(in + (long)c * Vh + hm[mu]);
                if (ROWS == 2) {
#pragma unroll
                    for (int c = 0; c < 3; ++c) v[c] = make_double2(flip(v[c].x, nb[mu]), flip(v[c].y, nb[mu]));
                }
#pragma unroll
                for (int a = 0; a < 3; ++a)
#pragma unroll
                    for (int b = 0; b < 3; ++b) cmsub_conj(acc[a], u[b * 3 + a], v[b]);
            }
        }
        if (ROWS == 2) {
#pragma unroll
            for (int c = 0; c < 3; ++c) acc[c] = make_double2(0.5 * acc[c].x, 0.5 * acc[c].y);
        }
        if (XPAY) {
            const double coeff = p.coeff_from_state ? p.mass2 + p.st->sigma0 : p.coeff;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double2 s = __ldg(p.src + (long)c * Vh + h);
                acc[c].x = fma(coeff, s.x, -acc[c].x);
                acc[c].y = fma(coeff, s.y, -acc[c].y);
                if (DOT) dot += s.x * acc[c].x + s.y * acc[c].y;
            }
        }
#pragma unroll
        for (int c = 0; c < 3; ++c) p.out[(long)c * Vh + h] = acc[c];
    }
    if (DOT) {
        // one partial sum per CTA; the r-update, which needs alpha, adds them up itself (blas.cu): no
        // ticket, no fence and no serial last-block pass at the end of the stencil
        const double b = block_sum<kBlock>(dot);
        if (threadIdx.x == 0) p.partial[blockIdx.x] = b;
    }
}

}  // namespace

int dslash_chunks(const Geom &g) { return (g.st + kBlock - 1) / kBlock; }
int dslash_grid_blocks(const Geom &g) { return dslash_chunks(g) * g.nt_run; }

namespace {

template <int ROWS, class WT>
void launch_variant(const Geom &g, const DslashParams &p, Launch L)
{
    const int blocks = dslash_grid_blocks(g);
    if (p.src == nullptr)
        launch_kernel_apw(dslash_kernel<false, false, ROWS, WT>, blocks, kBlock, L.s, L.pdl, L.apw, g, p);
    else if (p.dot_mode == 0)
        launch_kernel_apw(dslash_kernel<true, false, ROWS, WT>, blocks, kBlock, L.s, L.pdl, L.apw, g, p);
    else
        launch_kernel_apw(dslash_kernel<true, true, ROWS, WT>, blocks, kBlock, L.s, L.pdl, L.apw, g, p);
}

}  // namespace

int launch_dslash(const Geom &g, const DslashParams &p, Launch L)
{
    if (p.links32) launch_variant<3, float2>(g, p, L);
    else if (p.link_rows == 2) launch_variant<2, double2>(g, p, L);
    else launch_variant<3, double2>(g, p, L);
    return 1;
}

}  // namespace qcd
