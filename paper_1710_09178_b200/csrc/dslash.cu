// dslash.cu -- a2/a3/a4 of SURVEY 8(a): the even-odd staggered Dirac operator
//   out(x) = sum_mu [ W_mu(x) in(x+mu) - W_mu(x-mu)^dag in(x-mu) ],  x of parity out_parity
// (PAPER.md:106 with 1/2, eta and the t-seam sign folded into W, see layout.cu), optionally fused
// with out = coeff*src - (.) (the m^2 term of M^dag M) and with the partial sums of
// Re<src,out> whose last block runs the CG alpha/zeta step.
//
// HBM-bound stencil: 8 links (1152 B) + 48 B out per site, neighbour vectors mostly from L2/L1;
// 570 flop / 1248 B = 0.46 flop/B, so no tensor cores (BASELINE.json north_star).  One thread per
// output site, site-fastest planes: every load/store of a warp is a contiguous run of 16-byte
// elements (LDG.128/STG.128).
#include "cg_scalars.cuh"
#include "reduce.cuh"

namespace qcd {

namespace {

#ifndef QCD_DSLASH_BLOCK
#define QCD_DSLASH_BLOCK 128
#endif
constexpr int kBlock = QCD_DSLASH_BLOCK;
#ifndef QCD_DSLASH3_MINB
#define QCD_DSLASH3_MINB 4   // 128 registers: 24.4 / 120.5 / 393 us; unbounded (60 regs) 26.0 / 129 / 404; 1 (254 regs) 25.7 / 120.2 / 394
#endif
// minimum resident CTAs per SM asked of ptxas for the two-row kernel (caps its registers)
#ifndef QCD_DSLASH2_MINB
#define QCD_DSLASH2_MINB 4   // measured on B200 (32^3x8 / 48^3x12 / 64^3x16): 4 -> 16.8 / 83.4 / 274 us; 7 -> 17.1 / 88.6 / 276; 1 -> 18.9 / - / 296
#endif

// acc += w * v
__device__ __forceinline__ void cmad(double2 &acc, const double2 w, const double2 v)
{
    acc.x = fma(w.x, v.x, acc.x);
    acc.x = fma(-w.y, v.y, acc.x);
    acc.y = fma(w.x, v.y, acc.y);
    acc.y = fma(w.y, v.x, acc.y);
}
// acc -= conj(w) * v
__device__ __forceinline__ void cmsub_conj(double2 &acc, const double2 w, const double2 v)
{
    acc.x = fma(-w.x, v.x, acc.x);
    acc.x = fma(-w.y, v.y, acc.x);
    acc.y = fma(-w.x, v.y, acc.y);
    acc.y = fma(w.y, v.x, acc.y);
}

// x -> -x when neg (sign-bit flip on the integer pipe; the fp64 pipe stays free for the stencil)
__device__ __forceinline__ double flip(double x, int neg)
{
    return __hiloint2double(__double2hiint(x) ^ (neg << 31), __double2loint(x));
}

// Two-row storage ("stores and moves only two rows ... recovers the
// third by orthogonalization"): for U in SU(3), row_2 = conj(row_0 x row_1).  u[0..5] hold rows 0, 1.
__device__ __forceinline__ void third_row(double2 *u)
{
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int c1 = (c + 1) % 3, c2 = (c + 2) % 3;
        const double2 a1 = u[c1], a2 = u[c2], b1 = u[3 + c1], b2 = u[3 + c2];
        double tx = a1.x * b2.x;
        tx = fma(-a1.y, b2.y, tx);
        tx = fma(-a2.x, b1.x, tx);
        tx = fma(a2.y, b1.y, tx);
        double ty = a1.x * b2.y;
        ty = fma(a1.y, b2.x, ty);
        ty = fma(-a2.x, b1.y, ty);
        ty = fma(-a2.y, b1.x, ty);
        u[6 + c] = make_double2(tx, -ty);
    }
}

// ROWS == 3: W holds 1/2 eta s+ U (all nine entries, signs folded in at ingest).
// ROWS == 2: W holds rows 0 and 1 of the plain U; eta_mu(x), the t-seam sign and the 1/2 are applied
//            here.  All of them depend on the OUTPUT site only: eta_mu does not depend on x_mu, and
//            the seam sign of the backward hop is s-_mu(x).
template <bool XPAY, bool DOT, int ROWS>
__global__ void __launch_bounds__(kBlock, ROWS == 2 ? QCD_DSLASH2_MINB : QCD_DSLASH3_MINB)
dslash_kernel(const Geom g, const DslashParams p)
{
    constexpr int NW = 3 * ROWS;
    const int Vh = g.Vh;
    // CTA order.  A chunk is kBlock consecutive sites of one t-slice.  The chunks of a slice are cut
    // into groups of g.tgroup; CTAs walk group by group, and inside a group t runs slowest:
    //     blockIdx = (group * Nt + t) * tgroup + chunk_in_group        (last group may be shorter)
    // so the CTAs that read the same input sites as +-t neighbours are tgroup CTAs apart instead of a
    // whole t-slice of CTAs (1024 CTAs = 163 MB of link traffic at 64^3x16, more than L2 holds: ncu
    // showed 2.7-2.8 GB of DRAM reads per apply against 2.52 GB algorithmic), while each group still
    // streams tgroup * 2 KB contiguous bytes of every link plane.  tgroup == chunks: plain h order.
    const uint32_t per_group = (uint32_t)g.tgroup * (uint32_t)g.Nt;
    const uint32_t grp = blockIdx.x / per_group, rem = blockIdx.x - grp * per_group;
    const uint32_t first = grp * (uint32_t)g.tgroup;
    const uint32_t width = min((uint32_t)g.tgroup, (uint32_t)g.chunks - first);   // chunks in this group
    const uint32_t t = rem / width;
    const uint32_t chunk = first + (rem - t * width);
    const uint32_t sl = chunk * kBlock + threadIdx.x;          // index inside the t-slice
    const bool valid = sl < (uint32_t)g.st;
    const uint32_t h = t * (uint32_t)g.st + sl;
    double dot = 0.0;
    const int par = p.out_parity;
    int hp[4], hm[4];   // half indices of the 8 neighbours (all of the opposite parity)
    int nf[4] = {0, 0, 0, 0}, nb[4] = {0, 0, 0, 0};   // ROWS == 2: 1 where the hop carries a minus sign
    if (valid) {
        uint32_t q, xh, y, z;
        g.dxh.divmod(sl, q, xh);
        g.dy.divmod(q, z, y);
        const int r = (y + z + t + par) & 1;      // x = 2*xh + r
        {
            const int xh_p = r ? ((int)xh + 1 == g.Nxh ? 0 : (int)xh + 1) : (int)xh;
            const int xh_m = r ? (int)xh : (xh == 0 ? g.Nxh - 1 : (int)xh - 1);
            hp[0] = (int)h - (int)xh + xh_p;
            hm[0] = (int)h - (int)xh + xh_m;
            hp[1] = (int)h + ((int)y + 1 == g.Ny ? -(g.Ny - 1) * g.sy : g.sy);
            hm[1] = (int)h + (y == 0 ? (g.Ny - 1) * g.sy : -g.sy);
            hp[2] = (int)h + ((int)z + 1 == g.Nz ? -(g.Nz - 1) * g.sz : g.sz);
            hm[2] = (int)h + (z == 0 ? (g.Nz - 1) * g.sz : -g.sz);
            hp[3] = (int)h + ((int)t + 1 == g.Nt ? -(g.Nt - 1) * g.st : g.st);
            hm[3] = (int)h + (t == 0 ? (g.Nt - 1) * g.st : -g.st);
        }
        if (ROWS == 2) {
            const int x = 2 * (int)xh + r;
            nf[1] = nb[1] = x & 1;                       // eta_1 = (-1)^x
            nf[2] = nb[2] = (x + (int)y) & 1;            // eta_2 = (-1)^(x+y)
            const int e3 = (x + (int)y + (int)z) & 1;    // eta_3 = (-1)^(x+y+z)
            nf[3] = e3 ^ ((int)t + 1 == g.Nt);           // s+ on the hop t = Nt-1 -> 0  (C5)
            nb[3] = e3 ^ (t == 0);                       // s- on the hop t = 0 -> Nt-1
        }
    }
    // everything above is index arithmetic; from here on data of the preceding kernel is read
    pdl_wait();
    pdl_launch_dependents();
    if (p.st != nullptr && p.st->done) return;   // CG already converged: dead iteration
    if (valid) {
        const double2 *__restrict__ in = p.in;
        double2 acc[3];
        acc[0] = acc[1] = acc[2] = make_double2(0.0, 0.0);
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) {
            {   // forward hop: + W_mu(x) in(x+mu), link based at x (parity par)
                const double2 *__restrict__ w = p.W + ((long)(par * 4 + mu) * NW) * Vh + h;
                double2 u[9], v[3];
#pragma unroll
                for (int i = 0; i < NW; ++i) u[i] = __ldg(w + (long)i * Vh);
#pragma unroll
                for (int c = 0; c < 3; ++c) v[c] = __ldg(in + (long)c * Vh + hp[mu]);
                if (ROWS == 2) {
                    third_row(u);
#pragma unroll
                    for (int c = 0; c < 3; ++c) v[c] = make_double2(flip(v[c].x, nf[mu]), flip(v[c].y, nf[mu]));
                }
#pragma unroll
                for (int a = 0; a < 3; ++a)
#pragma unroll
                    for (int b = 0; b < 3; ++b) cmad(acc[a], u[a * 3 + b], v[b]);
            }
            {   // backward hop: - W_mu(x-mu)^dag in(x-mu), link based at x-mu (parity 1-par)
                const double2 *__restrict__ w = p.W + ((long)((1 - par) * 4 + mu) * NW) * Vh + hm[mu];
                double2 u[9], v[3];
#pragma unroll
                for (int i = 0; i < NW; ++i) u[i] = __ldg(w + (long)i * Vh);
#pragma unroll
                for (int c = 0; c < 3; ++c) v[c] = __ldg(in + (long)c * Vh + hm[mu]);
                if (ROWS == 2) {
                    third_row(u);
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
        double total;
        if (grid_sum_last_block<kBlock>(dot, p.partial, &p.st->counter, total))
            cg_step_alpha(p.st, total);
    }
}

}  // namespace

int dslash_chunks(const Geom &g) { return (g.st + kBlock - 1) / kBlock; }
int dslash_grid_blocks(const Geom &g) { return dslash_chunks(g) * g.Nt; }

int launch_dslash(const Geom &g, const DslashParams &p, Launch L)
{
    const int blocks = dslash_grid_blocks(g);
    if (p.link_rows == 2) {
        if (p.src == nullptr)
            launch_kernel_apw(dslash_kernel<false, false, 2>, blocks, kBlock, L.s, L.pdl, L.apw, g, p);
        else if (p.dot_mode == 0)
            launch_kernel_apw(dslash_kernel<true, false, 2>, blocks, kBlock, L.s, L.pdl, L.apw, g, p);
        else
            launch_kernel_apw(dslash_kernel<true, true, 2>, blocks, kBlock, L.s, L.pdl, L.apw, g, p);
    } else {
        if (p.src == nullptr)
            launch_kernel_apw(dslash_kernel<false, false, 3>, blocks, kBlock, L.s, L.pdl, L.apw, g, p);
        else if (p.dot_mode == 0)
            launch_kernel_apw(dslash_kernel<true, false, 3>, blocks, kBlock, L.s, L.pdl, L.apw, g, p);
        else
            launch_kernel_apw(dslash_kernel<true, true, 3>, blocks, kBlock, L.s, L.pdl, L.apw, g, p);
    }
    return 1;
}

}  // namespace qcd
