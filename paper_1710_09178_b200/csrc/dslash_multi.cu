// dslash_multi.cu -- a6 of SURVEY 8(a): the true residuals ||b - (M^dag M + sigma_k) x_k|| of all
// shifts need one M^dag M apply per shift, and every apply would stream the whole gauge field again
// (92 % of a Dslash's bytes).  Here one launch applies D to up to kMultiRhs vectors at once: each
// link is loaded (and, with two-row storage, rebuilt) once per site and used for all of them, so a
// batch of 4 moves 576 V + 4 * 48 V bytes instead of 4 * 624 V.  The second launch of a batch does
// not store its result: it forms (m^2 + sigma_k) x_k - D tmp_k, subtracts it from b and reduces the
// squared norm on the fly (no q vector, no separate norm kernel).
#include "dslash_site.cuh"
#include "reduce.cuh"

namespace qcd {

namespace {

constexpr int kBlock = kDslashBlock;
constexpr int NR = kMultiRhs;
#ifndef QCD_MULTI_MINB
#define QCD_MULTI_MINB 4   // 128 registers; measured at 32^3x8 (residual pass): 2 -> 82 us, 3 -> 67, 4 -> 53, 5 (spills) -> 75
#endif

template <bool RES, int ROWS>
__global__ void __launch_bounds__(kBlock, QCD_MULTI_MINB)
dslash_multi_kernel(const Geom g, const DslashMultiParams p)
{
    constexpr int NW = 3 * ROWS;
    const int Vh = g.Vh;
    const int par = p.out_parity;
    Site s;
    locate_tile<ROWS == 2>(g, par, p.reverse ? gridDim.x - 1 - blockIdx.x : blockIdx.x, threadIdx.x, s);
    // alternating sweeps with the tail kept in L2, as in dslash.cu (the two launches of a batch have opposite parity)
    const uint64_t pol = l2_policy(blockIdx.x + (unsigned)p.keep_tiles >= gridDim.x);
    pdl_wait();
    pdl_launch_dependents();
    double sum[NR];
#pragma unroll
    for (int j = 0; j < NR; ++j) sum[j] = 0.0;
    if (s.valid) {
        const uint32_t h = s.h;
        double2 acc[NR][3];
#pragma unroll
        for (int j = 0; j < NR; ++j) acc[j][0] = acc[j][1] = acc[j][2] = make_double2(0.0, 0.0);
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) {
            {   // forward hop
                double2 u[9];
                load_link_hint<ROWS>(p.W + ((long)(par * 4 + mu) * NW) * Vh + h, Vh, u, pol);
#pragma unroll
                for (int j = 0; j < NR; ++j) {
                    if (j < p.nrhs) {
                        const double2 *__restrict__ in = p.in + p.in_off[j] + s.hp[mu];
                        double2 v[3];
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            v[c] = __ldg(in + (long)c * Vh);
                            if (ROWS == 2) v[c] = make_double2(flip(v[c].x, s.nf[mu]), flip(v[c].y, s.nf[mu]));
                        }
#pragma unroll
                        for (int a = 0; a < 3; ++a)
#pragma unroll
                            for (int b = 0; b < 3; ++b) cmad(acc[j][a], u[a * 3 + b], v[b]);
                    }
                }
            }
            {   // backward hop
                double2 u[9];
                load_link_hint<ROWS>(p.W + ((long)((1 - par) * 4 + mu) * NW) * Vh + s.hm[mu], Vh, u, pol);
#pragma unroll
                for (int j = 0; j < NR; ++j) {
                    if (j < p.nrhs) {
                        const double2 *__restrict__ in = p.in + p.in_off[j] + s.hm[mu];
                        double2 v[3];
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            v[c] = __ldg(in + (long)c * Vh);
                            if (ROWS == 2) v[c] = make_double2(flip(v[c].x, s.nb[mu]), flip(v[c].y, s.nb[mu]));
                        }
#pragma unroll
                        for (int a = 0; a < 3; ++a)
#pragma unroll
                            for (int b = 0; b < 3; ++b) cmsub_conj(acc[j][a], u[b * 3 + a], v[b]);
                    }
                }
            }
        }
#pragma unroll
        for (int j = 0; j < NR; ++j) {
            if (j < p.nrhs) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    double2 a = acc[j][c];
                    if (ROWS == 2) a = make_double2(0.5 * a.x, 0.5 * a.y);
                    if (RES) {
                        // d = b - ((m^2 + sigma) x - D tmp)
                        const double2 x = __ldg(p.src + p.src_off[j] + (long)c * Vh + h);
                        const double2 bb = __ldg(p.b + (long)c * Vh + h);
                        const double dx = bb.x - fma(p.coeff[j], x.x, -a.x);
                        const double dy = bb.y - fma(p.coeff[j], x.y, -a.y);
                        sum[j] = fma(dx, dx, sum[j]);
                        sum[j] = fma(dy, dy, sum[j]);
                    } else {
                        p.out[p.out_off[j] + (long)c * Vh + h] = a;
                    }
                }
            }
        }
    }
    if (RES) {
        double total[NR];
        if (grid_sum_last_block_n<kBlock, NR>(sum, p.partial, p.counter, total)) {
            if (threadIdx.x == 0) {
#pragma unroll
                for (int j = 0; j < NR; ++j)       // unrolled: `total` stays in registers (no stack frame)
                    if (j < p.nrhs) *p.result[j] = total[j];
            }
        }
    }
}

}  // namespace

int launch_dslash_multi(const Geom &g, const DslashMultiParams &p, Launch L)
{
    const int blocks = dslash_grid_blocks(g);
    const bool res = p.b != nullptr;
    if (p.link_rows == 2) {
        if (res) launch_kernel_apw(dslash_multi_kernel<true, 2>, blocks, kBlock, L.s, L.pdl, L.apw, g, p);
        else launch_kernel_apw(dslash_multi_kernel<false, 2>, blocks, kBlock, L.s, L.pdl, L.apw, g, p);
    } else {
        if (res) launch_kernel_apw(dslash_multi_kernel<true, 3>, blocks, kBlock, L.s, L.pdl, L.apw, g, p);
        else launch_kernel_apw(dslash_multi_kernel<false, 3>, blocks, kBlock, L.s, L.pdl, L.apw, g, p);
    }
    return 1;
}

}  // namespace qcd
