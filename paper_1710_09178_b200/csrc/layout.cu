// layout.cu -- a1 of SURVEY 8(a): canonical (lexicographic AoS) <-> internal (parity-split SoA).
//
// Links: W_mu(x) = 1/2 eta_mu(x) s+_mu(x) U_mu(x).  The paper absorbs the staggered phases into the
// stored links; here the 1/2 of the M = m + D normalisation and the
// antiperiodic sign of the t-seam hop (C5) are folded in as well.  Because eta_mu does not depend on
// x_mu, and s-_mu(x) = s+_mu(x - mu), the backward hop at x needs exactly W_mu(x - mu)^dag.
#include "internal.cuh"

namespace qcd {

namespace {

constexpr int kBlock = 256;

// one thread per (half index h, parity of the base site): 4 links each.
// ROWS == 3: all nine entries with 1/2 eta s+ folded in.  ROWS == 2: rows 0 and 1 of the plain U,
// bit for bit ("stores and moves only two rows"); dslash.cu rebuilds the rest.
template <int ROWS>
__global__ void __launch_bounds__(kBlock)
ingest_links_kernel(Geom g, const double2 *__restrict__ U, double2 *__restrict__ W, int *not_su3)
{
    pdl_wait();
    pdl_launch_dependents();
    const int Vh = g.Vh;
    uint32_t tid = blockIdx.x * kBlock + threadIdx.x;
    if (tid >= 2u * Vh) return;
    int par = tid >= (uint32_t)Vh;
    uint32_t h = tid - par * Vh;
    uint32_t q, xh, y, z, t;
    g.dxh.divmod(h, q, xh);
    g.dy.divmod(q, q, y);
    g.dz.divmod(q, t, z);
    int x = 2 * xh + ((y + z + t + par) & 1);
    long l = 2L * h + (x & 1);                      // canonical address: h = l >> 1
    // eta_mu(x) = (-1)^(sum_{nu<mu} x_nu)
    double eta[4] = {1.0, (x & 1) ? -1.0 : 1.0, ((x + y) & 1) ? -1.0 : 1.0,
                     ((x + y + z) & 1) ? -1.0 : 1.0};
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
        double f = 0.5 * eta[mu];
        if (mu == 3 && t == (uint32_t)g.Nt - 1) f = -f;   // s+ across the t seam (C5)
        if (ROWS == 2) f = 1.0;
        const double2 *u = U + (l * 4 + mu) * 9;
        double2 *w = W + ((long)(par * 4 + mu) * (3 * ROWS)) * Vh + h;
#pragma unroll
        for (int c = 0; c < 3 * ROWS; ++c) {
            double2 v = u[c];
            w[(long)c * Vh] = make_double2(f * v.x, f * v.y);
        }
        if (ROWS == 2) {
            // two-row storage can only represent SU(3): refuse anything whose third row is not
            // conj(row_0 x row_1) (qcd_load_gauge reports it; "recovers the third by
            // orthogonalization" presupposes it)
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const int c1 = (c + 1) % 3, c2 = (c + 2) % 3;
                const double2 a1 = u[c1], a2 = u[c2], b1 = u[3 + c1], b2 = u[3 + c2], r = u[6 + c];
                const double tx = a1.x * b2.x - a1.y * b2.y - a2.x * b1.x + a2.y * b1.y;
                const double ty = a1.x * b2.y + a1.y * b2.x - a2.x * b1.y - a2.y * b1.x;
                if (!(fabs(r.x - tx) <= 1e-10 && fabs(r.y + ty) <= 1e-10)) *not_su3 = 1;
            }
        }
    }
}

// fp32 copy of the three-row links (NEXT-3): the same W_mu(x) = 1/2 eta s+ U, every entry rounded to
// fp32.  The factor is a signed power of two, so rounding commutes with it: W32 = 1/2 eta s+ fl32(U).
__global__ void __launch_bounds__(kBlock)
ingest_links32_kernel(Geom g, const double2 *__restrict__ U, float2 *__restrict__ W)
{
    pdl_wait();
    pdl_launch_dependents();
    const int Vh = g.Vh;
    uint32_t tid = blockIdx.x * kBlock + threadIdx.x;
    if (tid >= 2u * Vh) return;
    int par = tid >= (uint32_t)Vh;
    uint32_t h = tid - par * Vh;
    uint32_t q, xh, y, z, t;
    g.dxh.divmod(h, q, xh);
    g.dy.divmod(q, q, y);
    g.dz.divmod(q, t, z);
    int x = 2 * xh + ((y + z + t + par) & 1);
    long l = 2L * h + (x & 1);
    double eta[4] = {1.0, (x & 1) ? -1.0 : 1.0, ((x + y) & 1) ? -1.0 : 1.0, ((x + y + z) & 1) ? -1.0 : 1.0};
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
        double f = 0.5 * eta[mu];
        if (mu == 3 && t == (uint32_t)g.Nt - 1) f = -f;
        const double2 *u = U + (l * 4 + mu) * 9;
        float2 *w = W + ((long)(par * 4 + mu) * 9) * Vh + h;
#pragma unroll
        for (int c = 0; c < 9; ++c) {
            double2 v = u[c];
            w[(long)c * Vh] = make_float2((float)(f * v.x), (float)(f * v.y));
        }
    }
}

// canonical parity vector [j][3] (j == h) -> planes [3][Vh], sites h0 <= h < h1
__global__ void __launch_bounds__(kBlock)
pack_kernel(int Vh, int h0, int h1, const double2 *__restrict__ canon, double2 *__restrict__ v)
{
    pdl_wait();
    pdl_launch_dependents();
    int h = h0 + blockIdx.x * kBlock + threadIdx.x;
    if (h >= h1) return;
#pragma unroll
    for (int c = 0; c < 3; ++c) v[(long)c * Vh + h] = canon[3L * h + c];
}

__global__ void __launch_bounds__(kBlock)
unpack_kernel(int Vh, int h0, int h1, const double2 *__restrict__ v, double2 *__restrict__ canon)
{
    pdl_wait();
    pdl_launch_dependents();
    int h = h0 + blockIdx.x * kBlock + threadIdx.x;
    if (h >= h1) return;
#pragma unroll
    for (int c = 0; c < 3; ++c) canon[3L * h + c] = v[(long)c * Vh + h];
}

}  // namespace

int launch_ingest_links(const Geom &g, const double *links_canon, double2 *W, int link_rows, int *not_su3,
                        Launch L)
{
    int blocks = (2 * g.Vh + kBlock - 1) / kBlock;
    if (link_rows == 2)
        launch_kernel(ingest_links_kernel<2>, blocks, kBlock, L.s, L.pdl, g, (const double2 *)links_canon, W, not_su3);
    else
        launch_kernel(ingest_links_kernel<3>, blocks, kBlock, L.s, L.pdl, g, (const double2 *)links_canon, W, not_su3);
    return 1;
}

int launch_ingest_links32(const Geom &g, const double *links_canon, float2 *W32, Launch L)
{
    int blocks = (2 * g.Vh + kBlock - 1) / kBlock;
    launch_kernel(ingest_links32_kernel, blocks, kBlock, L.s, L.pdl, g, (const double2 *)links_canon, W32);
    return 1;
}

int launch_pack(const Geom &g, const double *canon, double2 *internal, Launch L, int h0, int h1)
{
    if (h1 < 0) h1 = g.Vh;
    int blocks = (h1 - h0 + kBlock - 1) / kBlock;
    launch_kernel(pack_kernel, blocks, kBlock, L.s, L.pdl, g.Vh, h0, h1, (const double2 *)canon, internal);
    return 1;
}

int launch_unpack(const Geom &g, const double2 *internal, double *canon, Launch L, int h0, int h1)
{
    if (h1 < 0) h1 = g.Vh;
    int blocks = (h1 - h0 + kBlock - 1) / kBlock;
    launch_kernel(unpack_kernel, blocks, kBlock, L.s, L.pdl, g.Vh, h0, h1, internal, (double2 *)canon);
    return 1;
}

}  // namespace qcd
