// dslash_site.cuh -- pieces shared by the Dslash kernels (dslash.cu, dslash_multi.cu): complex
// multiply-adds, the two-row reconstruction, and the map CTA/thread -> output site + neighbours.
#pragma once
#include "internal.cuh"

namespace qcd {

#ifndef QCD_DSLASH_BLOCK
#define QCD_DSLASH_BLOCK 128
#endif
constexpr int kDslashBlock = QCD_DSLASH_BLOCK;   // sites per CTA = one chunk of a t-slice

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

// Output site of this thread and the half indices of its 8 neighbours (all of the opposite parity).
struct Site {
    uint32_t h;        // half index of the output site
    bool valid;
    int hp[4], hm[4];  // half indices of x+mu, x-mu
    int nf[4], nb[4];  // two-row storage only: 1 where the forward / backward hop carries a minus sign
};

// CTA order.  A chunk is kDslashBlock consecutive sites of one t-slice.  The chunks of a slice are
// cut into groups of g.tgroup; CTAs walk group by group, and inside a group t runs slowest:
//     blockIdx = (group * nt_run + t - t0) * tgroup + chunk_in_group   (last group may be shorter;
//     a launch covers the t-slices t0 <= t < t0 + nt_run, normally all Nt of them)
// so the CTAs that read the same input sites as +-t neighbours are tgroup CTAs apart instead of a
// whole t-slice of CTAs (1024 CTAs = 163 MB of link traffic at 64^3x16, more than L2 holds: ncu
// showed 2.7-2.8 GB of DRAM reads per apply against 2.52 GB algorithmic), while each group still
// streams tgroup * 2 KB contiguous bytes of every link plane.  tgroup == chunks: plain h order.
// SIGNS: also derive eta_mu(x) and the t-seam signs (needed when the links are stored without them).
// tile (= CTA of the one-tile-per-CTA kernels) -> t-slice and first site of its chunk inside the slice
__device__ __forceinline__ void tile_origin(const Geom &g, uint32_t tile, uint32_t &t, uint32_t &sl0)
{
    const uint32_t per_group = (uint32_t)g.tgroup * (uint32_t)g.nt_run;
    const uint32_t grp = tile / per_group, rem = tile - grp * per_group;
    const uint32_t first = grp * (uint32_t)g.tgroup;
    const uint32_t width = min((uint32_t)g.tgroup, (uint32_t)g.chunks - first);   // chunks in this group
    const uint32_t tq = rem / width;
    t = (uint32_t)g.t0 + tq;
    sl0 = (first + (rem - tq * width)) * kDslashBlock;
}

template <bool SIGNS>
__device__ __forceinline__ void locate_tile(const Geom &g, int par, uint32_t tile, uint32_t lane, Site &s)
{
    uint32_t t, sl0;
    tile_origin(g, tile, t, sl0);
    const uint32_t sl = sl0 + lane;    // index inside the t-slice
    s.valid = sl < (uint32_t)g.st;
    const uint32_t h = t * (uint32_t)g.st + sl;
    s.h = h;
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) s.nf[mu] = s.nb[mu] = 0;
    if (s.valid) {
        uint32_t q, xh, y, z;
        g.dxh.divmod(sl, q, xh);
        g.dy.divmod(q, z, y);
        const int r = (y + z + t + par) & 1;      // x = 2*xh + r
        const int xh_p = r ? ((int)xh + 1 == g.Nxh ? 0 : (int)xh + 1) : (int)xh;
        const int xh_m = r ? (int)xh : (xh == 0 ? g.Nxh - 1 : (int)xh - 1);
        s.hp[0] = (int)h - (int)xh + xh_p;
        s.hm[0] = (int)h - (int)xh + xh_m;
        s.hp[1] = (int)h + ((int)y + 1 == g.Ny ? -(g.Ny - 1) * g.sy : g.sy);
        s.hm[1] = (int)h + (y == 0 ? (g.Ny - 1) * g.sy : -g.sy);
        s.hp[2] = (int)h + ((int)z + 1 == g.Nz ? -(g.Nz - 1) * g.sz : g.sz);
        s.hm[2] = (int)h + (z == 0 ? (g.Nz - 1) * g.sz : -g.sz);
        s.hp[3] = (int)h + ((int)t + 1 == g.Nt ? -(g.Nt - 1) * g.st : g.st);
        s.hm[3] = (int)h + (t == 0 ? (g.Nt - 1) * g.st : -g.st);
#ifdef QCD_DEBUG_BOUNDS   // build with QCD_NVCC_EXTRA=-DQCD_DEBUG_BOUNDS: any neighbour outside [0, Vh) traps
        for (int mu = 0; mu < 4; ++mu)
            if ((unsigned)s.hp[mu] >= (unsigned)g.Vh || (unsigned)s.hm[mu] >= (unsigned)g.Vh || h >= (uint32_t)g.Vh)
                __trap();
#endif
        if (SIGNS) {
            const int x = 2 * (int)xh + r;
            s.nf[1] = s.nb[1] = x & 1;                   // eta_1 = (-1)^x
            s.nf[2] = s.nb[2] = (x + (int)y) & 1;        // eta_2 = (-1)^(x+y)
            const int e3 = (x + (int)y + (int)z) & 1;    // eta_3 = (-1)^(x+y+z)
            s.nf[3] = e3 ^ ((int)t + 1 == g.Nt);         // s+ on the hop t = Nt-1 -> 0  (C5)
            s.nb[3] = e3 ^ (t == 0);                     // s- on the hop t = 0 -> Nt-1
        }
    }
}

template <bool SIGNS>
__device__ __forceinline__ void locate(const Geom &g, int par, Site &s)
{
    locate_tile<SIGNS>(g, par, blockIdx.x, threadIdx.x, s);
}

__device__ __forceinline__ double2 widen(double2 v) { return v; }
__device__ __forceinline__ double2 widen(float2 v) { return make_double2((double)v.x, (double)v.y); }

// u[0 .. 3*ROWS) <- the stored entries of one link (plane stride Vh); ROWS == 2: rebuild row 2.
// Streaming (evict-first) loads: every link is used once per apply, so the links should neither push the
// vectors out of L2 (the output of one Dslash is the gathered input of the next) nor cycle through it in
// LRU order.  Measured, us per apply at 32^3x8 / 48^3x12 / 64^3x16: __ldg 22.9 / 120.7 / 379.3, __ldcs
// 21.1 / 117.8 / 376.3.
template <int ROWS, class WT>
__device__ __forceinline__ void load_link(const WT *__restrict__ w, int Vh, double2 *u)
{
#pragma unroll
    for (int i = 0; i < 3 * ROWS; ++i) u[i] = widen(__ldcs(w + (long)i * Vh));
    if (ROWS == 2) third_row(u);
}

// The same with the L2 eviction priority as a run-time operand (one code path for both policies, chosen
// per CTA; dslash.cu): ld.global.nc, no L1 allocation (a link is used once), L2 priority from a
// createpolicy value -- evict_first reproduces the streaming load above (20.5 vs 20.6 us at 32^3x8).
__device__ __forceinline__ uint64_t l2_policy(bool keep)
{
    uint64_t pol;
    if (keep) asm("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(pol));
    else asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ double2 ld_hint(const double2 *p, uint64_t pol)
{
    double2 v;
    asm("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ float2 ld_hint(const float2 *p, uint64_t pol)
{
    float2 v;
    asm("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f32 {%0, %1}, [%2], %3;" : "=f"(v.x), "=f"(v.y) : "l"(p), "l"(pol));
    return v;
}
template <int ROWS, class WT>
__device__ __forceinline__ void load_link_hint(const WT *__restrict__ w, int Vh, double2 *u, uint64_t pol)
{
#pragma unroll
    for (int i = 0; i < 3 * ROWS; ++i) u[i] = widen(ld_hint(w + (long)i * Vh, pol));
    if (ROWS == 2) third_row(u);
}

}  // namespace qcd
