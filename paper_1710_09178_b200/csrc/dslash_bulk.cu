// dslash_bulk.cu -- the same operator as dslash.cu (a2/a3/a4 of SURVEY 8(a); PAPER.md:106, :112,
// :116-119), with the LINKS staged through shared memory by the bulk-copy engine instead of through
// registers ("staged through shared memory or TMA", BASELINE.json north_star).
// Selected by qcd_set_option(QCD_OPT_DSLASH_KERNEL, 1); results are bit-identical to dslash.cu
// (same arithmetic in the same order), only the way the link bytes reach the registers differs.
//
// Why it was built: the register-staged kernel keeps (threads resident) x (link loads ptxas hoists) bytes in
// flight, which 128 registers cap at about two hops per thread; ncu shows 22 % of the warp slots active and
// the DRAM pipe at 70-86 %.  Here a producer warp keeps kStages hops of the tile in flight with
// cp.async.bulk (SASS: UBLKCP), independent of the consumers' registers, and - when the grid is
// persistent - runs ahead across tile boundaries.  What came of it: DESIGN.md section 5 (it is slower).
//
// Tile = the 128 consecutive sites of a chunk (as in dslash.cu: same CTA order, same `locate`).  For a
// hop, every link plane the tile needs is ONE contiguous run of the plane array:
//     forward  mu      W[par][mu][c][h0 .. h0+n)
//     backward x       W[1-par][0][c][h0-1 .. h0+n)      (neighbour index h-1 or h, row wrap inside)
//     backward y, z    W[1-par][mu][c][h0-s_mu .. +n)    (sites with x_mu = 0 wrap: read directly)
//     backward t       W[1-par][3][c][h0 -+ s_t .. +n)   (the whole tile wraps or does not)
// and so is the neighbour vector (QCD_BULK_VEC: three more planes per stage; the run of the backward link
// for backward hops, the tile's own run shifted the other way for forward hops).  A stage is 3*ROWS + 3
// bulk copies of about 2 KB (one per plane, issued by one lane each), landing in smem[plane][i] behind an
// mbarrier (complete_tx).  A consumer thread reads its entries site-fastest (LDS.128, conflict-free) when
// its neighbour index lies inside the copied run, and falls back to a direct load when it does not
// (periodic wrap in y or z, a row cut by the tile boundary: a few per cent of the sites).
#include <algorithm>

#include "cg_scalars.cuh"
#include "dslash_site.cuh"
#include "reduce.cuh"

namespace qcd {

namespace {

constexpr int kTile = kDslashBlock;          // sites per tile = consumer threads
constexpr int kThreads = kTile + 32;         // + one producer warp
#ifndef QCD_BULK_VEC
#define QCD_BULK_VEC 1                       // 1: the neighbour vectors of a hop are staged with its links (3 more planes)
#endif
#ifndef QCD_BULK_STAGES
#define QCD_BULK_STAGES (QCD_BULK_VEC ? 2 : 4)   // hops in flight per CTA
#endif
#ifndef QCD_BULK_MINB3
#define QCD_BULK_MINB3 (QCD_BULK_VEC ? 4 : 3)    // resident CTAs per SM asked of ptxas, three-row links (49 / 73 KB smem each)
#endif
#ifndef QCD_BULK_MINB2
#define QCD_BULK_MINB2 4                     // two-row links (49 KB each)
#endif
constexpr int kStages = QCD_BULK_STAGES;
constexpr int kVecPlanes = QCD_BULK_VEC ? 3 : 0;   // colour planes of the neighbour vector staged per hop
constexpr int kPlane = kTile + 2;            // double2 per plane of a stage (runs are <= kTile + 1 long)

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)      // no arrival: more bytes will be announced
{
    asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    const uint32_t a = smem_u32(bar);
    uint32_t ok;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                     "selp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(a), "r"(parity) : "memory");
    } while (!ok);
}
// links are used once per apply: evict-first in L2, as the __ldcs of the register-staged kernel
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar, uint64_t pol)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(pol) : "memory");
}

// Source window of hop k (k = 2 mu + backward) of the tile whose first site is h0 (n sites, t-slice t):
// elements [lo, lo + len) of each of the hop's link planes are copied to smem[plane][0 .. len).
__device__ __forceinline__ void hop_window(const Geom &g, uint32_t t, int h0, int n, int hop, int &lo, int &len)
{
    int off = 0, l = n;
    if (hop & 1) {
        const int mu = hop >> 1;
        if (mu == 0) { off = -1; l = n + 1; }
        else if (mu == 1) off = -g.sy;
        else if (mu == 2) off = -g.sz;
        else off = t == 0 ? (g.Nt - 1) * g.st : -g.st;
    }
    int a = h0 + off, b = a + l;
    a = max(a, 0);
    b = min(b, g.Vh);
    lo = a;
    len = max(b - a, 0);
}

// Source window of the NEIGHBOUR VECTOR of hop k: backward hops gather at the same index as their link
// (x - mu); forward hops at x + mu: the tile's own run shifted by one row / plane / slice, or, for +x, the
// run [h0, h0 + n] (neighbour index h or h + 1).  Sites on the periodic wrap fall outside and gather directly.
__device__ __forceinline__ void vec_window(const Geom &g, uint32_t t, int h0, int n, int hop, int &lo, int &len)
{
    if (hop & 1) { hop_window(g, t, h0, n, hop, lo, len); return; }
    const int mu = hop >> 1;
    int off = 0, l = n;
    if (mu == 0) l = n + 1;
    else if (mu == 1) off = g.sy;
    else if (mu == 2) off = g.sz;
    else off = (int)t + 1 == g.Nt ? -(g.Nt - 1) * g.st : g.st;
    int a = h0 + off, b = a + l;
    a = max(a, 0);
    b = min(b, g.Vh);
    lo = a;
    len = max(b - a, 0);
}

// producer state: which (tile, hop) is issued next, into which stage
struct Issue {
    uint32_t tile;
    int hop, stage;
    uint32_t phase;      // parity of the `empty` phase the producer waits for is phase ^ 1
};

template <bool XPAY, bool DOT, int ROWS>
__global__ void __launch_bounds__(kThreads, ROWS == 2 ? QCD_BULK_MINB2 : QCD_BULK_MINB3)
dslash_bulk_kernel(const Geom g, const DslashParams p, const uint32_t ntiles)
{
    constexpr int NW = 3 * ROWS;
    constexpr int NP = NW + kVecPlanes;          // planes of a stage: the link entries, then the neighbour vector
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double2 *sbuf = reinterpret_cast<double2 *>(smem_raw);                            // [kStages][NP][kPlane]
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + (size_t)kStages * NP * kPlane * sizeof(double2));
    uint64_t *empty = full + kStages;
    const int Vh = g.Vh;
    const int par = p.out_parity;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const bool producer = warp == kTile / 32;

    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) {
            mbar_init(&full[s], 1);            // the producer's arrive.expect_tx
            mbar_init(&empty[s], kTile / 32);  // one arrive per consumer warp
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    // One hop of the producer: wait for the stage to be free, announce the bytes, issue the bulk copies.
    // The links are constant between qcd_load_gauge calls, the vectors are the predecessor's output: so the
    // hops issued BEFORE griddepcontrol.wait carry their links only (expect_tx without arrival), and the
    // vector planes of those stages follow after the wait with the arrival (part = 1 links, 2 vectors, 3 both).
    Issue is{blockIdx.x, 0, 0, 0};
    // L2 priority of the link bytes, per tile as in dslash.cu: the last keep_tiles tiles of the sweep keep
    const uint64_t pol_first = l2_policy(false), pol_keep = l2_policy(true);
    auto issue_part = [&](uint32_t seq, int hop, int stage, int part) {
        uint32_t t, sl0;
        tile_origin(g, p.reverse ? ntiles - 1 - seq : seq, t, sl0);
        const uint64_t pol = seq + (uint32_t)p.keep_tiles >= ntiles ? pol_keep : pol_first;
        const int n = min(kTile, g.st - (int)sl0);
        const int h0 = (int)(t * (uint32_t)g.st + sl0);
        int lo = 0, len = 0, vlo = 0, vlen = 0;
        if (part & 1) hop_window(g, t, h0, n, hop, lo, len);
        if (kVecPlanes && (part & 2)) vec_window(g, t, h0, n, hop, vlo, vlen);
        const uint32_t bytes = (uint32_t)(NW * len + kVecPlanes * vlen) * (uint32_t)sizeof(double2);
        const bool arrive = !kVecPlanes || (part & 2);         // the stage is complete with this part
        if (lane == 0) {
            if (arrive) {
                if (bytes > 0) mbar_arrive_expect_tx(&full[stage], bytes);
                else mbar_arrive(&full[stage]);
            } else if (bytes > 0) {
                mbar_expect_tx(&full[stage], bytes);
            }
        }
        __syncwarp();
        const int mu = hop >> 1;
        const long plane0 = (long)(((hop & 1) ? 1 - par : par) * 4 + mu) * NW;
        if ((part & 1) && lane < NW && len > 0)
            bulk_g2s(sbuf + ((size_t)stage * NP + lane) * kPlane, p.W + (plane0 + lane) * Vh + lo,
                     (uint32_t)len * (uint32_t)sizeof(double2), &full[stage], pol);
        if (kVecPlanes && (part & 2) && lane >= NW && lane < NP && vlen > 0)
            bulk_g2s(sbuf + ((size_t)stage * NP + lane) * kPlane, p.in + (long)(lane - NW) * Vh + vlo,
                     (uint32_t)vlen * (uint32_t)sizeof(double2), &full[stage], pol_keep);
    };
    auto advance = [&]() {
        if (++is.hop == 8) { is.hop = 0; is.tile += gridDim.x; }
        if (++is.stage == kStages) { is.stage = 0; is.phase ^= 1u; }
    };

    // Inside the CG, `done` was last written two or more kernels back: a dead iteration is recognised
    // early and requests nothing (a hint; the check after the wait decides, and a CTA that has requested
    // copies waits for them before it leaves).
    const bool dead_hint = p.st != nullptr && *(volatile const int *)&p.st->done;
    int early = 0;
    const Issue first = is;
    if (producer && !dead_hint)
        for (; early < kStages && is.tile < ntiles; ++early) {       // the ring is empty: no wait on `empty`
            issue_part(is.tile, is.hop, is.stage, 1);
            advance();
        }
    pdl_wait();
    pdl_launch_dependents();
    if (p.st != nullptr && p.st->done) {      // CG already converged: dead iteration
        if (producer && early > 0) {
            if (kVecPlanes && lane == 0)
                for (int s = 0; s < early; ++s) mbar_arrive(&full[s]);     // no vector part will follow
            __syncwarp();
            for (int s = 0; s < early; ++s) mbar_wait(&full[s], 0u);
        }
        return;
    }
    if (producer && kVecPlanes) {             // the vector planes of the hops issued before the wait
        Issue e = first;
        for (int s = 0; s < early; ++s) {
            issue_part(e.tile, e.hop, e.stage, 2);
            if (++e.hop == 8) { e.hop = 0; e.tile += gridDim.x; }
            ++e.stage;
        }
    }

    double dot = 0.0;
    if (producer) {
        while (is.tile < ntiles) {
            mbar_wait(&empty[is.stage], is.phase ^ 1u);
            issue_part(is.tile, is.hop, is.stage, 3);
            advance();
        }
    } else {
        int stage = 0;
        uint32_t phase = 0;
        for (uint32_t seq = blockIdx.x; seq < ntiles; seq += gridDim.x) {
            const uint32_t tile = p.reverse ? ntiles - 1 - seq : seq;
            const uint64_t pol = seq + (uint32_t)p.keep_tiles >= ntiles ? pol_keep : pol_first;
            Site site;
            locate_tile<ROWS == 2>(g, par, tile, threadIdx.x, site);
            const bool valid = site.valid;
            const int h = (int)site.h;
            const int h0 = h - (int)threadIdx.x;
            uint32_t t, sl0;
            tile_origin(g, tile, t, sl0);
            const int n = min(kTile, g.st - (int)sl0);
            const double2 *__restrict__ in = p.in;
            double2 acc[3];
            acc[0] = acc[1] = acc[2] = make_double2(0.0, 0.0);
            double2 vnext[3];
            if (!kVecPlanes && valid) {
#pragma unroll
                for (int c = 0; c < 3; ++c) vnext[c] = __ldg(in + (long)c * Vh + site.hp[0]);
            }
#pragma unroll
            for (int hop = 0; hop < 8; ++hop) {
                const int mu = hop >> 1;
                const bool bwd = hop & 1;
                double2 v[3], u[9];
                const int nbr = bwd ? site.hm[mu] : site.hp[mu];        // index of the neighbour site
                if (!kVecPlanes) {
#pragma unroll
                    for (int c = 0; c < 3; ++c) v[c] = vnext[c];
                    if (valid && hop < 7) {        // neighbour vector of the next hop: one hop ahead
                        const int nh = ((hop + 1) & 1) ? site.hm[(hop + 1) >> 1] : site.hp[(hop + 1) >> 1];
#pragma unroll
                        for (int c = 0; c < 3; ++c) vnext[c] = __ldg(in + (long)c * Vh + nh);
                    }
                }
                int lo, len, vlo = 0, vlen = 0;
                hop_window(g, t, h0, n, hop, lo, len);
                if (kVecPlanes) vec_window(g, t, h0, n, hop, vlo, vlen);
                const int src = bwd ? site.hm[mu] : h;        // index of this site's link in the plane
                const int idx = src - lo;
                const bool staged = (unsigned)idx < (unsigned)len;
                const int vidx = nbr - vlo;
                const bool vstaged = kVecPlanes && (unsigned)vidx < (unsigned)vlen;
                if (kVecPlanes && valid && !vstaged) {               // periodic wrap: gather directly, ahead of the wait
#pragma unroll
                    for (int c = 0; c < 3; ++c) v[c] = __ldg(in + (long)c * Vh + nbr);
                }
                mbar_wait(&full[stage], phase);
                if (valid) {
                    if (vstaged) {
                        const double2 *vp = sbuf + ((size_t)stage * NP + NW) * kPlane + vidx;
#pragma unroll
                        for (int c = 0; c < 3; ++c) v[c] = vp[c * kPlane];
                    }
                    if (staged) {
                        const double2 *sp = sbuf + (size_t)stage * NP * kPlane + idx;
#pragma unroll
                        for (int i = 0; i < NW; ++i) u[i] = sp[i * kPlane];
                    } else {
                        const double2 *__restrict__ w = p.W + ((long)((bwd ? 1 - par : par) * 4 + mu) * NW) * Vh + src;
#pragma unroll
                        for (int i = 0; i < NW; ++i) u[i] = ld_hint(w + (long)i * Vh, pol);
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[stage]);     // this warp has its entries in registers
                if (++stage == kStages) { stage = 0; phase ^= 1u; }
                if (valid) {
                    if (ROWS == 2) {
                        third_row(u);
                        const int neg = bwd ? site.nb[mu] : site.nf[mu];
#pragma unroll
                        for (int c = 0; c < 3; ++c) v[c] = make_double2(flip(v[c].x, neg), flip(v[c].y, neg));
                    }
                    if (!bwd) {
#pragma unroll
                        for (int a = 0; a < 3; ++a)
#pragma unroll
                            for (int b = 0; b < 3; ++b) cmad(acc[a], u[a * 3 + b], v[b]);
                    } else {
#pragma unroll
                        for (int a = 0; a < 3; ++a)
#pragma unroll
                            for (int b = 0; b < 3; ++b) cmsub_conj(acc[a], u[b * 3 + a], v[b]);
                    }
                }
            }
            if (valid) {
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
        }
    }
    if (DOT) {      // one partial per CTA, summed by the r-update (blas.cu)
        const double b = block_sum<kThreads>(dot);
        if (threadIdx.x == 0) p.partial[blockIdx.x] = b;
    }
}

template <bool XPAY, bool DOT, int ROWS>
cudaError_t launch_one(const Geom &g, const DslashParams &p, int grid, uint32_t ntiles, Launch L)
{
    constexpr size_t smem = (size_t)kStages * (3 * ROWS + kVecPlanes) * kPlane * sizeof(double2) + 2 * kStages * sizeof(uint64_t);
    static bool configured = false;          // one attribute call per instantiation (single device per process)
    auto kernel = dslash_bulk_kernel<XPAY, DOT, ROWS>;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3((unsigned)kThreads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = L.s;
    cudaLaunchAttribute attr[1];
    unsigned na = 0;
    if (L.pdl) {
        attr[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[na].val.programmaticStreamSerializationAllowed = 1;
        ++na;
    }
    cfg.attrs = attr;
    cfg.numAttrs = na;
    return cudaLaunchKernelEx(&cfg, kernel, g, p, ntiles);
}

}  // namespace

// persistent != 0: at most persistent CTAs per SM x 148 SMs walk the tiles round-robin (the producer
// streams across tile boundaries); 0: one CTA per tile
int dslash_bulk_grid_blocks(const Geom &g, int ctas_per_sm)
{
    const int ntiles = dslash_grid_blocks(g);
    return ctas_per_sm > 0 ? std::min(ntiles, 148 * ctas_per_sm) : ntiles;
}

int launch_dslash_bulk(const Geom &g, const DslashParams &p, int ctas_per_sm, Launch L)
{
    const int ntiles = dslash_grid_blocks(g);
    const int grid = dslash_bulk_grid_blocks(g, ctas_per_sm);
    const uint32_t nt = (uint32_t)ntiles;
    if (p.link_rows == 2) {
        if (p.src == nullptr) launch_one<false, false, 2>(g, p, grid, nt, L);
        else if (p.dot_mode == 0) launch_one<true, false, 2>(g, p, grid, nt, L);
        else launch_one<true, true, 2>(g, p, grid, nt, L);
    } else {
        if (p.src == nullptr) launch_one<false, false, 3>(g, p, grid, nt, L);
        else if (p.dot_mode == 0) launch_one<true, false, 3>(g, p, grid, nt, L);
        else launch_one<true, true, 3>(g, p, grid, nt, L);
    }
    return 1;
}

}  // namespace qcd
