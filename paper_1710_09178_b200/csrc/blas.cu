// blas.cu -- a5/a6 of SURVEY 8(a): fused BLAS-1 of the multishift CG.  Hand loops instead of BLAS
// calls, reductions with an explicit reduction variable (the paper's own finding), and
// light loops merged into heavier ones: the r-update carries the norm, the shift
// update streams x_k and p_k of every active shift in one pass over r ("the heaviest kernel which
// updates three large arrays").  All coefficients are read from the device-resident
// CgState; nothing returns to the host inside an iteration.
#include <algorithm>

#include <cooperative_groups.h>

#include "cg_scalars.cuh"
#include "reduce.cuh"

namespace qcd {

namespace {

constexpr int kBlock = 256;
constexpr int kMaxBlocks = 148 * 16;  // grid-stride above this: a multiple of the SM count

// r = b ; p_k = b (all k) ; rho = rho_b = <b,b> ; x_k are zeroed by a memset
__global__ void __launch_bounds__(kBlock)
cg_init_kernel(long n2, const double2 *__restrict__ b, double2 *__restrict__ r,
               double2 *__restrict__ p, long pstride, int nshift, double *partial, CgState *st,
               int Vh, int halo)
{
    pdl_wait();
    pdl_launch_dependents();
    double s = 0.0;
    for (long i = (long)blockIdx.x * kBlock + threadIdx.x; i < n2; i += (long)gridDim.x * kBlock) {
        double2 v = __ldg(b + i);
        if (halo > 0) {        // slab mode: the first and the last t-slice (halo sites each) are not this rank's
            const int h = (int)(i % Vh);
            if (h < halo || h >= Vh - halo) v = make_double2(0.0, 0.0);
        }
        r[i] = v;
        for (int k = 0; k < nshift; ++k) p[k * pstride + i] = v;
        s += v.x * v.x + v.y * v.y;
    }
    double total;
    if (grid_sum_last_block<kBlock>(s, partial, &st->counter, total)) {
        if (threadIdx.x == 0) {
            st->rho = total;
            st->rho_b = total;
            if (total == 0.0) { st->done = 1; st->done_prev = 1; }   // b = 0: x_k = 0 is exact
        }
    }
}

// r -= alpha q ; rho' = <r,r> ; last block: zeta_new, alpha_k, beta, beta_k, zeta rotation, freezing,
// stop test.  alpha = rho / <p_0,q> is formed here, by every CTA for itself, from the per-CTA partial
// sums the second Dslash of the iteration left in pap_partial[0 .. npap): same loads, same order, same
// tree in every CTA, so all CTAs hold the same bits (and runs repeat bit for bit).  That takes the
// ticket, the fence and the serial last-block pass out of the stencil: one reduction tail per
// iteration instead of two.
// LOOP: the kernel is a node of the WHILE graph of QCD_OPT_CG_GRAPH = 2 and sets its condition.  A
// separate instantiation, because a kernel that references the device-side graph API is invisible to
// ncu (the launch list of the default path would lose its r-update rows).
constexpr int kRUnroll = 4;                       // independent 16-byte loads per array per thread
constexpr int kRChunk = kBlock * kRUnroll;
constexpr int kRMaxBlocks = 148 * 4;

template <bool LOOP, bool SPLIT = false>
__global__ void __launch_bounds__(kBlock)
cg_update_r_kernel(long n2, double2 *ring, const double2 *__restrict__ q,
                   const double *__restrict__ pap_partial, int npap, double *partial, CgState *st,
                   cudaGraphConditionalHandle loop)
{
    pdl_wait();
    pdl_launch_dependents();
    if (blockIdx.x == 0 && threadIdx.x == 0) st->enq += 1;     // read by the flush kernel only
    if (st->done) {                       // dead iteration after convergence
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            st->done_prev = 1;
            if (LOOP) cudaGraphSetConditional(loop, 0);
        }
        return;
    }
    // this is iteration n = st->iter + 1 (st->iter is advanced by the last block only, after every CTA has
    // read it): r_{n-1} is ring slot (n - 2) mod defer, r_n goes to slot (n - 1) mod defer
    const int m = st->defer, it = st->iter;
    const double2 *rin = ring + (long)((it + m - 1) % m) * n2;     // == r when defer == 1: no __restrict__
    double2 *r = ring + (long)(it % m) * n2;
    // the first chunk of r and q is requested BEFORE the alpha reduction: the loads do not depend on it and
    // overlap its two barriers and its round trip to L2 (normally the only chunk: the grid covers the vector)
    long base = (long)blockIdx.x * kRChunk + threadIdx.x;
    double2 rv[kRUnroll], qv[kRUnroll];
#pragma unroll
    for (int e = 0; e < kRUnroll; ++e) {
        const long i = base + (long)e * kBlock;
        if (i < n2) { rv[e] = rin[i]; qv[e] = __ldg(q + i); }
    }
    double t = 0.0;
    for (int i = threadIdx.x; i < npap; i += kBlock) t += __ldcg(pap_partial + i);
    const double pAp = block_sum<kBlock>(t);
    const double alpha = st->rho / pAp;   // st->rho is rewritten by the last block only, after every CTA has read it
    double s = 0.0;
    while (base < n2) {
#pragma unroll
        for (int e = 0; e < kRUnroll; ++e) {
            const long i = base + (long)e * kBlock;
            if (i < n2) {
                rv[e].x = fma(-alpha, qv[e].x, rv[e].x);
                rv[e].y = fma(-alpha, qv[e].y, rv[e].y);
                r[i] = rv[e];
                s += rv[e].x * rv[e].x + rv[e].y * rv[e].y;
            }
        }
        base += (long)gridDim.x * kRChunk;
#pragma unroll
        for (int e = 0; e < kRUnroll; ++e) {
            const long i = base + (long)e * kBlock;
            if (i < n2) { rv[e] = rin[i]; qv[e] = __ldg(q + i); }
        }
    }
    double total;
    if (grid_sum_last_block<kBlock>(s, partial, &st->counter, total)) {
        if (SPLIT) {                      // slab mode: the sum over the ranks and the scalar step follow (api.cu)
            if (threadIdx.x == 0) st->red[1] = total;
            return;
        }
        cg_step_alpha(st, pAp);
        __syncthreads();
        cg_step_beta(st, total);
        // device-side loop (QCD_OPT_CG_GRAPH = 2): this iteration's shift update still runs (it is part
        // of the loop body); the WHILE node then stops when the stop test above has set `done`
        if (LOOP && threadIdx.x == 0) cudaGraphSetConditional(loop, st->done ? 0u : 1u);
    }
}

// r-update AND base-shift update in one cooperative kernel (QCD_OPT_CG_FUSE = 1; SURVEY 7 hard part 3: "a
// cooperative persistent kernel with grid.sync() for the BLAS-1 half of the iteration").  Phase 1 is the
// r-update above; after grid.sync() every CTA adds the per-CTA partial sums of ||r'||^2 itself (consumer
// side, fixed order: same bits everywhere), forms beta, and updates x_0, p_0; CTA 0 then runs the scalar
// recurrences for all shifts.  For the base shift zeta stays exactly 1 (delta_0 = 0 in the recurrence),
// so alpha_0 = alpha, the r-coefficient is 1 and beta_0 = beta: bit-identical to the two-kernel path.
// Saves a kernel boundary, the ticket and the serial last-block pass; needs the whole grid co-resident.
__global__ void __launch_bounds__(kBlock)
cg_update_r_base_kernel(long n2, double2 *ring, const double2 *__restrict__ q,
                        const double *__restrict__ pap_partial, int npap, double *partial,
                        double2 *__restrict__ x, double2 *__restrict__ p, CgState *st, int y_only)
{
    pdl_wait();
    pdl_launch_dependents();
    cooperative_groups::grid_group grid = cooperative_groups::this_grid();
    if (blockIdx.x == 0 && threadIdx.x == 0) st->enq += 1;
    if (st->done) {                       // dead iteration (every CTA sees the same flag: it is written after the grid sync only)
        if (blockIdx.x == 0 && threadIdx.x == 0) st->done_prev = 1;
        return;
    }
    const int m = st->defer, it = st->iter;
    const double rho = st->rho;
    const double2 *rin = ring + (long)((it + m - 1) % m) * n2;
    double2 *r = ring + (long)(it % m) * n2;
    // y-only form: x is the accumulator y, which takes c_0 alpha p_0 where x_0 would take alpha p_0
    double2 *__restrict__ x0 = y_only ? x : x + st->xoff[0];
    const double cy0 = y_only ? st->cy[0] : 1.0;
    double t = 0.0;
    for (int i = threadIdx.x; i < npap; i += kBlock) t += __ldcg(pap_partial + i);
    const double pAp = block_sum<kBlock>(t);
    const double alpha = rho / pAp;
    double s = 0.0;
    for (long base = (long)blockIdx.x * kRChunk + threadIdx.x; base < n2; base += (long)gridDim.x * kRChunk) {
        double2 rv[kRUnroll], qv[kRUnroll];
#pragma unroll
        for (int e = 0; e < kRUnroll; ++e) {
            const long i = base + (long)e * kBlock;
            if (i < n2) { rv[e] = rin[i]; qv[e] = __ldg(q + i); }
        }
#pragma unroll
        for (int e = 0; e < kRUnroll; ++e) {
            const long i = base + (long)e * kBlock;
            if (i < n2) {
                rv[e].x = fma(-alpha, qv[e].x, rv[e].x);
                rv[e].y = fma(-alpha, qv[e].y, rv[e].y);
                r[i] = rv[e];
                s += rv[e].x * rv[e].x + rv[e].y * rv[e].y;
            }
        }
    }
    const double bsum = block_sum<kBlock>(s);
    if (threadIdx.x == 0) partial[blockIdx.x] = bsum;
    __threadfence();
    grid.sync();
    double u = 0.0;
    for (unsigned i = threadIdx.x; i < gridDim.x; i += kBlock) u += __ldcg(partial + i);
    const double rho_new = block_sum<kBlock>(u);
    const double beta = rho_new / rho;
    const double ax = y_only ? cy0 * alpha : alpha;
    for (long base = (long)blockIdx.x * kRChunk + threadIdx.x; base < n2; base += (long)gridDim.x * kRChunk) {
        double2 rv[kRUnroll], xv[kRUnroll], pv[kRUnroll];
#pragma unroll
        for (int e = 0; e < kRUnroll; ++e) {
            const long i = base + (long)e * kBlock;
            if (i < n2) { rv[e] = r[i]; xv[e] = x0[i]; pv[e] = p[i]; }
        }
#pragma unroll
        for (int e = 0; e < kRUnroll; ++e) {
            const long i = base + (long)e * kBlock;
            if (i < n2) {
                xv[e].x = fma(ax, pv[e].x, xv[e].x);
                xv[e].y = fma(ax, pv[e].y, xv[e].y);
                pv[e].x = fma(beta, pv[e].x, 1.0 * rv[e].x);
                pv[e].y = fma(beta, pv[e].y, 1.0 * rv[e].y);
                x0[i] = xv[e];
                p[i] = pv[e];
            }
        }
    }
    if (blockIdx.x == 0) {                // the scalar recurrences of all shifts, history, freezing, stop test
        cg_step_alpha(st, pAp);
        __syncthreads();
        cg_step_beta(st, rho_new);
    }
}

// for every shift k updated this iteration:  x_k += alpha_k p_k ;  p_k = zeta_k^new r + beta_k p_k
// ("the heaviest kernel which updates three large arrays").  Work is cut into units of
// (chunk of kShiftChunk elements, shift): unit u -> shift u % nl, chunk u / nl, dealt round-robin to
// the CTAs, so the load per SM is even for any number of active shifts and any lattice size, and the
// CTAs that share a chunk of r run next to each other (L2).  Each thread streams kShiftUnroll
// independent (x, p) pairs per unit.
constexpr int kShiftUnroll = 4;
constexpr int kShiftChunk = kBlock * kShiftUnroll;

__global__ void __launch_bounds__(kBlock)
cg_update_shifts_kernel(long n2, const double2 *__restrict__ ring, double2 *__restrict__ x,
                        double2 *__restrict__ p, long pstride, const CgState *__restrict__ st, int base_only)
{
    pdl_wait();
    pdl_launch_dependents();
    if (st->done_prev) return;
    __shared__ double s_a[kMaxShifts], s_z[kMaxShifts], s_b[kMaxShifts];
    __shared__ long long s_x[kMaxShifts], s_p[kMaxShifts];
    const double2 *__restrict__ r = ring + (long)((st->iter - 1) % st->defer) * n2;   // r of the iteration just done
    const int nl = base_only ? 1 : st->nlist;       // base_only: the shifts k >= 1 are updated by the flush kernel
    if (threadIdx.x < nl) {
        const int k = base_only ? 0 : st->list[threadIdx.x];
        s_a[threadIdx.x] = st->coef_a[k];
        s_z[threadIdx.x] = st->coef_z[k];
        s_b[threadIdx.x] = st->coef_b[k];
        s_x[threadIdx.x] = st->xoff[k];
        s_p[threadIdx.x] = (long long)k * pstride;
    }
    __syncthreads();
    const unsigned nchunk = (unsigned)((n2 + kShiftChunk - 1) / kShiftChunk);
    const unsigned nunit = nchunk * (unsigned)nl;
    for (unsigned u = blockIdx.x; u < nunit; u += gridDim.x) {
        const unsigned c = u / (unsigned)nl, j = u - c * (unsigned)nl;
        const long base = (long)c * kShiftChunk + threadIdx.x;
        double2 *__restrict__ xp = x + s_x[j];
        double2 *__restrict__ pp = p + s_p[j];
        const double a = s_a[j], z = s_z[j], bb = s_b[j];
        double2 rv[kShiftUnroll], xv[kShiftUnroll], pv[kShiftUnroll];
#pragma unroll
        for (int e = 0; e < kShiftUnroll; ++e) {
            const long i = base + (long)e * kBlock;
            if (i < n2) { xv[e] = xp[i]; pv[e] = pp[i]; rv[e] = __ldg(r + i); }
        }
#pragma unroll
        for (int e = 0; e < kShiftUnroll; ++e) {
            const long i = base + (long)e * kBlock;
            if (i < n2) {
                xv[e].x = fma(a, pv[e].x, xv[e].x);
                xv[e].y = fma(a, pv[e].y, xv[e].y);
                pv[e].x = fma(bb, pv[e].x, z * rv[e].x);
                pv[e].y = fma(bb, pv[e].y, z * rv[e].y);
                xp[i] = xv[e];
                pp[i] = pv[e];
            }
        }
    }
}

// Deferred updates of the shifts k >= 1.  Only p_0 is needed inside the iteration (the next matvec acts
// on it); x_k and p_k of the other shifts are needed at the end.  So their updates
//     x_k += alpha_k^(n) p_k ;  p_k = zeta_k^(n) r_n + beta_k^(n) p_k          n = lo + 1 .. hi
// are applied in ONE pass per `defer` iterations from the stored coefficients (CgState::hist_*) and the
// ring of the last `defer` residuals: x_k and p_k then move once per defer iterations instead of once
// per iteration, 96 V/defer bytes per shift and iteration instead of 96 V -- the traffic of "the heaviest
// kernel which updates three large arrays" divided by defer.  Every element sees exactly
// the operations of the undeferred kernel in the same order: the results are bit-identical.
// The kernel flushes the iterations (enq - window, min(enq, iter)]: enq counts the enqueued iterations
// (dead ones included), iter the executed ones; neither is written while this kernel runs.
#ifndef QCD_FLUSH_BLOCK
#define QCD_FLUSH_BLOCK 256
#endif
#ifndef QCD_FLUSH_SHIFTS
#define QCD_FLUSH_SHIFTS 2
#endif
// x_k, p_k of the deferred shifts are touched once per flush: QCD_FLUSH_STREAM = 1 loads and stores them with the
// streaming (evict-first) policy, so that a flush does not push the links and the iteration's vectors out of L2
#ifndef QCD_FLUSH_STREAM
#define QCD_FLUSH_STREAM 0
#endif
#if QCD_FLUSH_STREAM
#define QCD_FLUSH_LD(ptr) __ldcs(ptr)
#define QCD_FLUSH_ST(ptr, v) __stcs(ptr, v)
#else
#define QCD_FLUSH_LD(ptr) (*(ptr))
#define QCD_FLUSH_ST(ptr, v) (*(ptr) = (v))
#endif
constexpr int kFlushBlock = QCD_FLUSH_BLOCK;
constexpr int kFlushShifts = QCD_FLUSH_SHIFTS;   // shifts whose x_k, p_k a thread has in flight at once

__global__ void __launch_bounds__(kFlushBlock)
cg_flush_shifts_kernel(long n2, const double2 *__restrict__ ring, double2 *__restrict__ x,
                       double2 *__restrict__ p, long pstride, const CgState *__restrict__ st, int window)
{
    pdl_wait();
    pdl_launch_dependents();
    const int m = st->defer;
    const int lo = st->enq - window, hi = min(st->enq, st->iter);
    const int cnt = hi - lo;                       // iterations lo + 1 .. hi, 0 <= cnt <= window <= m
    if (cnt <= 0) return;
    __shared__ double s_a[kMaxDefer][kMaxShifts], s_z[kMaxDefer][kMaxShifts], s_b[kMaxDefer][kMaxShifts];
    __shared__ long long s_x[kMaxShifts], s_p[kMaxShifts];
    __shared__ int s_steps[kMaxShifts];            // leading iterations of the window shift j takes part in
    __shared__ int s_n;
    __shared__ int s_all[kMaxShifts], s_map[kMaxShifts];
    const int ns = st->nshift;
    if (threadIdx.x < kMaxShifts) {                // thread k: how many leading iterations of the window shift k is in
        const int k = threadIdx.x;
        int steps = 0;                             // activity only ever ends: a prefix of the window
        if (k >= 1 && k < ns)
            while (steps < cnt && st->hist_on[(lo + steps) % m][k]) ++steps;
        s_all[k] = steps;
    }
    __syncthreads();
    if (threadIdx.x == 0) {                        // compact: the shifts that have anything to do
        int nl = 0;
        for (int k = 1; k < ns; ++k)
            if (s_all[k] > 0) {
                s_map[nl] = k;
                s_steps[nl] = s_all[k];
                s_x[nl] = st->xoff[k];
                s_p[nl] = (long long)k * pstride;
                ++nl;
            }
        s_n = nl;
    }
    __syncthreads();
    for (int idx = threadIdx.x; idx < cnt * s_n; idx += kFlushBlock) {
        const int j = idx / s_n, l = idx - j * s_n, k = s_map[l], slot = (lo + j) % m;
        s_a[j][l] = st->hist_a[slot][k];           // slots beyond a shift's last step are never used
        s_z[j][l] = st->hist_z[slot][k];
        s_b[j][l] = st->hist_b[slot][k];
    }
    __syncthreads();
    const int nl = s_n;
    if (nl == 0) return;
    for (long i = (long)blockIdx.x * kFlushBlock + threadIdx.x; i < n2; i += (long)gridDim.x * kFlushBlock) {
        double2 rv[kMaxDefer];
#pragma unroll
        for (int j = 0; j < kMaxDefer; ++j)
            if (j < cnt) rv[j] = __ldg(ring + (long)((lo + j) % m) * n2 + i);
        for (int l = 0; l < nl; l += kFlushShifts) {       // kFlushShifts shifts in flight per thread
            double2 xv[kFlushShifts], pv[kFlushShifts];
            int steps[kFlushShifts];
#pragma unroll
            for (int s = 0; s < kFlushShifts; ++s) {
                steps[s] = 0;
                if (l + s < nl) {
                    xv[s] = QCD_FLUSH_LD(x + s_x[l + s] + i);
                    pv[s] = QCD_FLUSH_LD(p + s_p[l + s] + i);
                    steps[s] = s_steps[l + s];
                }
            }
#pragma unroll
            for (int j = 0; j < kMaxDefer; ++j) {
#pragma unroll
                for (int s = 0; s < kFlushShifts; ++s) {
                    if (j < steps[s]) {
                        const double a = s_a[j][l + s], z = s_z[j][l + s], b = s_b[j][l + s];
                        xv[s].x = fma(a, pv[s].x, xv[s].x);
                        xv[s].y = fma(a, pv[s].y, xv[s].y);
                        pv[s].x = fma(b, pv[s].x, z * rv[j].x);
                        pv[s].y = fma(b, pv[s].y, z * rv[j].y);
                    }
                }
            }
#pragma unroll
            for (int s = 0; s < kFlushShifts; ++s) {
                if (l + s < nl) {
                    QCD_FLUSH_ST(x + s_x[l + s] + i, xv[s]);
                    QCD_FLUSH_ST(p + s_p[l + s] + i, pv[s]);
                }
            }
        }
    }
}

// y-only form of the shift update (QCD_OPT_Y_ONLY): when only y = sum_k c_k x_k is wanted (eq. 8,
// the heat bath and the action need (M^dag M)^(1/b) phi, not the x_k), the x_k never
// have to exist: x_k += alpha_k p_k turns into y += c_k alpha_k p_k, accumulated in registers over the
// active shifts of an element.  Per active shift the kernel then moves p_k in and out (48 V bytes)
// instead of x_k and p_k (96 V bytes); r and y once per element.
__global__ void __launch_bounds__(kBlock)
cg_update_shifts_y_kernel(long n2, const double2 *__restrict__ ring, double2 *__restrict__ y,
                          double2 *__restrict__ p, long pstride, const CgState *__restrict__ st, int base_only)
{
    pdl_wait();
    pdl_launch_dependents();
    if (st->done_prev) return;
    const double2 *__restrict__ r = ring + (long)((st->iter - 1) % st->defer) * n2;
    __shared__ double s_ca[kMaxShifts], s_z[kMaxShifts], s_b[kMaxShifts];
    __shared__ long long s_p[kMaxShifts];
    const int nl = base_only ? 1 : st->nlist;       // base_only: the shifts k >= 1 are updated by the flush kernel
    if (threadIdx.x < nl) {
        const int k = base_only ? 0 : st->list[threadIdx.x];
        s_ca[threadIdx.x] = st->cy[k] * st->coef_a[k];
        s_z[threadIdx.x] = st->coef_z[k];
        s_b[threadIdx.x] = st->coef_b[k];
        s_p[threadIdx.x] = (long long)k * pstride;
    }
    __syncthreads();
    for (long i = (long)blockIdx.x * kBlock + threadIdx.x; i < n2; i += (long)gridDim.x * kBlock) {
        const double2 rv = __ldg(r + i);
        double2 yv = y[i];
        int j = 0;
        for (; j + 1 < nl; j += 2) {                 // two shifts in flight per thread
            double2 *pa = p + s_p[j] + i, *pb = p + s_p[j + 1] + i;
            double2 va = *pa, vb = *pb;
            yv.x = fma(s_ca[j], va.x, yv.x);
            yv.y = fma(s_ca[j], va.y, yv.y);
            yv.x = fma(s_ca[j + 1], vb.x, yv.x);
            yv.y = fma(s_ca[j + 1], vb.y, yv.y);
            va.x = fma(s_b[j], va.x, s_z[j] * rv.x);
            va.y = fma(s_b[j], va.y, s_z[j] * rv.y);
            vb.x = fma(s_b[j + 1], vb.x, s_z[j + 1] * rv.x);
            vb.y = fma(s_b[j + 1], vb.y, s_z[j + 1] * rv.y);
            *pa = va;
            *pb = vb;
        }
        if (j < nl) {
            double2 *pa = p + s_p[j] + i;
            double2 va = *pa;
            yv.x = fma(s_ca[j], va.x, yv.x);
            yv.y = fma(s_ca[j], va.y, yv.y);
            va.x = fma(s_b[j], va.x, s_z[j] * rv.x);
            va.y = fma(s_b[j], va.y, s_z[j] * rv.y);
            *pa = va;
        }
        y[i] = yv;
    }
}

// Deferred form of the y-only update: y += sum_{k>=1} sum_n c_k alpha_k^(n) p_k^(n) and the p_k recurrences of
// the last `window` iterations in one pass (see cg_flush_shifts_kernel): p_k of the shifts k >= 1 moves
// once per defer iterations, y and the ring of residuals once per flush.
__global__ void __launch_bounds__(kFlushBlock)
cg_flush_shifts_y_kernel(long n2, const double2 *__restrict__ ring, double2 *__restrict__ y,
                         double2 *__restrict__ p, long pstride, const CgState *__restrict__ st, int window)
{
    pdl_wait();
    pdl_launch_dependents();
    const int m = st->defer;
    const int lo = st->enq - window, hi = min(st->enq, st->iter);
    const int cnt = hi - lo;
    if (cnt <= 0) return;
    __shared__ double s_ca[kMaxDefer][kMaxShifts], s_z[kMaxDefer][kMaxShifts], s_b[kMaxDefer][kMaxShifts];
    __shared__ long long s_p[kMaxShifts];
    __shared__ int s_steps[kMaxShifts], s_all[kMaxShifts], s_map[kMaxShifts];
    __shared__ int s_n;
    const int ns = st->nshift;
    if (threadIdx.x < kMaxShifts) {
        const int k = threadIdx.x;
        int steps = 0;
        if (k >= 1 && k < ns)
            while (steps < cnt && st->hist_on[(lo + steps) % m][k]) ++steps;
        s_all[k] = steps;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int nl = 0;
        for (int k = 1; k < ns; ++k)
            if (s_all[k] > 0) {
                s_map[nl] = k;
                s_steps[nl] = s_all[k];
                s_p[nl] = (long long)k * pstride;
                ++nl;
            }
        s_n = nl;
    }
    __syncthreads();
    for (int idx = threadIdx.x; idx < cnt * s_n; idx += kFlushBlock) {
        const int j = idx / s_n, l = idx - j * s_n, k = s_map[l], slot = (lo + j) % m;
        s_ca[j][l] = st->cy[k] * st->hist_a[slot][k];
        s_z[j][l] = st->hist_z[slot][k];
        s_b[j][l] = st->hist_b[slot][k];
    }
    __syncthreads();
    const int nl = s_n;
    if (nl == 0) return;
    for (long i = (long)blockIdx.x * kFlushBlock + threadIdx.x; i < n2; i += (long)gridDim.x * kFlushBlock) {
        double2 rv[kMaxDefer];
#pragma unroll
        for (int j = 0; j < kMaxDefer; ++j)
            if (j < cnt) rv[j] = __ldg(ring + (long)((lo + j) % m) * n2 + i);
        double2 yv = y[i];
        int l = 0;
        for (; l + 1 < nl; l += 2) {                // two shifts in flight per thread
            double2 *pa = p + s_p[l] + i, *pb = p + s_p[l + 1] + i;
            double2 pva = *pa, pvb = *pb;
            const int sa = s_steps[l], sb = s_steps[l + 1];
#pragma unroll
            for (int j = 0; j < kMaxDefer; ++j) {
                if (j < sa) {
                    yv.x = fma(s_ca[j][l], pva.x, yv.x);
                    yv.y = fma(s_ca[j][l], pva.y, yv.y);
                    pva.x = fma(s_b[j][l], pva.x, s_z[j][l] * rv[j].x);
                    pva.y = fma(s_b[j][l], pva.y, s_z[j][l] * rv[j].y);
                }
                if (j < sb) {
                    yv.x = fma(s_ca[j][l + 1], pvb.x, yv.x);
                    yv.y = fma(s_ca[j][l + 1], pvb.y, yv.y);
                    pvb.x = fma(s_b[j][l + 1], pvb.x, s_z[j][l + 1] * rv[j].x);
                    pvb.y = fma(s_b[j][l + 1], pvb.y, s_z[j][l + 1] * rv[j].y);
                }
            }
            *pa = pva; *pb = pvb;
        }
        if (l < nl) {
            double2 *pa = p + s_p[l] + i;
            double2 pva = *pa;
            const int sa = s_steps[l];
#pragma unroll
            for (int j = 0; j < kMaxDefer; ++j) {
                if (j < sa) {
                    yv.x = fma(s_ca[j][l], pva.x, yv.x);
                    yv.y = fma(s_ca[j][l], pva.y, yv.y);
                    pva.x = fma(s_b[j][l], pva.x, s_z[j][l] * rv[j].x);
                    pva.y = fma(s_b[j][l], pva.y, s_z[j][l] * rv[j].y);
                }
            }
            *pa = pva;
        }
        y[i] = yv;
    }
}

struct CombineArgs {
    long long xoff[kMaxShifts];
    double c[kMaxShifts];
    int n;
};

// y = c_0 b + sum_k c_k x_k   (eq. 8; b == nullptr: without the c_0 term)
__global__ void __launch_bounds__(kBlock)
combine_kernel(long n2, const double2 *__restrict__ x, const CombineArgs a, double c0,
               const double2 *__restrict__ b, double2 *__restrict__ y)
{
    pdl_wait();
    pdl_launch_dependents();
    for (long i = (long)blockIdx.x * kBlock + threadIdx.x; i < n2; i += (long)gridDim.x * kBlock) {
        double2 s = make_double2(0.0, 0.0);
        if (b != nullptr) {
            const double2 v = __ldg(b + i);
            s = make_double2(c0 * v.x, c0 * v.y);
        }
#pragma unroll 4
        for (int k = 0; k < a.n; ++k) {
            const double2 v = __ldg(x + a.xoff[k] + i);
            s.x = fma(a.c[k], v.x, s.x);
            s.y = fma(a.c[k], v.y, s.y);
        }
        y[i] = s;
    }
}

// y += c_0 b, in place: the c_0 term of eq. 8 on the y-only path, where y has been accumulated by the
// iteration itself (a kernel of its own: y is read and written through the same, unrestricted pointer)
__global__ void __launch_bounds__(kBlock)
add_c0_kernel(long n2, double c0, const double2 *__restrict__ b, double2 *y)
{
    pdl_wait();
    pdl_launch_dependents();
    for (long i = (long)blockIdx.x * kBlock + threadIdx.x; i < n2; i += (long)gridDim.x * kBlock) {
        const double2 v = __ldg(b + i);
        double2 s = y[i];
        s.x = fma(c0, v.x, s.x);
        s.y = fma(c0, v.y, s.y);
        y[i] = s;
    }
}

// out = b - q ; *result = ||out||^2   (outer residual of the mixed-precision refinement, NEXT-3)
__global__ void __launch_bounds__(kBlock)
residual_kernel(long n2, const double2 *__restrict__ b, const double2 *__restrict__ q, double2 *__restrict__ out,
                double *partial, unsigned *counter, double *result, int Vh, int halo)
{
    pdl_wait();
    pdl_launch_dependents();
    double s = 0.0;
    for (long i = (long)blockIdx.x * kBlock + threadIdx.x; i < n2; i += (long)gridDim.x * kBlock) {
        const double2 bv = __ldg(b + i), qv = __ldg(q + i);
        double2 d = make_double2(bv.x - qv.x, bv.y - qv.y);
        if (halo > 0) {        // slab mode: halo slices are not this rank's
            const int h = (int)(i % Vh);
            if (h < halo || h >= Vh - halo) d = make_double2(0.0, 0.0);
        }
        out[i] = d;
        s += d.x * d.x + d.y * d.y;
    }
    double total;
    if (grid_sum_last_block<kBlock>(s, partial, counter, total))
        if (threadIdx.x == 0) *result = total;
}

}  // namespace

int blas_grid_blocks(long n2)
{
    long b = (n2 + kBlock - 1) / kBlock;
    return (int)(b < kMaxBlocks ? (b > 0 ? b : 1) : kMaxBlocks);
}

int launch_cg_init(long n2, const double2 *b, double2 *r, double2 *p, long pstride, int nshift,
                   double *partial, CgState *st, int Vh, int halo, Launch L)
{
    launch_kernel(cg_init_kernel, blas_grid_blocks(n2), kBlock, L.s, L.pdl, n2, b, r, p, pstride, nshift, partial, st, Vh, halo);
    return 1;
}

int cg_update_r_grid_blocks(long n2)
{
    long b = (n2 + kRChunk - 1) / kRChunk;
    return (int)(b < kRMaxBlocks ? (b > 0 ? b : 1) : kRMaxBlocks);
}

int launch_cg_update_r(long n2, double2 *ring, const double2 *q, const double *pap_partial, int npap,
                       double *partial, CgState *st, unsigned long long loop_handle, Launch L)
{
    const int grid = cg_update_r_grid_blocks(n2);
    if (loop_handle)
        launch_kernel(cg_update_r_kernel<true>, grid, kBlock, L.s, L.pdl, n2, ring, q, pap_partial, npap, partial, st,
                      (cudaGraphConditionalHandle)loop_handle);
    else
        launch_kernel(cg_update_r_kernel<false>, grid, kBlock, L.s, L.pdl, n2, ring, q, pap_partial, npap, partial, st,
                      (cudaGraphConditionalHandle)0);
    return 1;
}

namespace {

__global__ void __launch_bounds__(kBlock)
sum_partials_kernel(const double *__restrict__ partial, int n, double *out)
{
    double t = 0.0;
    for (int i = threadIdx.x; i < n; i += kBlock) t += __ldcg(partial + i);
    const double total = block_sum<kBlock>(t);
    if (threadIdx.x == 0) *out = total;
}

__global__ void __launch_bounds__(kMaxShifts)
cg_scalars_kernel(CgState *st)
{
    if (st->done) return;                 // dead iteration
    cg_step_alpha(st, st->red[0]);
    __syncthreads();
    cg_step_beta(st, st->red[1]);
}

__global__ void cg_after_init_kernel(CgState *st)
{
    const double rho = st->rho;           // all-reduced ||b||^2
    st->rho_b = rho;
    st->done = st->done_prev = rho == 0.0 ? 1 : 0;
}

}  // namespace

int launch_cg_update_r_split(long n2, double2 *ring, const double2 *q, const double *pap, double *partial,
                             CgState *st, Launch L)
{
    launch_kernel(cg_update_r_kernel<false, true>, cg_update_r_grid_blocks(n2), kBlock, L.s, L.pdl, n2, ring, q, pap, 1,
                  partial, st, (cudaGraphConditionalHandle)0);
    return 1;
}

int launch_sum_partials(const double *partial, int n, double *out, Launch L)
{
    launch_kernel(sum_partials_kernel, 1, kBlock, L.s, L.pdl, partial, n, out);
    return 1;
}

int launch_cg_scalars(CgState *st, Launch L)
{
    launch_kernel(cg_scalars_kernel, 1, kMaxShifts, L.s, L.pdl, st);
    return 1;
}

int launch_cg_after_init(CgState *st, Launch L)
{
    launch_kernel(cg_after_init_kernel, 1, 1, L.s, L.pdl, st);
    return 1;
}

// 0 if the cooperative launch is not possible (grid would not be co-resident)
int launch_cg_update_r_base(long n2, double2 *ring, const double2 *q, const double *pap_partial, int npap,
                            double *partial, double2 *x, double2 *p, CgState *st, int y_only, Launch L)
{
    static int max_blocks = -1;
    if (max_blocks < 0) {
        int per_sm = 0, dev = 0, sms = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, cg_update_r_base_kernel, kBlock, 0) != cudaSuccess) per_sm = 0;
        max_blocks = per_sm * sms;
    }
    if (max_blocks <= 0) return 0;
    const int grid = std::min(cg_update_r_grid_blocks(n2), max_blocks);
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3((unsigned)kBlock);
    cfg.stream = L.s;
    cudaLaunchAttribute attr[2];
    unsigned na = 0;
    attr[na].id = cudaLaunchAttributeCooperative;
    attr[na].val.cooperative = 1;
    ++na;
    if (L.pdl) {
        attr[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[na].val.programmaticStreamSerializationAllowed = 1;
        ++na;
    }
    cfg.attrs = attr;
    cfg.numAttrs = na;
    cudaLaunchKernelEx(&cfg, cg_update_r_base_kernel, n2, ring, q, pap_partial, npap, partial, x, p, st, y_only);
    return 1;
}

int launch_cg_update_shifts(long n2, const double2 *ring, double2 *x, double2 *p, long pstride,
                            CgState *st, int base_only, Launch L)
{
    // the number of active shifts is only known on the device: size the grid for all of them
    long units = (n2 + kShiftChunk - 1) / kShiftChunk * (base_only ? 1 : kMaxShifts);
    int grid = (int)(units < 148 * 8 ? (units > 0 ? units : 1) : 148 * 8);
    launch_kernel(cg_update_shifts_kernel, grid, kBlock, L.s, L.pdl, n2, ring, x, p, pstride, st, base_only);
    return 1;
}

int launch_cg_flush_shifts(long n2, const double2 *ring, double2 *x, double2 *p, long pstride,
                           const CgState *st, int window, Launch L)
{
    long blocks = (n2 + kFlushBlock - 1) / kFlushBlock;
    int grid = (int)(blocks < 148 * 8 ? (blocks > 0 ? blocks : 1) : 148 * 8);
    launch_kernel(cg_flush_shifts_kernel, grid, kFlushBlock, L.s, L.pdl, n2, ring, x, p, pstride, st, window);
    return 1;
}

int launch_cg_update_shifts_y(long n2, const double2 *ring, double2 *y, double2 *p, long pstride,
                              CgState *st, int base_only, Launch L)
{
    long blocks = (n2 + kBlock - 1) / kBlock;
    int grid = (int)(blocks < 148 * 8 ? (blocks > 0 ? blocks : 1) : 148 * 8);
    launch_kernel(cg_update_shifts_y_kernel, grid, kBlock, L.s, L.pdl, n2, ring, y, p, pstride, st, base_only);
    return 1;
}

int launch_cg_flush_shifts_y(long n2, const double2 *ring, double2 *y, double2 *p, long pstride,
                             const CgState *st, int window, Launch L)
{
    long blocks = (n2 + kFlushBlock - 1) / kFlushBlock;
    int grid = (int)(blocks < 148 * 8 ? (blocks > 0 ? blocks : 1) : 148 * 8);
    launch_kernel(cg_flush_shifts_y_kernel, grid, kFlushBlock, L.s, L.pdl, n2, ring, y, p, pstride, st, window);
    return 1;
}

int launch_residual(long n2, const double2 *b, const double2 *q, double2 *out, double *partial, unsigned *counter,
                    double *result, int Vh, int halo, Launch L)
{
    launch_kernel(residual_kernel, blas_grid_blocks(n2), kBlock, L.s, L.pdl, n2, b, q, out, partial, counter, result, Vh, halo);
    return 1;
}

int launch_add_c0(long n2, double c0, const double2 *b, double2 *y, Launch L)
{
    launch_kernel(add_c0_kernel, blas_grid_blocks(n2), kBlock, L.s, L.pdl, n2, c0, b, y);
    return 1;
}

int launch_combine(long n2, const double2 *x, const long long *xoff_host, const double *residues,
                   int nshift, double c0, const double2 *b, double2 *y, Launch L)
{
    CombineArgs a;
    a.n = nshift;
    for (int k = 0; k < nshift; ++k) { a.xoff[k] = xoff_host[k]; a.c[k] = residues[k]; }
    launch_kernel(combine_kernel, blas_grid_blocks(n2), kBlock, L.s, L.pdl, n2, x, a, c0, b, y);
    return 1;
}

}  // namespace qcd
