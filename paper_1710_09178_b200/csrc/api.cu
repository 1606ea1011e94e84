// api.cu -- the C ABI of include/qcd.h: context, argument checking, workspace, and the host-side
// driver of the multishift CG (enqueue-only inside the iteration loop; the host only polls a pinned
// copy of the device's `done` flag once per batch, lagged by one batch, to stop enqueuing).
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstddef>
#include <cstdint>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "internal.cuh"

using namespace qcd;

constexpr int kMaxSlabs = 16;  // t-slabs of the pipelined qcd_dslash_host

struct qcd_ctx {
    Geom g{};
    double mass = 0.0;
    cudaStream_t stream = nullptr;
    int device = 0;
    long n2 = 0;              // double2 elements per internal vector = 3*Vh
    size_t vec_bytes = 0;     // bytes of one parity vector (either layout)
    double2 *W = nullptr;     // [2][4][9][Vh] (3-row) or [2][4][6][Vh] (2-row) in the same buffer
    bool gauge_loaded = false;
    int link_rows = 3;        // layout of the LOADED field
    int opt_link_rows = 3;    // layout the next qcd_load_gauge will build
    // workspace (grow-only, freed by qcd_destroy)
    double2 *tmp = nullptr, *q = nullptr, *r = nullptr;
    double2 *p = nullptr;  int p_cap = 0;
    double2 *xws = nullptr; int x_cap = 0;
    double *partial = nullptr;          // per-CTA partial sums of the ticketed reductions
    double *pap_partial = nullptr;      // per-CTA partial sums of <p_0,q>, written by the Dslash, read by the r-update
    CgState *st = nullptr;
    double *results = nullptr;          // device, kMaxShifts doubles
    CgState *h_state = nullptr;         // pinned
    int *h_done = nullptr;              // pinned [2]
    double *h_results = nullptr;        // pinned
    cudaEvent_t ev[2] = {nullptr, nullptr};
    // staging for the *_host entry points
    double *stage_links = nullptr;      // canonical gauge field on device
    double *stage_vec = nullptr;        // one canonical parity vector on device
    double *stage_out = nullptr;        // second one: output side of the pipelined qcd_dslash_host
    cudaStream_t s_in = nullptr, s_out = nullptr;        // copy-in / copy-out streams of that pipeline
    cudaEvent_t ev_pipe[2 * kMaxSlabs + 2] = {};         // [0] start, [1..S] slab uploaded, [S+1..2S] slab computed, last: done
    double2 *hv_a = nullptr, *hv_b = nullptr, *hv_y = nullptr;   // internal vectors
    long launches = 0;
    // coefficients of qcd_apply_pow, cached per (num, den, n, xmin, xmax): the Remez run takes ~1 s
    struct PowFit { int num, den, n; double xmin, xmax, c0, delta; std::vector<double> coef, shift; };
    std::vector<PowFit> pow_cache;
    std::string err;
    // options (qcd_set_option)
    bool opt_pdl = true;                // programmatic dependent launch on every kernel
    int opt_cg_graph = 1;               // 0: plain launches; 1: one captured graph per batch; 2: device-side WHILE loop
    unsigned long long loop_handle = 0; // conditional handle while the body of the loop graph is captured
    bool opt_y_only = false;            // qcd_inv_sqrt / qcd_apply_pow accumulate y directly, no x_k
    int opt_cg_batch = 8;               // iterations enqueued per batch / per graph (rounded up to a multiple of defer)
    // slab (distributed) mode: the lattice of this context is a t-slab with one halo slice
    // on either side; halo fills and sums over the ranks are the caller's (qcd_set_slab)
    bool slab = false;
    qcd_halo_fn halo = nullptr;
    qcd_allreduce_fn allreduce = nullptr;
    void *slab_user = nullptr;
    bool opt_cg_fuse = true;            // QCD_OPT_CG_FUSE: r-update + base-shift update as one cooperative kernel
    int opt_cg_defer = kMaxDefer;       // QCD_OPT_CG_DEFER: iterations per deferred update of the shifts k >= 1
    int cur_defer = 1;                  // the value the solve being enqueued uses (1 for y-only and single-shift solves)
    int r_slots = 0;                    // vectors allocated in the residual ring c->r
    // NEXT-3 (mixed precision): fp32 copy of the three-row links and the buffers of the refinement
    float2 *W32 = nullptr;
    bool links32_loaded = false;
    bool opt_mixed = false;             // QCD_OPT_MIXED: build W32 at the next load; qcd_multishift_cg refines per shift
    int opt_mixed_switch_exp = 5;       // stage 1 stops at 10^-exp
    bool opt_operator_links32 = false;  // qcd_dslash / qcd_mdagm apply the fp32-link operator
    bool use_links32 = false;           // transient: the launches being enqueued use W32
    double2 *mx_r = nullptr, *mx_e = nullptr;
    int opt_sweep_alternate = 1;        // 0 off, 1 (or 2) on
    bool sweep_on = false;              // decided at qcd_load_gauge: even-output Dslash launches walk the tiles
                                        // backwards and the links are loaded with the ordinary (keep) policy
    size_t l2_bytes = 0;
    int opt_keep_mb = 48;               // QCD_OPT_SWEEP_KEEP_MB: link bytes at the end of a sweep left in L2 with ordinary priority
    int opt_dslash_kernel = 0;          // 0: register-staged links (dslash.cu); 1: bulk-copy staged (dslash_bulk.cu)
    int opt_dslash_persist = 0;         // bulk kernel: CTAs per SM of a persistent grid (0: one CTA per tile)
    // cached graph of one batch of CG iterations (valid for exactly the key below)
    cudaGraphExec_t cg_exec = nullptr;  // the entry of cg_cache selected by the last ensure_cg_graph
    cudaStream_t cap_stream = nullptr;  // capture-only stream (never executes work)
    struct CgKey {
        int parity = -1, batch = 0, rows = 0, kern = 0, persist = 0, defer = 0; bool fuse = false; bool pdl = false, apw = false, yonly = false, l32 = false; double mass = 0.0;
        const void *x = nullptr, *p = nullptr, *q = nullptr, *r = nullptr, *tmp = nullptr;
        bool operator==(const CgKey &o) const {
            return parity == o.parity && batch == o.batch && rows == o.rows && kern == o.kern && persist == o.persist && defer == o.defer && fuse == o.fuse && pdl == o.pdl && apw == o.apw && yonly == o.yonly && l32 == o.l32 && mass == o.mass &&
                   x == o.x && p == o.p && q == o.q && r == o.r && tmp == o.tmp;
        }
    };
    struct CgGraph { CgKey key; cudaGraphExec_t exec; long launches; };   // launches: kernels one replay runs
    long cg_exec_launches = 0;          // of the selected graph
    std::vector<CgGraph> cg_cache;      // a few graphs: the mixed-precision solve alternates between two
    // L2 persistence of part of the gauge field (set at qcd_load_gauge; apw_on == false: none)
    cudaAccessPolicyWindow apw{};
    bool apw_on = false;
    long opt_l2_persist_mb = 0;         // QCD_OPT_L2_PERSIST_MB
    Launch L() const { return Launch{stream, opt_pdl && !slab, nullptr}; }
    // Dslash launches: they read links before their PDL wait, so the first one after a gauge load must
    // be fully serialised behind the ingest kernel
    bool fresh_gauge = false;
    Launch Ld() { const bool pdl = opt_pdl && !fresh_gauge && !slab; fresh_gauge = false; return Launch{stream, pdl, apw_on ? &apw : nullptr}; }
};

static std::string g_create_err;

namespace {

qcd_status fail(qcd_ctx *c, qcd_status s, const std::string &msg)
{
    if (c) c->err = msg; else g_create_err = msg;
    return s;
}

#define QCD_CUDA(ctx, call)                                                                    \
    do {                                                                                       \
        cudaError_t e_ = (call);                                                               \
        if (e_ != cudaSuccess)                                                                 \
            return fail(ctx, e_ == cudaErrorMemoryAllocation ? QCD_ENOMEM : QCD_ECUDA,         \
                        std::string(#call) + ": " + cudaGetErrorString(e_));                   \
    } while (0)

template <class T>
cudaError_t dev_alloc(T **p, size_t count) { return cudaMalloc((void **)p, count * sizeof(T)); }

qcd_status check_launch(qcd_ctx *c, const char *what)
{
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(c, QCD_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
    return QCD_OK;
}

// Dslash CTA order (dslash.cu).  Plain lexicographic order is best while one t-slice of CTAs moves
// less link data than L2 can hold behind it (measured on B200: 121.6 us plain vs 122.4-126 grouped at
// 48^3x12, 432 chunks = 69 MB per slice); beyond that the +-t reuse falls out of L2 and groups of 256
// chunks win (64^3x16, 1024 chunks = 163 MB per slice: 380 us vs 398 plain).
int auto_tgroup(const Geom &g) { return g.chunks >= 640 ? 256 : g.chunks; }

// QCD_OPT_L2_PERSIST_MB: keep part of the gauge field in the persisting set-aside of L2, so that
// repeated applies on a lattice a little larger than L2 re-read less from HBM.  Off by default:
// measured on B200 at 32^3x8 it speeds back-to-back two-row Dslash applies up (16.9 -> 12.5 us at
// 48 MB) but does nothing for three-row links (151 MB) and slows the CG down as soon as the
// set-aside takes L2 away from the solver's vectors (3-row: 8.26 -> 8.98 ms at 32 MB, 11.6 at 64).
void setup_l2_window(qcd_ctx *c)
{
    c->apw_on = false;
    const long mb = c->opt_l2_persist_mb;
    if (mb <= 0) return;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, c->device) != cudaSuccess) return;
    size_t persist = std::min((size_t)mb << 20, (size_t)prop.persistingL2CacheMaxSize);
    if (persist == 0 || cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, persist) != cudaSuccess) return;
    const size_t link_bytes = (size_t)c->g.Vh * 2 * 4 * 3 * c->link_rows * sizeof(double2);
    const size_t window = std::min(link_bytes, (size_t)prop.accessPolicyMaxWindowSize);
    c->apw.base_ptr = c->W;
    c->apw.num_bytes = window;
    c->apw.hitRatio = (float)std::min(1.0, (double)persist / (double)window);
    c->apw.hitProp = cudaAccessPropertyPersisting;
    c->apw.missProp = cudaAccessPropertyStreaming;
    c->apw_on = true;
}

// QCD_OPT_SWEEP_ALTERNATE.  D_oe and D_eo read the SAME links (each reads the forward links of its output
// parity and the backward links of the other), and inside M^dag M, the CG and any power iteration they
// alternate.  Walking the lattice in ascending order for odd outputs and in descending order for even
// outputs lets every apply START on the links its predecessor touched LAST.  Those are still in L2 if
// they were loaded with the ordinary priority while the rest of the sweep streamed past them with
// evict-first: the last QCD_OPT_SWEEP_KEEP_MB of link data of every sweep are loaded "keep", everything
// before "streaming" (per-CTA createpolicy operand of the link loads, dslash.cu).  Measured on B200, us per
// apply in back-to-back (D_oe, D_eo) pairs, one direction + all streaming -> alternating + 48 MB kept:
// 32^3x8 20.5 -> 16.0 (two-row 14.8 -> 11.9), 48^3x12 117.5 -> 112, 64^3x16 372.9 -> 367-370; 12-shift
// solve at 32^3x8 5.27 -> 4.81 ms.  Keeping everything (the ordinary policy on all links) gives 18.1 us at
// 32^3x8 and nothing at the larger sizes; 15 MB gives 18.0, 30 MB 16.9, 60 MB 16.2, 90 MB 16.9.  An
// isolated launch behind a flushed L2 pays for it: 29.1 -> 30.7 us at 32^3x8.
void decide_sweep(qcd_ctx *c) { c->sweep_on = c->opt_sweep_alternate != 0; }

// CTAs at the end of a sweep whose links stay in L2 with the ordinary priority: opt_keep_mb of link data
// (a CTA reads 8 links of 128 sites)
int keep_tiles(const qcd_ctx *c)
{
    const long per_tile = 128L * 8 * 3 * c->link_rows * (long)sizeof(double2);
    const long n = (long)c->opt_keep_mb * 1000000L / per_tile;
    return (int)std::min<long>(n, dslash_grid_blocks(c->g));
}

bool bad_parity(int p) { return p != QCD_EVEN && p != QCD_ODD; }

// every device buffer is accessed with 16-byte loads and stores (double2)
bool misaligned(const void *p) { return ((uintptr_t)p & 15u) != 0; }
// [a, a + na) and [b, b + nb) (bytes) share at least one byte
bool overlap(const void *a, size_t na, const void *b, size_t nb)
{
    const uintptr_t x = (uintptr_t)a, y = (uintptr_t)b;
    return x < y + nb && y < x + na;
}

qcd_status ensure_host_staging(qcd_ctx *c)
{
    if (!c->stage_vec) QCD_CUDA(c, cudaMalloc((void **)&c->stage_vec, c->vec_bytes));
    if (!c->hv_a) QCD_CUDA(c, dev_alloc(&c->hv_a, (size_t)c->n2));
    if (!c->hv_b) QCD_CUDA(c, dev_alloc(&c->hv_b, (size_t)c->n2));
    return QCD_OK;
}

qcd_status ensure_cg_workspace(qcd_ctx *c, int nshift, bool need_x)
{
    if (!c->q) {
        QCD_CUDA(c, dev_alloc(&c->q, (size_t)c->n2));
        QCD_CUDA(c, cudaMemsetAsync(c->q, 0, c->vec_bytes, c->stream));   // slab mode: its halo slices are never written
    }
    if (c->r_slots < kMaxDefer) {          // the residual ring (deferred shift updates, blas.cu)
        if (c->r) cudaFree(c->r);
        c->r = nullptr; c->r_slots = 0;
        QCD_CUDA(c, dev_alloc(&c->r, (size_t)c->n2 * kMaxDefer));
        c->r_slots = kMaxDefer;
    }
    if (c->p_cap < nshift) {
        if (c->p) cudaFree(c->p);
        c->p = nullptr; c->p_cap = 0;
        QCD_CUDA(c, dev_alloc(&c->p, (size_t)c->n2 * nshift));
        c->p_cap = nshift;
    }
    if (need_x && c->x_cap < nshift) {
        if (c->xws) cudaFree(c->xws);
        c->xws = nullptr; c->x_cap = 0;
        QCD_CUDA(c, dev_alloc(&c->xws, (size_t)c->n2 * nshift));
        c->x_cap = nshift;
    }
    return QCD_OK;
}

// out = D_{out_parity,other} in, with optional epilogue; counts the launch
qcd_status run_dslash(qcd_ctx *c, int out_parity, const double2 *in, double2 *out,
                      const double2 *src, double coeff, bool coeff_from_state, int dot_mode,
                      bool gated)
{
    DslashParams p{};
    p.W = c->W; p.link_rows = c->link_rows; p.in = in; p.out = out; p.out_parity = out_parity;
    p.W32 = c->W32; p.links32 = c->use_links32 ? 1 : 0;
    p.reverse = c->sweep_on && out_parity == QCD_EVEN ? 1 : 0;
    p.keep_tiles = c->sweep_on ? keep_tiles(c) : 0;
    p.src = src; p.coeff = coeff; p.coeff_from_state = coeff_from_state ? 1 : 0;
    p.mass2 = c->mass * c->mass;
    p.dot_mode = dot_mode; p.partial = c->pap_partial;
    p.st = (gated || dot_mode || coeff_from_state) ? c->st : nullptr;
    if (c->slab) {       // the caller fills the two halo slices of the input; the owned slices 1 .. Nt-2 are computed
        c->halo(c->slab_user, (double *)in, (void *)c->stream);
        Geom g = c->g;
        g.t0 = 1; g.nt_run = g.Nt - 2;
        p.keep_tiles = std::min(p.keep_tiles, dslash_grid_blocks(g));
        c->launches += launch_dslash(g, p, c->Ld());
        return QCD_OK;
    }
    if (c->opt_dslash_kernel == 1 && !c->use_links32) c->launches += launch_dslash_bulk(c->g, p, c->opt_dslash_persist, c->Ld());
    else c->launches += launch_dslash(c->g, p, c->Ld());
    return QCD_OK;
}

// slab mode: sum `count` doubles of the device-resident state over the ranks (stream-ordered)
void slab_allreduce(qcd_ctx *c, double *d_buf, int count) { c->allreduce(c->slab_user, d_buf, count, (void *)c->stream); }
double *state_field(qcd_ctx *c, size_t offset) { return (double *)((char *)c->st + offset); }

// one multishift-CG iteration: 4 kernels, all scalars stay on the device.  With deferred
// shift updates (cur_defer > 1) the fourth kernel updates the base shift only; the caller enqueues
// enqueue_cg_flush after every cur_defer-th iteration.
void enqueue_cg_iteration(qcd_ctx *c, int parity, double2 *x, bool y_only)
{
    // tmp = D_{q,p} p_0 ; q = (m^2 + sigma_0) p_0 - D_{p,q} tmp, <p_0,q> -> alpha, zeta_new
    run_dslash(c, 1 - parity, c->p, c->tmp, nullptr, 0.0, false, 0, true);
    run_dslash(c, parity, c->tmp, c->q, c->p, 0.0, true, 1, true);
    if (c->slab) {       // the two inner products leave the rank between the kernels (reading N4)
        Geom g = c->g;
        g.t0 = 1; g.nt_run = g.Nt - 2;
        double *red = state_field(c, offsetof(CgState, red));
        c->launches += launch_sum_partials(c->pap_partial, dslash_grid_blocks(g), red, c->L());
        slab_allreduce(c, red, 1);                                   // <p_0,q>
        c->launches += launch_cg_update_r_split(c->n2, c->r, c->q, red, c->partial, c->st, c->L());
        slab_allreduce(c, red + 1, 1);                               // ||r'||^2
        c->launches += launch_cg_scalars(c->st, c->L());
        c->launches += launch_cg_update_shifts(c->n2, c->r, x, c->p, c->n2, c->st, c->cur_defer > 1 ? 1 : 0, c->L());
        return;
    }
    const int npap = c->opt_dslash_kernel == 1 && !c->use_links32 ? dslash_bulk_grid_blocks(c->g, c->opt_dslash_persist)
                                               : dslash_grid_blocks(c->g);
    if (c->opt_cg_fuse && c->cur_defer > 1 && c->loop_handle == 0) {
        const int n = launch_cg_update_r_base(c->n2, c->r, c->q, c->pap_partial, npap, c->partial, x, c->p, c->st,
                                              y_only ? 1 : 0, c->L());
        c->launches += n;
        if (n) return;
    }
    c->launches += launch_cg_update_r(c->n2, c->r, c->q, c->pap_partial, npap, c->partial, c->st, c->loop_handle, c->L());
    if (y_only)      // `x` is the single vector y
        c->launches += launch_cg_update_shifts_y(c->n2, c->r, x, c->p, c->n2, c->st, c->cur_defer > 1 ? 1 : 0, c->L());
    else
        c->launches += launch_cg_update_shifts(c->n2, c->r, x, c->p, c->n2, c->st, c->cur_defer > 1 ? 1 : 0, c->L());
}

// the deferred updates of the shifts k >= 1 for the last `window` enqueued iterations
void enqueue_cg_flush(qcd_ctx *c, double2 *x, bool y_only, int window)
{
    if (y_only) c->launches += launch_cg_flush_shifts_y(c->n2, c->r, x, c->p, c->n2, c->st, window, c->L());
    else c->launches += launch_cg_flush_shifts(c->n2, c->r, x, c->p, c->n2, c->st, window, c->L());
}

// `count` iterations with the flushes that belong to them (count is a multiple of cur_defer, or the tail
// of a solve enqueued without graphs)
void enqueue_cg_iterations(qcd_ctx *c, int parity, double2 *x, bool y_only, int count)
{
    const int m = c->cur_defer;
    for (int i = 1; i <= count; ++i) {
        enqueue_cg_iteration(c, parity, x, y_only);
        if (m > 1 && (i % m == 0 || i == count)) enqueue_cg_flush(c, x, y_only, i % m == 0 ? m : i % m);
    }
}

// Capture `batch` iterations into a graph (once per distinct set of buffers, parity and mass);
// batch == 0: the device-side loop graph.
qcd_status ensure_cg_graph(qcd_ctx *c, int parity, double2 *x, int batch, bool y_only)
{
    qcd_ctx::CgKey key;
    key.parity = parity; key.batch = batch; key.rows = c->link_rows; key.kern = c->opt_dslash_kernel; key.persist = c->opt_dslash_persist; key.defer = c->cur_defer; key.fuse = c->opt_cg_fuse; key.pdl = c->opt_pdl; key.apw = c->apw_on; key.yonly = y_only; key.mass = c->mass;
    key.x = x; key.p = c->p; key.q = c->q; key.r = c->r; key.tmp = c->tmp; key.l32 = c->use_links32;
    for (auto &e : c->cg_cache)
        if (e.key == key) { c->cg_exec = e.exec; c->cg_exec_launches = e.launches; return QCD_OK; }
    c->cg_exec = nullptr;
    if (c->cg_cache.size() >= 4) { cudaGraphExecDestroy(c->cg_cache.front().exec); c->cg_cache.erase(c->cg_cache.begin()); }
    if (!c->cap_stream)
        QCD_CUDA(c, cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking));
    cudaStream_t user = c->stream;
    const long launches0 = c->launches;
    c->stream = c->cap_stream;
    cudaError_t e;
    if (batch > 0) {
        e = cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal);
        if (e == cudaSuccess) {
            enqueue_cg_iterations(c, parity, x, y_only, batch);
            cudaGraph_t graph = nullptr;
            e = cudaStreamEndCapture(c->cap_stream, &graph);
            if (e == cudaSuccess) e = cudaGraphInstantiate(&c->cg_exec, graph, 0);
            if (graph) cudaGraphDestroy(graph);
        }
    } else {
        // batch == 0: ONE graph for the whole solve.  A WHILE conditional node whose body is one CG
        // iteration; the r-update's last block sets the condition from the device-side stop test, so
        // the loop ends right after the converging iteration: no dead launches, no host polling.
        cudaGraph_t graph = nullptr;
        cudaGraphConditionalHandle handle = 0;
        e = cudaGraphCreate(&graph, 0);
        if (e == cudaSuccess) e = cudaGraphConditionalHandleCreate(&handle, graph, 1, cudaGraphCondAssignDefault);
        cudaGraphNodeParams np{};
        np.type = cudaGraphNodeTypeConditional;
        np.conditional.handle = handle;
        np.conditional.type = cudaGraphCondTypeWhile;
        np.conditional.size = 1;
        cudaGraphNode_t node = nullptr;
        if (e == cudaSuccess) e = cudaGraphAddNode(&node, graph, nullptr, 0, &np);
        if (e == cudaSuccess) {
            cudaGraph_t body = np.conditional.phGraph_out[0];
            e = cudaStreamBeginCaptureToGraph(c->cap_stream, body, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal);
            if (e == cudaSuccess) {
                c->loop_handle = (unsigned long long)handle;
                enqueue_cg_iterations(c, parity, x, y_only, c->cur_defer);     // body: defer iterations + their flush
                c->loop_handle = 0;
                cudaGraph_t same = nullptr;
                e = cudaStreamEndCapture(c->cap_stream, &same);
            }
        }
        if (e == cudaSuccess) e = cudaGraphInstantiate(&c->cg_exec, graph, 0);
        if (graph) cudaGraphDestroy(graph);
    }
    c->stream = user;
    c->cg_exec_launches = c->launches - launches0;
    c->launches = launches0;          // capturing launches nothing
    if (e != cudaSuccess) {
        c->cg_exec = nullptr;
        return fail(c, QCD_ECUDA, std::string("CG graph capture: ") + cudaGetErrorString(e));
    }
    c->cg_cache.push_back({key, c->cg_exec, c->cg_exec_launches});
    return QCD_OK;
}

}  // namespace

extern "C" {

const char *qcd_version(void) { return "qcd_b200 0.1 (sm_100a)"; }

qcd_status qcd_create(const int dims[4], double mass, void *cuda_stream, qcd_ctx **out)
{
    if (!out) return fail(nullptr, QCD_EINVAL, "qcd_create: out is NULL");
    *out = nullptr;
    if (!dims) return fail(nullptr, QCD_EINVAL, "qcd_create: dims is NULL");
    for (int i = 0; i < 4; ++i)
        if (dims[i] < 2 || (dims[i] & 1))
            return fail(nullptr, QCD_EINVAL, "qcd_create: every extent must be even and >= 2");
    if (!(mass == mass)) return fail(nullptr, QCD_EINVAL, "qcd_create: mass is NaN");
    const long long V = 1LL * dims[0] * dims[1] * dims[2] * dims[3];
    if (V / 2 * 72 >= (1LL << 31))
        return fail(nullptr, QCD_EINVAL, "qcd_create: lattice too large for 32-bit link indexing");

    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess)
        return fail(nullptr, QCD_ECUDA, std::string("qcd_create: no CUDA device: ") + cudaGetErrorString(e));
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, dev);
    if (e != cudaSuccess)
        return fail(nullptr, QCD_ECUDA, std::string("qcd_create: ") + cudaGetErrorString(e));
    if (prop.major != 10)
        return fail(nullptr, QCD_ECUDA, "qcd_create: device is not sm_100 (B200); there is no fallback path");

    qcd_ctx *c = new (std::nothrow) qcd_ctx;
    if (!c) return fail(nullptr, QCD_ENOMEM, "qcd_create: host allocation failed");
    c->device = dev;
    c->l2_bytes = (size_t)prop.l2CacheSize;
    c->mass = mass;
    c->stream = (cudaStream_t)cuda_stream;
    Geom &g = c->g;
    g.Nx = dims[0]; g.Ny = dims[1]; g.Nz = dims[2]; g.Nt = dims[3];
    g.Nxh = g.Nx / 2;
    g.Vh = (int)(V / 2);
    g.sy = g.Nxh; g.sz = g.Nxh * g.Ny; g.st = g.Nxh * g.Ny * g.Nz;
    g.dxh.init(g.Nxh); g.dy.init(g.Ny); g.dz.init(g.Nz);
    g.t0 = 0; g.nt_run = g.Nt;
    g.chunks = dslash_chunks(g);
    g.tgroup = auto_tgroup(g);
    c->n2 = 3L * g.Vh;
    c->vec_bytes = (size_t)c->n2 * sizeof(double2);

    auto cleanup = [&](qcd_status s, const std::string &m) { qcd_destroy(c); return fail(nullptr, s, m); };
    const int nblk = std::max(dslash_grid_blocks(g), blas_grid_blocks(c->n2));
    if (dev_alloc(&c->W, (size_t)72 * g.Vh) != cudaSuccess ||
        dev_alloc(&c->tmp, (size_t)c->n2) != cudaSuccess ||
        dev_alloc(&c->partial, (size_t)nblk * kMultiRhs) != cudaSuccess ||
        dev_alloc(&c->pap_partial, (size_t)dslash_grid_blocks(g)) != cudaSuccess ||
        dev_alloc(&c->st, 1) != cudaSuccess ||
        dev_alloc(&c->results, (size_t)kMaxShifts + 1) != cudaSuccess)
        return cleanup(QCD_ENOMEM, "qcd_create: device allocation failed");
    if (cudaMallocHost((void **)&c->h_state, sizeof(CgState)) != cudaSuccess ||
        cudaMallocHost((void **)&c->h_done, 2 * sizeof(int)) != cudaSuccess ||
        cudaMallocHost((void **)&c->h_results, (kMaxShifts + 1) * sizeof(double)) != cudaSuccess)
        return cleanup(QCD_ENOMEM, "qcd_create: pinned allocation failed");
    if (cudaEventCreateWithFlags(&c->ev[0], cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev[1], cudaEventDisableTiming) != cudaSuccess ||
        cudaMemset(c->st, 0, sizeof(CgState)) != cudaSuccess)
        return cleanup(QCD_ECUDA, "qcd_create: event/memset failed");
    *out = c;
    return QCD_OK;
}

qcd_status qcd_destroy(qcd_ctx *c)
{
    if (!c) return QCD_OK;
    cudaStreamSynchronize(c->stream);
    for (auto &e : c->cg_cache) cudaGraphExecDestroy(e.exec);
    if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
    cudaFree(c->W); cudaFree(c->tmp); cudaFree(c->q); cudaFree(c->r); cudaFree(c->p);
    cudaFree(c->xws); cudaFree(c->partial); cudaFree(c->pap_partial); cudaFree(c->st); cudaFree(c->results);
    if (c->s_in) cudaStreamDestroy(c->s_in);
    if (c->s_out) cudaStreamDestroy(c->s_out);
    for (auto &e : c->ev_pipe) if (e) cudaEventDestroy(e);
    cudaFree(c->stage_out);
    cudaFree(c->stage_links); cudaFree(c->stage_vec); cudaFree(c->hv_a); cudaFree(c->hv_b);
    cudaFree(c->hv_y); cudaFree(c->W32); cudaFree(c->mx_r); cudaFree(c->mx_e);
    if (c->h_state) cudaFreeHost(c->h_state);
    if (c->h_done) cudaFreeHost(c->h_done);
    if (c->h_results) cudaFreeHost(c->h_results);
    for (auto &e : c->ev) if (e) cudaEventDestroy(e);
    delete c;
    return QCD_OK;
}

qcd_status qcd_set_mass(qcd_ctx *c, double mass)
{
    if (!c) return QCD_EINVAL;
    if (!(mass == mass)) return fail(c, QCD_EINVAL, "qcd_set_mass: mass is NaN");
    c->mass = mass;
    return QCD_OK;
}

qcd_status qcd_set_stream(qcd_ctx *c, void *cuda_stream)
{
    if (!c) return QCD_EINVAL;
    c->stream = (cudaStream_t)cuda_stream;
    return QCD_OK;
}

qcd_status qcd_set_option(qcd_ctx *c, int option, long value)
{
    if (!c) return QCD_EINVAL;
    switch (option) {
    case QCD_OPT_PDL: c->opt_pdl = value != 0; return QCD_OK;
    case QCD_OPT_CG_GRAPH:
        if (value < 0 || value > 2) return fail(c, QCD_EINVAL, "qcd_set_option: CG graph mode must be 0, 1 or 2");
        c->opt_cg_graph = (int)value;
        return QCD_OK;
    case QCD_OPT_CG_BATCH:
        if (value < 1 || value > 1024) return fail(c, QCD_EINVAL, "qcd_set_option: batch must be in [1, 1024]");
        c->opt_cg_batch = (int)value;
        return QCD_OK;
    case QCD_OPT_SWEEP_KEEP_MB:
        if (value < 0 || value > 4096) return fail(c, QCD_EINVAL, "qcd_set_option: keep size must be in [0, 4096] MB");
        c->opt_keep_mb = (int)value;
        for (auto &e : c->cg_cache) cudaGraphExecDestroy(e.exec);
        c->cg_cache.clear(); c->cg_exec = nullptr;
        return QCD_OK;
    case QCD_OPT_CG_FUSE: c->opt_cg_fuse = value != 0; return QCD_OK;
    case QCD_OPT_CG_DEFER:
        if (value < 1 || value > kMaxDefer) return fail(c, QCD_EINVAL, "qcd_set_option: defer must be in [1, 8]");
        c->opt_cg_defer = (int)value;
        return QCD_OK;
    case QCD_OPT_TGROUP:
        if (value < 0) return fail(c, QCD_EINVAL, "qcd_set_option: tgroup must be >= 0");
        c->g.tgroup = value == 0 ? auto_tgroup(c->g) : value > c->g.chunks ? c->g.chunks : (int)value;
        for (auto &e : c->cg_cache) cudaGraphExecDestroy(e.exec);   // Geom is baked in
        c->cg_cache.clear(); c->cg_exec = nullptr;
        return QCD_OK;
    case QCD_OPT_Y_ONLY: c->opt_y_only = value != 0; return QCD_OK;
    case QCD_OPT_SWEEP_ALTERNATE:
        if (value < 0 || value > 2) return fail(c, QCD_EINVAL, "qcd_set_option: sweep mode must be 0, 1 or 2");
        c->opt_sweep_alternate = (int)value;
        decide_sweep(c);
        for (auto &e : c->cg_cache) cudaGraphExecDestroy(e.exec);   // baked into the captured launches
        c->cg_cache.clear(); c->cg_exec = nullptr;
        return QCD_OK;
    case QCD_OPT_MIXED: c->opt_mixed = value != 0; return QCD_OK;
    case QCD_OPT_MIXED_SWITCH_EXP:
        if (value < 1 || value > 15) return fail(c, QCD_EINVAL, "qcd_set_option: switch exponent must be in [1, 15]");
        c->opt_mixed_switch_exp = (int)value;
        return QCD_OK;
    case QCD_OPT_OPERATOR_LINKS32: c->opt_operator_links32 = value != 0; return QCD_OK;
    case QCD_OPT_DSLASH_KERNEL:
        if (value != 0 && value != 1) return fail(c, QCD_EINVAL, "qcd_set_option: Dslash kernel must be 0 or 1");
        c->opt_dslash_kernel = (int)value;
        return QCD_OK;
    case QCD_OPT_DSLASH_PERSIST:
        if (value < 0 || value > 8) return fail(c, QCD_EINVAL, "qcd_set_option: CTAs per SM must be in [0, 8]");
        c->opt_dslash_persist = (int)value;
        return QCD_OK;
    case QCD_OPT_L2_PERSIST_MB:
        if (value < 0) return fail(c, QCD_EINVAL, "qcd_set_option: L2 persist size must be >= 0");
        c->opt_l2_persist_mb = value;
        return QCD_OK;
    case QCD_OPT_LINK_ROWS:
        if (value != 2 && value != 3) return fail(c, QCD_EINVAL, "qcd_set_option: link rows must be 2 or 3");
        c->opt_link_rows = (int)value;
        return QCD_OK;
    default: return fail(c, QCD_EINVAL, "qcd_set_option: unknown option");
    }
}

long qcd_vector_doubles(const qcd_ctx *c) { return c ? 2 * c->n2 : 0; }
long qcd_launch_count(const qcd_ctx *c) { return c ? c->launches : 0; }
const char *qcd_last_error(const qcd_ctx *c) { return c ? c->err.c_str() : g_create_err.c_str(); }

qcd_status qcd_load_gauge(qcd_ctx *c, const double *d_links)
{
    if (!c) return QCD_EINVAL;
    if (!d_links || misaligned(d_links))
        return fail(c, QCD_EINVAL, "qcd_load_gauge: NULL or misaligned (16 bytes) links");
    int *flag = &c->st->not_su3;
    QCD_CUDA(c, cudaMemsetAsync(flag, 0, sizeof(int), c->stream));
    c->gauge_loaded = false;
    c->launches += launch_ingest_links(c->g, d_links, c->W, c->opt_link_rows, flag, c->L());
    qcd_status s = check_launch(c, "qcd_load_gauge");
    if (s != QCD_OK) return s;
    if (c->opt_link_rows == 2) {        // the one case in which this call synchronises (see qcd.h)
        QCD_CUDA(c, cudaMemcpyAsync(&c->h_done[0], flag, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
        QCD_CUDA(c, cudaStreamSynchronize(c->stream));
        if (c->h_done[0])
            return fail(c, QCD_EINVAL, "qcd_load_gauge: two-row storage needs links in SU(3); a third row "
                                       "differs from conj(row0 x row1) by more than 1e-10");
    }
    c->links32_loaded = false;
    if (c->opt_mixed) {                 // NEXT-3: fp32 copy of the (three-row) links for the inner operator
        if (!c->W32) QCD_CUDA(c, dev_alloc(&c->W32, (size_t)72 * c->g.Vh));
        c->launches += launch_ingest_links32(c->g, d_links, c->W32, c->L());
        if ((s = check_launch(c, "qcd_load_gauge (fp32 copy)")) != QCD_OK) return s;
        c->links32_loaded = true;
    }
    c->gauge_loaded = true; c->link_rows = c->opt_link_rows; setup_l2_window(c); decide_sweep(c);
    c->fresh_gauge = true;
    return QCD_OK;
}

qcd_status qcd_load_gauge_host(qcd_ctx *c, const double *h_links)
{
    if (!c) return QCD_EINVAL;
    if (!h_links) return fail(c, QCD_EINVAL, "qcd_load_gauge_host: NULL links");
    const size_t bytes = (size_t)144 * c->g.Vh * sizeof(double);   // 72 V doubles
    if (!c->stage_links) QCD_CUDA(c, cudaMalloc((void **)&c->stage_links, bytes));
    QCD_CUDA(c, cudaMemcpyAsync(c->stage_links, h_links, bytes, cudaMemcpyHostToDevice, c->stream));
    qcd_status s = qcd_load_gauge(c, c->stage_links);
    if (s != QCD_OK) return s;
    QCD_CUDA(c, cudaStreamSynchronize(c->stream));
    return QCD_OK;
}

qcd_status qcd_pack(qcd_ctx *c, int parity, const double *d_canon, double *d_internal)
{
    if (!c) return QCD_EINVAL;
    if (bad_parity(parity) || !d_canon || !d_internal || misaligned(d_canon) || misaligned(d_internal) ||
        overlap(d_canon, c->vec_bytes, d_internal, c->vec_bytes))
        return fail(c, QCD_EINVAL, "qcd_pack: bad parity, NULL, misaligned (16 bytes) or overlapping buffers");
    c->launches += launch_pack(c->g, d_canon, (double2 *)d_internal, c->L());
    return check_launch(c, "qcd_pack");
}

qcd_status qcd_unpack(qcd_ctx *c, int parity, const double *d_internal, double *d_canon)
{
    if (!c) return QCD_EINVAL;
    if (bad_parity(parity) || !d_canon || !d_internal || misaligned(d_canon) || misaligned(d_internal) ||
        overlap(d_canon, c->vec_bytes, d_internal, c->vec_bytes))
        return fail(c, QCD_EINVAL, "qcd_unpack: bad parity, NULL, misaligned (16 bytes) or overlapping buffers");
    c->launches += launch_unpack(c->g, (const double2 *)d_internal, d_canon, c->L());
    return check_launch(c, "qcd_unpack");
}

qcd_status qcd_dslash(qcd_ctx *c, int out_parity, const double *d_in, double *d_out)
{
    if (!c) return QCD_EINVAL;
    if (bad_parity(out_parity) || !d_in || !d_out || misaligned(d_in) || misaligned(d_out) ||
        overlap(d_in, c->vec_bytes, d_out, c->vec_bytes))
        return fail(c, QCD_EINVAL, "qcd_dslash: bad parity, NULL, misaligned (16 bytes) or overlapping buffers");
    if (!c->gauge_loaded) return fail(c, QCD_ESTATE, "qcd_dslash: no gauge field loaded");
    if (c->opt_operator_links32 && !c->links32_loaded)
        return fail(c, QCD_ESTATE, "qcd_dslash: QCD_OPT_OPERATOR_LINKS32 needs a gauge field loaded with QCD_OPT_MIXED = 1");
    c->use_links32 = c->opt_operator_links32;
    run_dslash(c, out_parity, (const double2 *)d_in, (double2 *)d_out, nullptr, 0.0, false, 0, false);
    c->use_links32 = false;
    return check_launch(c, "qcd_dslash");
}

qcd_status qcd_set_slab(qcd_ctx *c, int enable, qcd_halo_fn halo, qcd_allreduce_fn allreduce, void *user)
{
    if (!c) return QCD_EINVAL;
    if (enable && (!halo || !allreduce)) return fail(c, QCD_EINVAL, "qcd_set_slab: both callbacks are needed");
    if (enable && c->g.Nt < 4) return fail(c, QCD_EINVAL, "qcd_set_slab: a slab needs two halo slices and at least two owned ones");
    c->slab = enable != 0;
    c->halo = halo; c->allreduce = allreduce; c->slab_user = user;
    if (c->slab && c->q) QCD_CUDA(c, cudaMemsetAsync(c->q, 0, c->vec_bytes, c->stream));   // its halo slices must be zero
    for (auto &e : c->cg_cache) cudaGraphExecDestroy(e.exec);
    c->cg_cache.clear(); c->cg_exec = nullptr;
    return QCD_OK;
}

qcd_status qcd_dslash_range(qcd_ctx *c, int out_parity, const double *d_in, double *d_out, int t0, int nt,
                            const double *d_src, double coeff)
{
    if (!c) return QCD_EINVAL;
    if (bad_parity(out_parity) || !d_in || !d_out || misaligned(d_in) || misaligned(d_out) || misaligned(d_src) ||
        overlap(d_in, c->vec_bytes, d_out, c->vec_bytes) || (d_src && overlap(d_src, c->vec_bytes, d_out, c->vec_bytes)))
        return fail(c, QCD_EINVAL, "qcd_dslash_range: bad parity, NULL, misaligned (16 bytes) or overlapping buffers");
    if (t0 < 0 || nt < 1 || t0 + nt > c->g.Nt)
        return fail(c, QCD_EINVAL, "qcd_dslash_range: need 0 <= t0, 1 <= nt, t0 + nt <= Nt");
    if (!c->gauge_loaded) return fail(c, QCD_ESTATE, "qcd_dslash_range: no gauge field loaded");
    Geom g = c->g;
    g.t0 = t0; g.nt_run = nt;
    DslashParams p{};
    p.W = c->W; p.link_rows = c->link_rows; p.in = (const double2 *)d_in; p.out = (double2 *)d_out;
    p.out_parity = out_parity; p.src = (const double2 *)d_src; p.coeff = coeff;
    p.reverse = c->sweep_on && out_parity == QCD_EVEN ? 1 : 0;
    p.keep_tiles = c->sweep_on ? keep_tiles(c) : 0;
    if (c->opt_dslash_kernel == 1) c->launches += launch_dslash_bulk(g, p, c->opt_dslash_persist, c->Ld());
    else c->launches += launch_dslash(g, p, c->Ld());
    return check_launch(c, "qcd_dslash_range");
}

qcd_status qcd_mdagm(qcd_ctx *c, int parity, const double *d_in, double *d_out)
{
    if (!c) return QCD_EINVAL;
    if (bad_parity(parity) || !d_in || !d_out || misaligned(d_in) || misaligned(d_out) ||
        overlap(d_in, c->vec_bytes, d_out, c->vec_bytes))
        return fail(c, QCD_EINVAL, "qcd_mdagm: bad parity, NULL, misaligned (16 bytes) or overlapping buffers");
    if (!c->gauge_loaded) return fail(c, QCD_ESTATE, "qcd_mdagm: no gauge field loaded");
    if (c->opt_operator_links32 && !c->links32_loaded)
        return fail(c, QCD_ESTATE, "qcd_mdagm: QCD_OPT_OPERATOR_LINKS32 needs a gauge field loaded with QCD_OPT_MIXED = 1");
    const double2 *in = (const double2 *)d_in;
    c->use_links32 = c->opt_operator_links32;
    run_dslash(c, 1 - parity, in, c->tmp, nullptr, 0.0, false, 0, false);
    run_dslash(c, parity, c->tmp, (double2 *)d_out, in, c->mass * c->mass, false, 0, false);
    c->use_links32 = false;
    return check_launch(c, "qcd_mdagm");
}

}  // extern "C"

namespace {

// qcd_multishift_cg with the optional c_0 term of eq. 8: y = c0 b + sum_k residues[k] x_k
qcd_status multishift_cg_impl(qcd_ctx *c, int parity, const double *d_b, int nshift,
                              const double *shifts, const double *residues, double tol,
                              int max_iter, double *d_x, double *d_y, int *iterations,
                              double *true_res, bool with_c0, double c0, bool y_only = false,
                              bool finish = true)
{
    if (!c) return QCD_EINVAL;
    if (bad_parity(parity) || !d_b || !shifts || !residues || !iterations || !true_res)
        return fail(c, QCD_EINVAL, "qcd_multishift_cg: NULL argument or bad parity");
    if (nshift < 1 || nshift > kMaxShifts)
        return fail(c, QCD_EINVAL, "qcd_multishift_cg: nshift must be in [1, QCD_MAX_SHIFTS]");
    if (!(tol > 0.0) || max_iter < 1)
        return fail(c, QCD_EINVAL, "qcd_multishift_cg: tol must be > 0 and max_iter >= 1");
    for (int k = 0; k < nshift; ++k)
        if (!(shifts[k] >= 0.0)) return fail(c, QCD_EINVAL, "qcd_multishift_cg: shifts must be >= 0");
    if (misaligned(d_b) || misaligned(d_x) || misaligned(d_y))
        return fail(c, QCD_EINVAL, "qcd_multishift_cg: device buffers must be 16-byte aligned");
    // x is zeroed before b is read and y is written while b and x are read: no overlap allowed
    if ((d_x && overlap(d_b, c->vec_bytes, d_x, c->vec_bytes * nshift)) ||
        (d_y && overlap(d_b, c->vec_bytes, d_y, c->vec_bytes)) ||
        (d_x && d_y && overlap(d_y, c->vec_bytes, d_x, c->vec_bytes * nshift)))
        return fail(c, QCD_EINVAL, "qcd_multishift_cg: d_b, d_x and d_y must not overlap");
    if (!c->gauge_loaded) return fail(c, QCD_ESTATE, "qcd_multishift_cg: no gauge field loaded");
    y_only = y_only && d_x == nullptr && d_y != nullptr;
    if (c->slab && (y_only || c->use_links32))
        return fail(c, QCD_EINVAL, "qcd_multishift_cg: slab mode supports the plain fp64 solver only");
    qcd_status s = ensure_cg_workspace(c, nshift, d_x == nullptr && !y_only);
    if (s != QCD_OK) return s;

    const long n2 = c->n2;
    cudaStream_t st = c->stream;
    const double2 *b = (const double2 *)d_b;
    // y-only: the "x buffer" of the iteration is the single accumulator y
    double2 *x = y_only ? (double2 *)d_y : d_x ? (double2 *)d_x : c->xws;

    // base system = smallest shift (C12): sort, remember the caller's order
    std::vector<int> order(nshift);
    for (int k = 0; k < nshift; ++k) order[k] = k;
    std::stable_sort(order.begin(), order.end(), [&](int a, int bb) { return shifts[a] < shifts[bb]; });

    CgState &h = *c->h_state;
    QCD_CUDA(c, cudaStreamSynchronize(st));   // h_state may still be in flight from a previous solve
    std::memset(&h, 0, sizeof h);
    h.alpha_old = 1.0; h.beta_old = 0.0;
    h.tol = tol; h.freeze = 0.1;
    h.nshift = nshift; h.max_iter = max_iter;
    // deferred updates of the shifts k >= 1 (blas.cu); pointless for a single shift
    const int defer = nshift == 1 ? 1 : std::max(1, std::min(c->opt_cg_defer, kMaxDefer));
    h.defer = defer;
    c->cur_defer = defer;
    std::vector<long long> xoff_caller(nshift);
    for (int k = 0; k < nshift; ++k) {
        h.sigma[k] = shifts[order[k]];
        h.zeta[k] = h.zeta_old[k] = h.zeta_new[k] = 1.0;
        h.active[k] = 1;
        h.xoff[k] = (long long)(d_x ? order[k] : k) * n2;
        xoff_caller[order[k]] = h.xoff[k];
        h.cy[k] = residues[order[k]];
    }
    h.sigma0 = h.sigma[0];
    QCD_CUDA(c, cudaMemcpyAsync(c->st, &h, sizeof h, cudaMemcpyHostToDevice, st));
    QCD_CUDA(c, cudaMemsetAsync(x, 0, (size_t)n2 * (y_only ? 1 : nshift) * sizeof(double2), st));
    // the initial residual b is slot defer - 1 of the ring: "r after iteration 0"
    c->launches += launch_cg_init(n2, b, c->r + (long)(defer - 1) * n2, c->p, n2, nshift, c->partial, c->st,
                                  c->g.Vh, c->slab ? c->g.st : 0, c->L());

    if (c->slab) {       // ||b||^2 over all ranks; a rank whose part of the source vanishes must still iterate
        slab_allreduce(c, state_field(c, offsetof(CgState, rho)), 1);
        c->launches += launch_cg_after_init(c->st, c->L());
    }

    // iteration loop: enqueue only (one graph replay, or 4 launches per iteration, per batch)
    const int batch = std::max(1, std::min(c->opt_cg_batch, max_iter));
    const bool use_graph = c->opt_cg_graph == 1 && !c->slab;    // slab mode: the callbacks are not captured
    if (c->opt_cg_graph == 2 && !c->slab) {
        if ((s = ensure_cg_graph(c, parity, x, 0, y_only)) != QCD_OK) return s;
        QCD_CUDA(c, cudaGraphLaunch(c->cg_exec, st));     // launch count added below, once iter is known
    } else {
    if (use_graph && (s = ensure_cg_graph(c, parity, x, batch, y_only)) != QCD_OK) return s;
    int enq = 0, cur = 0;
    bool pending = false, finished = false;
    c->h_done[0] = c->h_done[1] = 0;
    while (!finished && enq < max_iter) {
        // a graph always holds `batch` iterations; iterations past max_iter exit early on the device
        const int nb = use_graph ? batch : std::min(batch, max_iter - enq);
        if (use_graph) {
            QCD_CUDA(c, cudaGraphLaunch(c->cg_exec, st));
            c->launches += c->cg_exec_launches;
        } else {
            enqueue_cg_iterations(c, parity, x, y_only, nb);
        }
        enq += nb;
        if (pending) {
            QCD_CUDA(c, cudaEventSynchronize(c->ev[1 - cur]));
            if (c->h_done[1 - cur]) finished = true;
        }
        QCD_CUDA(c, cudaMemcpyAsync(&c->h_done[cur], &c->st->done, sizeof(int), cudaMemcpyDeviceToHost, st));
        QCD_CUDA(c, cudaEventRecord(c->ev[cur], st));
        pending = true;
        cur = 1 - cur;
    }
    }

    // finish (a6): true residuals recomputed from x_k, kMultiRhs shifts per pass over the links;
    // the p_k are dead by now and serve as the tmp vectors.  y = sum_k c_k x_k.
    if (c->slab && finish) {        // true residuals shift by shift: halo fills are per vector; norms summed over the ranks
        if (!c->mx_r) QCD_CUDA(c, dev_alloc(&c->mx_r, (size_t)n2));
        for (int k = 0; k < nshift; ++k) {
            double2 *xk = x + h.xoff[k];
            run_dslash(c, 1 - parity, xk, c->tmp, nullptr, 0.0, false, 0, false);
            run_dslash(c, parity, c->tmp, c->q, xk, c->mass * c->mass + h.sigma[k], false, 0, false);
            c->launches += launch_residual(n2, b, c->q, c->mx_r, c->partial, &c->st->counter, c->results + order[k],
                                           c->g.Vh, c->g.st, c->L());
        }
        slab_allreduce(c, c->results, nshift);
    }
    for (int k0 = 0; k0 < (y_only || !finish || c->slab ? 0 : nshift); k0 += kMultiRhs) {
        const int nb = std::min(kMultiRhs, nshift - k0);
        DslashMultiParams mp{};
        mp.W = c->W; mp.link_rows = c->link_rows; mp.nrhs = nb;
        mp.partial = c->partial; mp.counter = &c->st->counter;
        mp.keep_tiles = c->sweep_on ? keep_tiles(c) : 0;
        mp.out_parity = 1 - parity;                      // tmp_j = D_{q,p} x_j
        mp.reverse = c->sweep_on && mp.out_parity == QCD_EVEN ? 1 : 0;
        mp.in = x; mp.out = c->p;
        for (int j = 0; j < nb; ++j) { mp.in_off[j] = h.xoff[k0 + j]; mp.out_off[j] = (long long)(k0 + j) * n2; }
        c->launches += launch_dslash_multi(c->g, mp, c->Ld());
        mp.out_parity = parity;                          // || b - ((m^2 + sigma_j) x_j - D_{p,q} tmp_j) ||^2
        mp.reverse = c->sweep_on && mp.out_parity == QCD_EVEN ? 1 : 0;
        mp.in = c->p; mp.out = nullptr; mp.src = x; mp.b = b;
        for (int j = 0; j < nb; ++j) {
            mp.in_off[j] = (long long)(k0 + j) * n2;
            mp.src_off[j] = h.xoff[k0 + j];
            mp.coeff[j] = c->mass * c->mass + h.sigma[k0 + j];
            mp.result[j] = c->results + order[k0 + j];
        }
        c->launches += launch_dslash_multi(c->g, mp, c->Ld());
    }
    if (y_only) {
        if (with_c0) c->launches += launch_add_c0(n2, c0, b, x, c->L());      // y += c0 b, in place
    } else if (d_y)
        c->launches += launch_combine(n2, x, xoff_caller.data(), residues, nshift, c0,
                                      with_c0 ? b : nullptr, (double2 *)d_y, c->L());
    s = check_launch(c, "qcd_multishift_cg");
    if (s != QCD_OK) return s;
    QCD_CUDA(c, cudaMemcpyAsync(c->h_results, c->results, nshift * sizeof(double), cudaMemcpyDeviceToHost, st));
    QCD_CUDA(c, cudaMemcpyAsync(&h, c->st, sizeof h, cudaMemcpyDeviceToHost, st));
    QCD_CUDA(c, cudaStreamSynchronize(st));

    *iterations = h.iter;
    if (c->opt_cg_graph == 2) {          // the loop body (defer iterations and their flush) ran ceil(iter/defer) times
        const long bodies = std::max((h.iter + defer - 1) / defer, 1);
        c->launches += bodies * c->cg_exec_launches;
    }
    const double rho_b = h.rho_b;
    for (int k = 0; k < nshift; ++k)
        true_res[k] = rho_b > 0.0 ? std::sqrt(c->h_results[k] / rho_b) : 0.0;
    if (y_only || !finish)      // no x_k to recompute from: the recursion's own estimate |zeta_k| sqrt(rho/rho_b),
        for (int k = 0; k < nshift; ++k)        // and the freezing threshold for the frozen shifts
            true_res[order[k]] = rho_b > 0.0 ? (h.active[k] ? std::fabs(h.zeta[k]) * std::sqrt(h.rho / rho_b)
                                                            : h.freeze * tol) : 0.0;
    const bool converged = rho_b == 0.0 || std::sqrt(h.rho / rho_b) <= tol;
    if (!converged) return fail(c, QCD_ENOTCONV, "qcd_multishift_cg: max_iter reached");
    return QCD_OK;
}

// SURVEY 8(f) NEXT-3 (reading N3; oracle/mixed_precision.py): the mixed-precision
// form of the solve.  Stage 1: the fp64 multishift CG down to the loose tolerance 10^-switch_exp.
// Stage 2: every shift on its own by defect correction -- outer residual with the fp64 operator, inner
// single-shift CG on the fp32-link operator (dslash_kernel<.,.,3,float2>) to
// tau = max(tol ||b|| / (2 ||r||), 1e-2), x_k += e -- until ||b - (A + sigma_k) x_k|| <= tol ||b||.
// `iterations` = stage-1 iterations + all inner iterations.
qcd_status mixed_multishift_cg(qcd_ctx *c, int parity, const double *d_b, int nshift, const double *shifts,
                               const double *residues, double tol, int max_iter, double *d_x, double *d_y,
                               int *iterations, double *true_res)
{
    constexpr int kMaxRounds = 60;
    constexpr double kInnerFloor = 1e-2;
    if (!iterations || !true_res) return fail(c, QCD_EINVAL, "qcd_multishift_cg: NULL argument");
    const double loose = std::max(tol, std::pow(10.0, -(double)c->opt_mixed_switch_exp));
    qcd_status s = multishift_cg_impl(c, parity, d_b, nshift, shifts, residues, loose, max_iter, d_x, nullptr,
                                      iterations, true_res, false, 0.0, false, /*finish=*/false);
    if (s != QCD_OK && s != QCD_ENOTCONV) return s;
    const long n2 = c->n2;
    if (!c->mx_r) QCD_CUDA(c, dev_alloc(&c->mx_r, (size_t)n2));
    if (!c->mx_e) QCD_CUDA(c, dev_alloc(&c->mx_e, (size_t)n2));
    const double rho_b = c->h_state->rho_b;
    std::vector<int> order(nshift);
    for (int k = 0; k < nshift; ++k) order[k] = k;
    std::stable_sort(order.begin(), order.end(), [&](int a, int bb) { return shifts[a] < shifts[bb]; });
    std::vector<long long> xoff(nshift);                  // caller index -> offset of x_k
    for (int k = 0; k < nshift; ++k) xoff[order[k]] = (long long)(d_x ? order[k] : k) * n2;
    double2 *xbase = d_x ? (double2 *)d_x : c->xws;
    const double2 *b = (const double2 *)d_b;
    int total_it = *iterations;
    bool all_ok = true;
    for (int k = 0; k < nshift && rho_b > 0.0; ++k) {
        double2 *xk = xbase + xoff[k];
        const double coeff = c->mass * c->mass + shifts[k];
        for (int round = 0;; ++round) {
            // r = b - ((m^2 + sigma_k) x_k - D_{p,q} D_{q,p} x_k), fp64 links
            run_dslash(c, 1 - parity, xk, c->tmp, nullptr, 0.0, false, 0, false);
            run_dslash(c, parity, c->tmp, c->q, xk, coeff, false, 0, false);
            c->launches += launch_residual(n2, b, c->q, c->mx_r, c->partial, &c->st->counter, c->results, c->g.Vh, 0, c->L());
            if ((s = check_launch(c, "qcd_multishift_cg (mixed)")) != QCD_OK) return s;
            QCD_CUDA(c, cudaMemcpyAsync(c->h_results, c->results, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
            QCD_CUDA(c, cudaStreamSynchronize(c->stream));
            const double rr = c->h_results[0];
            true_res[k] = std::sqrt(rr / rho_b);
            if (true_res[k] <= tol) break;
            if (round == kMaxRounds || total_it >= max_iter) { all_ok = false; break; }
            const double tau = std::max(0.5 * tol / true_res[k], kInnerFloor);
            const double one = 1.0;
            int its = 0;
            double tr_in = 0.0;
            c->use_links32 = true;
            s = multishift_cg_impl(c, parity, (const double *)c->mx_r, 1, &shifts[k], &one, tau,
                                   std::max(1, max_iter - total_it), (double *)c->mx_e, nullptr, &its, &tr_in,
                                   false, 0.0, false, /*finish=*/false);
            c->use_links32 = false;
            if (s != QCD_OK && s != QCD_ENOTCONV) return s;
            total_it += its;
            c->launches += launch_add_c0(n2, 1.0, c->mx_e, xk, c->L());     // x_k += e
        }
    }
    if (rho_b == 0.0)
        for (int k = 0; k < nshift; ++k) true_res[k] = 0.0;
    if (d_y)
        c->launches += launch_combine(n2, xbase, xoff.data(), residues, nshift, 0.0, nullptr, (double2 *)d_y, c->L());
    if ((s = check_launch(c, "qcd_multishift_cg (mixed)")) != QCD_OK) return s;
    QCD_CUDA(c, cudaStreamSynchronize(c->stream));
    *iterations = total_it;
    if (!all_ok) return fail(c, QCD_ENOTCONV, "qcd_multishift_cg (mixed): max_iter or the round limit reached");
    return QCD_OK;
}

}  // namespace

extern "C" {

qcd_status qcd_multishift_cg(qcd_ctx *c, int parity, const double *d_b, int nshift,
                             const double *shifts, const double *residues, double tol,
                             int max_iter, double *d_x, double *d_y, int *iterations,
                             double *true_res)
{
    if (c && c->opt_mixed && c->links32_loaded)
        return mixed_multishift_cg(c, parity, d_b, nshift, shifts, residues, tol, max_iter, d_x, d_y,
                                   iterations, true_res);
    return multishift_cg_impl(c, parity, d_b, nshift, shifts, residues, tol, max_iter, d_x, d_y,
                              iterations, true_res, false, 0.0);
}

qcd_status qcd_inv_sqrt_coeffs(int n, double xmin, double xmax, double *c0, double *coef,
                               double *shift, double *delta)
{
    if (!c0 || !coef || !shift)
        return fail(nullptr, QCD_EINVAL, "qcd_inv_sqrt_coeffs: NULL output");
    const int rc = zolotarev_inv_sqrt(n, xmin, xmax, c0, coef, shift, delta);
    if (rc == 2)
        return fail(nullptr, QCD_ENOTCONV, "qcd_inv_sqrt_coeffs: a coefficient is not representable in "
                                           "double precision for this n and interval");
    if (rc != 0)
        return fail(nullptr, QCD_EINVAL,
                    "qcd_inv_sqrt_coeffs: need 1 <= n <= QCD_MAX_SHIFTS and 0 < xmin < xmax");
    return QCD_OK;
}

qcd_status qcd_pow_coeffs(int num, int den, int n, double xmin, double xmax, double *c0,
                          double *coef, double *shift, double *delta)
{
    if (!c0 || !coef || !shift) return fail(nullptr, QCD_EINVAL, "qcd_pow_coeffs: NULL output");
    if (den != 0 && 2 * num == -den)                 // alpha = -1/2: the closed form
        return qcd_inv_sqrt_coeffs(n, xmin, xmax, c0, coef, shift, delta);
    const int rc = remez_pow(num, den, n, xmin, xmax, c0, coef, shift, delta);
    if (rc == 1)
        return fail(nullptr, QCD_EINVAL, "qcd_pow_coeffs: need 0 < |num/den| < 1, 1 <= n <= "
                                         "QCD_MAX_SHIFTS and 0 < xmin < xmax");
    if (rc != 0) return fail(nullptr, QCD_ENOTCONV, "qcd_pow_coeffs: the Remez iteration did not converge");
    return QCD_OK;
}

qcd_status qcd_apply_pow(qcd_ctx *c, int parity, const double *d_phi, int num, int den, int n,
                         double xmin, double xmax, double tol, int max_iter, double *d_out,
                         int *iterations, double *true_res, double *delta)
{
    if (!c) return QCD_EINVAL;
    if (!d_out || !d_phi || overlap(d_phi, c->vec_bytes, d_out, c->vec_bytes))
        return fail(c, QCD_EINVAL, "qcd_apply_pow: NULL or overlapping d_phi / d_out");
    const qcd_ctx::PowFit *fit = nullptr;
    for (const auto &f : c->pow_cache)
        if (f.num == num && f.den == den && f.n == n && f.xmin == xmin && f.xmax == xmax) fit = &f;
    if (!fit) {
        qcd_ctx::PowFit f{num, den, n, xmin, xmax, 0.0, 0.0, {}, {}};
        f.coef.resize(kMaxShifts); f.shift.resize(kMaxShifts);
        const qcd_status s = qcd_pow_coeffs(num, den, n, xmin, xmax, &f.c0, f.coef.data(), f.shift.data(), &f.delta);
        if (s != QCD_OK) return fail(c, s, qcd_last_error(nullptr));
        if (c->pow_cache.size() >= 16) c->pow_cache.erase(c->pow_cache.begin());
        c->pow_cache.push_back(std::move(f));
        fit = &c->pow_cache.back();
    }
    if (delta) *delta = fit->delta;
    return multishift_cg_impl(c, parity, d_phi, n, fit->shift.data(), fit->coef.data(), tol, max_iter,
                              nullptr, d_out, iterations, true_res, true, fit->c0, c->opt_y_only);
}

qcd_status qcd_inv_sqrt(qcd_ctx *c, int parity, const double *d_phi, int n, double xmin,
                        double xmax, double tol, int max_iter, double *d_out, int *iterations,
                        double *true_res, double *delta)
{
    if (!c) return QCD_EINVAL;
    if (!d_out || !d_phi || overlap(d_phi, c->vec_bytes, d_out, c->vec_bytes))
        return fail(c, QCD_EINVAL, "qcd_inv_sqrt: NULL or overlapping d_phi / d_out");
    double c0, coef[kMaxShifts], shift[kMaxShifts];
    const qcd_status cs = qcd_inv_sqrt_coeffs(n, xmin, xmax, &c0, coef, shift, delta);
    if (cs != QCD_OK) return fail(c, cs, qcd_last_error(nullptr));
    return multishift_cg_impl(c, parity, d_phi, n, shift, coef, tol, max_iter, nullptr, d_out,
                              iterations, true_res, true, c0, c->opt_y_only);
}

qcd_status qcd_dslash_host(qcd_ctx *c, int out_parity, const double *h_in, double *h_out)
{
    if (!c) return QCD_EINVAL;
    if (c->slab) return fail(c, QCD_EINVAL, "qcd_dslash_host: not available in slab mode (qcd_set_slab)");
    if (bad_parity(out_parity) || !h_in || !h_out)
        return fail(c, QCD_EINVAL, "qcd_dslash_host: bad argument");
    if (!c->gauge_loaded) return fail(c, QCD_ESTATE, "qcd_dslash_host: no gauge field loaded");
    qcd_status s = ensure_host_staging(c);
    if (s != QCD_OK) return s;
    // Pipeline over t-slabs: a slab of the canonical vector is one contiguous range of sites, and
    // the stencil of slab i needs slabs i-1, i, i+1 only.  Upload + pack on one stream, Dslash +
    // unpack of a slab on the context's stream as soon as its neighbours have arrived, download on a
    // third stream: the PCIe link runs in both directions at once and the kernels hide behind it.
    // Slabs: the largest divisor of Nt (at most kMaxSlabs) that keeps a slab at 1.5 MB or more: below
    // that the ~6 API calls per slab cost more host time than the transfer they overlap.  The last
    // three slabs can only be computed after the last upload, so more slabs mean a shorter tail.
    int S = 1;
    for (int cand = kMaxSlabs; cand >= 3; --cand)
        if (c->g.Nt % cand == 0 && c->vec_bytes / cand >= (3u << 19)) { S = cand; break; }
    if (S < 3) {                                    // too few t-slices, or too small to be worth it
        QCD_CUDA(c, cudaMemcpyAsync(c->stage_vec, h_in, c->vec_bytes, cudaMemcpyHostToDevice, c->stream));
        if ((s = qcd_pack(c, 1 - out_parity, c->stage_vec, (double *)c->hv_a)) != QCD_OK) return s;
        if ((s = qcd_dslash(c, out_parity, (double *)c->hv_a, (double *)c->hv_b)) != QCD_OK) return s;
        if ((s = qcd_unpack(c, out_parity, (double *)c->hv_b, c->stage_vec)) != QCD_OK) return s;
        QCD_CUDA(c, cudaMemcpyAsync(h_out, c->stage_vec, c->vec_bytes, cudaMemcpyDeviceToHost, c->stream));
        QCD_CUDA(c, cudaStreamSynchronize(c->stream));
        return QCD_OK;
    }
    if (!c->stage_out) QCD_CUDA(c, cudaMalloc((void **)&c->stage_out, c->vec_bytes));
    if (!c->s_in) QCD_CUDA(c, cudaStreamCreateWithFlags(&c->s_in, cudaStreamNonBlocking));
    if (!c->s_out) QCD_CUDA(c, cudaStreamCreateWithFlags(&c->s_out, cudaStreamNonBlocking));
    for (int i = 0; i < 2 * S + 2; ++i)
        if (!c->ev_pipe[i]) QCD_CUDA(c, cudaEventCreateWithFlags(&c->ev_pipe[i], cudaEventDisableTiming));
    cudaEvent_t ev_start = c->ev_pipe[0], ev_done = c->ev_pipe[2 * S + 1];
    cudaEvent_t *ev_up = &c->ev_pipe[1], *ev_cmp = &c->ev_pipe[1 + S];
    const int nts = c->g.Nt / S;                    // t-slices per slab
    const int hs = nts * c->g.st;                   // sites per slab
    const size_t slab_doubles = (size_t)hs * 6, slab_bytes = slab_doubles * sizeof(double);
    const Launch Lin{c->s_in, c->opt_pdl, nullptr};
    QCD_CUDA(c, cudaEventRecord(ev_start, c->stream));      // order after earlier work on the user's stream
    QCD_CUDA(c, cudaStreamWaitEvent(c->s_in, ev_start, 0));
    QCD_CUDA(c, cudaStreamWaitEvent(c->s_out, ev_start, 0));
    for (int i = 0; i < S; ++i) {
        QCD_CUDA(c, cudaMemcpyAsync(c->stage_vec + i * slab_doubles, h_in + i * slab_doubles, slab_bytes,
                                    cudaMemcpyHostToDevice, c->s_in));
        c->launches += launch_pack(c->g, c->stage_vec, c->hv_a, Lin, i * hs, (i + 1) * hs);
        QCD_CUDA(c, cudaEventRecord(ev_up[i], c->s_in));
    }
    for (int n = 0; n < S; ++n) {
        const int i = n < S - 1 ? n + 1 : 0;         // slabs 1 .. S-1, then slab 0 (it needs slab S-1)
        const int need = i == 0 ? S - 1 : std::min(i + 1, S - 1);   // uploads complete in order
        QCD_CUDA(c, cudaStreamWaitEvent(c->stream, ev_up[need], 0));
        Geom g = c->g;
        g.t0 = i * nts; g.nt_run = nts;
        DslashParams p{};
        p.W = c->W; p.link_rows = c->link_rows; p.in = c->hv_a; p.out = c->hv_b; p.out_parity = out_parity;
        if (c->opt_dslash_kernel == 1) c->launches += launch_dslash_bulk(g, p, c->opt_dslash_persist, c->Ld());
        else c->launches += launch_dslash(g, p, c->Ld());
        c->launches += launch_unpack(c->g, c->hv_b, c->stage_out, c->L(), i * hs, (i + 1) * hs);
        QCD_CUDA(c, cudaEventRecord(ev_cmp[i], c->stream));
        QCD_CUDA(c, cudaStreamWaitEvent(c->s_out, ev_cmp[i], 0));
        QCD_CUDA(c, cudaMemcpyAsync(h_out + i * slab_doubles, c->stage_out + i * slab_doubles, slab_bytes,
                                    cudaMemcpyDeviceToHost, c->s_out));
    }
    QCD_CUDA(c, cudaEventRecord(ev_done, c->s_out));
    QCD_CUDA(c, cudaStreamWaitEvent(c->stream, ev_done, 0));
    if ((s = check_launch(c, "qcd_dslash_host")) != QCD_OK) return s;
    QCD_CUDA(c, cudaStreamSynchronize(c->stream));
    return QCD_OK;
}

qcd_status qcd_mdagm_host(qcd_ctx *c, int parity, const double *h_in, double *h_out)
{
    if (!c) return QCD_EINVAL;
    if (c->slab) return fail(c, QCD_EINVAL, "qcd_mdagm_host: not available in slab mode (qcd_set_slab)");
    if (bad_parity(parity) || !h_in || !h_out)
        return fail(c, QCD_EINVAL, "qcd_mdagm_host: bad argument");
    qcd_status s = ensure_host_staging(c);
    if (s != QCD_OK) return s;
    QCD_CUDA(c, cudaMemcpyAsync(c->stage_vec, h_in, c->vec_bytes, cudaMemcpyHostToDevice, c->stream));
    if ((s = qcd_pack(c, parity, c->stage_vec, (double *)c->hv_a)) != QCD_OK) return s;
    if ((s = qcd_mdagm(c, parity, (double *)c->hv_a, (double *)c->hv_b)) != QCD_OK) return s;
    if ((s = qcd_unpack(c, parity, (double *)c->hv_b, c->stage_vec)) != QCD_OK) return s;
    QCD_CUDA(c, cudaMemcpyAsync(h_out, c->stage_vec, c->vec_bytes, cudaMemcpyDeviceToHost, c->stream));
    QCD_CUDA(c, cudaStreamSynchronize(c->stream));
    return QCD_OK;
}

qcd_status qcd_multishift_cg_host(qcd_ctx *c, int parity, const double *h_b, int nshift,
                                  const double *shifts, const double *residues, double tol,
                                  int max_iter, double *h_x, double *h_y, int *iterations,
                                  double *true_res)
{
    if (!c) return QCD_EINVAL;
    if (c->slab) return fail(c, QCD_EINVAL, "qcd_multishift_cg_host: not available in slab mode (qcd_set_slab)");
    if (!h_b) return fail(c, QCD_EINVAL, "qcd_multishift_cg_host: NULL source");
    if (nshift < 1 || nshift > kMaxShifts)
        return fail(c, QCD_EINVAL, "qcd_multishift_cg_host: nshift must be in [1, QCD_MAX_SHIFTS]");
    qcd_status s = ensure_host_staging(c);
    if (s != QCD_OK) return s;
    if ((s = ensure_cg_workspace(c, nshift, true)) != QCD_OK) return s;
    if (!c->hv_y) QCD_CUDA(c, dev_alloc(&c->hv_y, (size_t)c->n2));
    QCD_CUDA(c, cudaMemcpyAsync(c->stage_vec, h_b, c->vec_bytes, cudaMemcpyHostToDevice, c->stream));
    if ((s = qcd_pack(c, parity, c->stage_vec, (double *)c->hv_a)) != QCD_OK) return s;
    qcd_status solve = qcd_multishift_cg(c, parity, (double *)c->hv_a, nshift, shifts, residues, tol,
                                         max_iter, nullptr, (double *)c->hv_y, iterations, true_res);
    if (solve != QCD_OK && solve != QCD_ENOTCONV) return solve;
    if (h_x) {
        // workspace x is in sorted-shift order; return it in the caller's order
        std::vector<int> order(nshift);
        for (int k = 0; k < nshift; ++k) order[k] = k;
        std::stable_sort(order.begin(), order.end(), [&](int a, int bb) { return shifts[a] < shifts[bb]; });
        for (int k = 0; k < nshift; ++k) {
            if ((s = qcd_unpack(c, parity, (double *)(c->xws + (long)k * c->n2), c->stage_vec)) != QCD_OK) return s;
            QCD_CUDA(c, cudaMemcpyAsync(h_x + (size_t)order[k] * 2 * c->n2, c->stage_vec, c->vec_bytes,
                                        cudaMemcpyDeviceToHost, c->stream));
        }
    }
    if (h_y) {
        if ((s = qcd_unpack(c, parity, (double *)c->hv_y, c->stage_vec)) != QCD_OK) return s;
        QCD_CUDA(c, cudaMemcpyAsync(h_y, c->stage_vec, c->vec_bytes, cudaMemcpyDeviceToHost, c->stream));
    }
    QCD_CUDA(c, cudaStreamSynchronize(c->stream));
    return solve;
}

}  // extern "C"
