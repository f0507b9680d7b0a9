// Solving phase, host side: queue of (field, scale) right-hand sides, K columns in flight,
// CUDA-graph iteration loop polled every `check_every` iterations, converged columns finalised and refilled
// from the queue.  The device code is in kernels.cuh.
#include <algorithm>
#include <cmath>
#include <cstddef>
#include <cstring>
#include <vector>

#include "kernels.cuh"

namespace ifl {
namespace {

constexpr int MAX_RHS = 65536;
constexpr int64_t MG_DEVICE_TURNOVER_ROWS = 400000;   // see solve_all
constexpr int MAX_BLOCKS_PER_SM = 8;

struct Workspace {
    Ctrl* ctrl;
    double* partials;
    double *x, *z, *p0, *p1, *q, *t, *t2;
    double *energy, *relres, *ells, *k_mid, *E, *epair;
    int32_t *iters, *status;
    QEntry* queue;    // right-hand sides of the multigrid stream, read by the turnover on the device (k_turn_plan)
    void* mg_extra;   // buffers of the multigrid path (mg_solve.cuh), NULL if the handle has no hierarchy
    size_t bytes;
};

inline size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }
inline size_t mg_extra_bytes(const if_mesh_s* h, int order_n);   // mg_solve.cuh (included below)

Workspace layout_workspace(const if_mesh_s* h, int order_n, int batch, void* base) {
    Workspace w{};
    char* p = static_cast<char*>(base);
    size_t off = 0;
    auto take = [&](size_t bytes) { void* r = p ? p + off : nullptr; off += align_up(bytes); return r; };
    const size_t vec = (size_t)h->n_vert * batch * sizeof(double);
    const size_t gmax = (size_t)h->n_sm * MAX_BLOCKS_PER_SM;
    w.ctrl = (Ctrl*)take(sizeof(Ctrl));
    w.partials = (double*)take(3 * gmax * KMAX * sizeof(double));
    w.x = (double*)take(vec);
    w.z = (double*)take(vec);
    w.p0 = (double*)take(vec);
    w.p1 = (double*)take(vec);
    w.q = (double*)take(vec);
    w.t = order_n >= 2 ? (double*)take(vec) : nullptr;
    w.t2 = order_n >= 3 ? (double*)take(vec) : nullptr;
    w.energy = (double*)take(MAX_RHS * sizeof(double));
    w.relres = (double*)take(MAX_RHS * sizeof(double));
    w.ells = (double*)take(MAX_RHS * sizeof(double));
    w.k_mid = (double*)take(MAX_RHS * sizeof(double));
    w.E = (double*)take(MAX_RHS * sizeof(double));
    w.epair = (double*)take(MAX_RHS * sizeof(double));
    w.iters = (int32_t*)take(MAX_RHS * sizeof(int32_t));
    w.status = (int32_t*)take(MAX_RHS * sizeof(int32_t));
    w.mg_extra = nullptr;
    w.queue = nullptr;
    if (batch == KMAX && h->mg_levels > 1) {
        w.queue = (QEntry*)take(MAX_RHS * sizeof(QEntry));
        w.mg_extra = take(mg_extra_bytes(h, order_n));
    }
    w.bytes = off;
    return w;
}

enum Job { JOB_FILTER, JOB_SPECTRUM, JOB_APPLY };

struct Rhs { double ell; int f; int j; };

// persistent grids: one wave of resident blocks, sized from the real occupancy of each kernel
struct Grids { int plain, cga, cgb, update, stream; };
struct MgGrids { int ax = 0, mgr = 0, mgr0 = 0; };   // level-0 kernels of the multigrid cycle

struct Run {
    const if_mesh_s* h;
    MeshView m;
    Workspace w;
    cudaStream_t st;
    int order_n;
    Options opt;
    Grids g;
    bool vec = false;  // vector filter: columns (2i, 2i+1) are the (u, v) of one coupled system (IF_FLAG_VECTOR)
    bool mg = false;   // this phase runs multigrid-preconditioned CG (mg_solve.cuh) instead of Jacobi-PCG
    MgGrids mgg;
    int mg_nu[3] = {1, 1, 2};   // Jacobi sweeps per side of the V cycle on the mesh, on level 1, below (mg_solve.cuh)
    const void* mgb = nullptr;  // MgBuffers of the phase in progress once the stream's tail has been compacted (mg_buffers)
};

template <class Kern>
int resident_grid(Kern kern, size_t smem, int n_sm, int64_t work_items, int* grid, int block = BLOCK) {
    if (smem > 0)   // static + dynamic shared memory may pass 48 KB: always opt in
        IF_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    IF_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, block, smem));
    if (occ < 1) {
        fprintf(stderr, "[implicit_filter] kernel does not fit an SM (dynamic shared memory %zu bytes)\n", smem);
        return IF_ECUDA;
    }
    occ = std::min(occ, MAX_BLOCKS_PER_SM);
    *grid = (int)std::max<int64_t>(1, std::min<int64_t>(work_items, (int64_t)n_sm * occ));
    return IF_OK;
}

template <int K, bool VEC>
int setup_grids_v(Run& r) {
    const int64_t nv = r.h->n_vert;
    const int n_sm = r.h->n_sm;
    const int64_t tiles = (nv + TILE_ROWS - 1) / TILE_ROWS;
    const int64_t passes = (nv + BLOCK / (K / 2) - 1) / (BLOCK / (K / 2));
    int rc;
    if ((rc = resident_grid(k_spmm<K, MODE_PLAIN, VEC>, TileSmem<K, MODE_PLAIN, VEC>::bytes, n_sm, tiles, &r.g.plain, SpmmCfg<K, MODE_PLAIN>::NT))) return rc;
    if (r.order_n == 1) {
        if ((rc = resident_grid(k_spmm<K, MODE_CG1, VEC>, TileSmem<K, MODE_CG1, VEC>::bytes, n_sm, tiles, &r.g.cga, SpmmCfg<K, MODE_CG1>::NT))) return rc;
    } else {
        if ((rc = resident_grid(k_spmm<K, MODE_CG2A, VEC>, TileSmem<K, MODE_CG2A, VEC>::bytes, n_sm, tiles, &r.g.cga, SpmmCfg<K, MODE_CG2A>::NT))) return rc;
    }
    if ((rc = resident_grid(k_spmm<K, MODE_CG2B, VEC>, TileSmem<K, MODE_CG2B, VEC>::bytes, n_sm, tiles, &r.g.cgb, SpmmCfg<K, MODE_CG2B>::NT))) return rc;
    if ((rc = resident_grid(k_update<K>, 0, n_sm, passes, &r.g.update))) return rc;
    r.g.stream = (int)std::max<int64_t>(1, std::min<int64_t>(passes, (int64_t)n_sm * 4));
    return IF_OK;
}
template <int K>
int setup_grids(Run& r) { return r.vec ? setup_grids_v<K, true>(r) : setup_grids_v<K, false>(r); }

template <int K, int MODE>
int launch_spmm(const Run& r, int grid, const SpmmArgs& a) {
    // the vector filter's variants: every mode of the Jacobi path, and the level-0 kernels of the multigrid cycle for
    // (smoothing and residuals on the coupled operator, mg_solve.cuh)
    constexpr bool CG_MODE = MODE == MODE_PLAIN || MODE == MODE_CG1 || MODE == MODE_CG2A || MODE == MODE_CG2B ||
                             MODE == MODE_AX || MODE == MODE_MGR || MODE == MODE_MGR0;
    if constexpr (CG_MODE) {
        if (r.vec) {
            k_spmm<K, MODE, true><<<grid, SpmmCfg<K, MODE>::NT, TileSmem<K, MODE, true>::bytes, r.st>>>(r.m, r.w.ctrl, r.w.partials, a);
            IF_LAUNCH_CHECK();
            return IF_OK;
        }
    }
    k_spmm<K, MODE><<<grid, SpmmCfg<K, MODE>::NT, TileSmem<K, MODE>::bytes, r.st>>>(r.m, r.w.ctrl, r.w.partials, a);
    IF_LAUNCH_CHECK();
    return IF_OK;
}

// Events recorded (as external event-record nodes) between the kernel groups of ONE iteration of a captured graph, so
// that the per-launch duration of every group is measured live on the launching stream (if_stats).  mark(g) closes an
// interval that belongs to group g (the first mark only opens one).
constexpr int TIMER_GROUPS = 8;
struct IterTimer {
    static constexpr int MAXE = 40;
    cudaEvent_t ev[MAXE] = {};
    int gid[MAXE] = {};
    int n = 0, created = 0;
    int create() {
        for (created = 0; created < MAXE; ++created) IF_CUDA_TRY(cudaEventCreate(&ev[created]));
        return IF_OK;
    }
    void destroy() {
        for (int i = 0; i < created; ++i) cudaEventDestroy(ev[i]);
        created = n = 0;
    }
    int mark(cudaStream_t st, int g) {
        if (n >= created) return IF_OK;
        gid[n] = g;
        IF_CUDA_TRY(cudaEventRecordWithFlags(ev[n], st, cudaEventRecordExternal));
        ++n;
        return IF_OK;
    }
};

}  // namespace
}  // namespace ifl
#include "mg_solve.cuh"
namespace ifl {
namespace {

// `count` more factors t <- M^-1 S t of the higher-order operators, alternating between w.t and w.t2; *t = the result
template <int K>
int more_factors(const Run& r, int count, double** t) {
    int rc;
    for (int k = 0; k < count; ++k) {
        double* dst = *t == r.w.t ? r.w.t2 : r.w.t;
        SpmmArgs f{*t, nullptr, nullptr, dst, nullptr, 1, 0};
        if ((rc = launch_spmm<K, MODE_PLAIN>(r, r.g.plain, f))) return rc;
        *t = dst;
    }
    return IF_OK;
}

// One CG iteration: kernel A (two launches for n = 2) and kernel B.  The direction buffers are picked on the device
// from ctrl->cur_p, so every iteration is the same launch sequence and a graph may resume at any iteration.
template <int K>
int enqueue_iteration(const Run& r, IterTimer* tm = nullptr) {
    int rc;
    if (tm && (rc = tm->mark(r.st, -1))) return rc;
    if (r.order_n == 1) {
        SpmmArgs a{r.w.z, r.w.p0, r.w.x, r.w.q, r.w.p1, 0, 1};
        if ((rc = launch_spmm<K, MODE_CG1>(r, r.g.cga, a))) return rc;
    } else {
        // S (M^-1 S)^(n-1) p' one factor at a time: t = M^-1 S p', n - 2 more factors t <- M^-1 S t
        // between the two buffers, q = M p' + c S t
        SpmmArgs a{r.w.z, r.w.p0, r.w.x, r.w.t, r.w.p1, 0, 1};
        if ((rc = launch_spmm<K, MODE_CG2A>(r, r.g.cga, a))) return rc;
        double* t = r.w.t;
        if ((rc = more_factors<K>(r, r.order_n - 2, &t))) return rc;
        SpmmArgs b{t, r.w.p0, nullptr, r.w.q, r.w.p1, 0, 1};
        if ((rc = launch_spmm<K, MODE_CG2B>(r, r.g.cgb, b))) return rc;
    }
    if (tm && (rc = tm->mark(r.st, 0))) return rc;
    k_update<K><<<r.g.update, BLOCK, 0, r.st>>>(r.m, r.w.ctrl, r.w.partials, r.w.z, r.w.q, r.order_n);
    IF_LAUNCH_CHECK();
    if (tm && (rc = tm->mark(r.st, 1))) return rc;
    return IF_OK;
}

// Two instantiations of the iteration graph, launched alternately: while one runs, the host reads the timing
// events of the other (an event must not be re-recorded while it is being read).
struct GraphSet {
    cudaGraphExec_t exec[2] = {nullptr, nullptr};
    IterTimer tev[2];
    ~GraphSet() {
        for (int i = 0; i < 2; ++i) { if (exec[i]) cudaGraphExecDestroy(exec[i]); tev[i].destroy(); }
    }
};

// What `enqueue(timer)` launches on `st`, captured twice into two graph instances (launched alternately, so that the
// timing events of one can be read while the other runs).  A stream that cannot be captured (the legacy default
// stream) leaves gs empty: the caller launches directly.  *launches_per_graph = kernels in one instance.
template <class F>
int capture_graphs(cudaStream_t st, GraphSet& gs, long long* launches_per_graph, F&& enqueue) {
    *launches_per_graph = 0;
    if (st == nullptr || st == cudaStreamLegacy) return IF_OK;
    for (int gi = 0; gi < 2; ++gi) {
        if (gs.tev[gi].create() != IF_OK) return IF_ECUDA;
        cudaGraph_t graph = nullptr;
        if (cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
            cudaGetLastError();   // stream cannot be captured: direct launches
            if (gs.exec[0]) { cudaGraphExecDestroy(gs.exec[0]); gs.exec[0] = nullptr; }
            return IF_OK;
        }
        const long long before = g_launches.load();
        const int rcc = enqueue(&gs.tev[gi]);
        *launches_per_graph = g_launches.load() - before;
        g_launches -= *launches_per_graph;   // captured, not launched
        cudaError_t e = cudaStreamEndCapture(st, &graph);
        if (rcc != IF_OK || e != cudaSuccess) { if (graph) cudaGraphDestroy(graph); cudaGetLastError(); return IF_ECUDA; }
        e = cudaGraphInstantiate(&gs.exec[gi], graph, 0);
        cudaGraphDestroy(graph);
        if (e != cudaSuccess) { gs.exec[gi] = nullptr; cudaGetLastError(); return IF_ECUDA; }
    }
    return IF_OK;
}

struct KernelTimes { double ms[TIMER_GROUPS] = {}; int64_t samples = 0; };   // per group, summed over samples

// one timed iteration of a finished graph launch into the per-group sums (events recorded inside the graph)
inline void add_timing_sample(KernelTimes& times, const IterTimer& te) {
    double ms[TIMER_GROUPS] = {};
    bool ok = te.n > 1;
    for (int i = 1; i < te.n && ok; ++i) {
        float dt = 0.f;
        ok = cudaEventElapsedTime(&dt, te.ev[i - 1], te.ev[i]) == cudaSuccess;
        if (ok && te.gid[i] >= 0 && te.gid[i] < TIMER_GROUPS) ms[te.gid[i]] += dt;
    }
    if (ok) {
        for (int g = 0; g < TIMER_GROUPS; ++g) times.ms[g] += ms[g];
        times.samples += 1;
    } else {
        cudaGetLastError();
    }
}

struct PollState {
    Snapshot* snap = nullptr;          // pinned [4]
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
    bool own_pinned = false;
    if_mesh_s* h = nullptr;
    ~PollState() {
        for (auto& e : ev) if (e) cudaEventDestroy(e);
        if (own_pinned && snap) cudaFreeHost(snap);
        else if (h) h->pinned_busy.store(0);
    }
};

// (Re)start the columns in `mask` from their right-hand sides: ingest, y = S (M^-1 S)^(n-1) phi, CG start.
template <int K>
int start_columns(const Run& r, unsigned mask, const StartParams& sp, const double* d_fields) {
    const if_mesh_s* h = r.h;
    const unsigned eg = (unsigned)((h->n_vert * K + BLOCK - 1) / BLOCK);
    int rc;
    if (r.mg) {   // multigrid path: the column joins the stream, its first iteration forms r0 (k_mg_start)
        const MgBuffers b = mg_buffers(r);
        k_mg_start<K><<<r.g.stream, BLOCK, 0, r.st>>>(r.m, r.w.ctrl, r.w.partials, sp, mask, d_fields, b.x, b.zb, b.r[0],
                                                      b.r[1], b.p[0], b.p[1]);
        IF_LAUNCH_CHECK();
        const MgLevel& gl = h->mg[h->mg_levels - 1];      // K^-1 of the coarsest level for the new columns' c1
        if (gl.n <= MG_COARSEST) {
            k_mg_coarse_factor<<<K, 64, MG_FACTOR_SMEM, r.st>>>(mg_mat(gl), r.w.ctrl, mask, b.coarse_inv);
            IF_LAUNCH_CHECK();
        }
        return IF_OK;
    }
    k_ingest<K><<<eg, BLOCK, 0, r.st>>>(r.m, sp, mask, d_fields, r.w.x);
    IF_LAUNCH_CHECK();
    if (r.order_n == 1) {
        SpmmArgs a{r.w.x, nullptr, nullptr, r.w.q, nullptr, 0, 0};
        if ((rc = launch_spmm<K, MODE_PLAIN>(r, r.g.plain, a))) return rc;
    } else {
        SpmmArgs a{r.w.x, nullptr, nullptr, r.w.t, nullptr, 1, 0};
        if ((rc = launch_spmm<K, MODE_PLAIN>(r, r.g.plain, a))) return rc;
        double* t = r.w.t;
        if ((rc = more_factors<K>(r, r.order_n - 2, &t))) return rc;
        SpmmArgs b{t, nullptr, nullptr, r.w.q, nullptr, 0, 0};
        if ((rc = launch_spmm<K, MODE_PLAIN>(r, r.g.plain, b))) return rc;
    }
    k_init<K><<<r.g.stream, BLOCK, 0, r.st>>>(r.m, r.w.ctrl, r.w.partials, sp, mask, r.w.x, r.w.q, r.w.z, r.w.p0,
                                              r.w.p1, r.order_n);
    IF_LAUNCH_CHECK();
    return IF_OK;
}

// The columns in `mask` have stopped: energy or scatter of x, and the per-right-hand-side results.
template <int K>
int finalize_columns(const Run& r, Job job, unsigned mask, double* d_out, const double* d_fields) {
    const if_mesh_s* h = r.h;
    if (job == JOB_SPECTRUM) {
        k_energy<K><<<r.g.stream, BLOCK, 0, r.st>>>(r.m, r.w.ctrl, r.w.partials, mask, r.w.x, r.w.p0, r.w.p1,
                                                    h->total_area, r.w.energy);
        IF_LAUNCH_CHECK();
    } else {
        const int sgrid = (int)std::min<int64_t>((h->n_vert + 31) / 32, (int64_t)h->n_sm * 8);
        k_scatter<K><<<sgrid, BLOCK, 0, r.st>>>(r.m, r.w.ctrl, mask, r.w.x, r.w.p0, r.w.p1, 1, d_out, d_fields,
                                                (r.opt.flags & IF_FLAG_HIGHPASS) ? 1 : 0);
        IF_LAUNCH_CHECK();
    }
    k_stats<<<1, 32, 0, r.st>>>(r.w.ctrl, K, mask, r.w.iters, r.w.status, r.w.relres);
    IF_LAUNCH_CHECK();
    return IF_OK;
}

Ctrl fresh_ctrl(const Run& r) {
    Ctrl hc;
    memset(&hc, 0, sizeof(hc));
    for (int c = 0; c < KMAX; ++c) { hc.field[c] = -1; hc.done[c] = 1; }
    hc.all_done = 1;
    hc.max_iter = r.opt.max_iter;
    hc.tol2 = r.opt.tol * r.opt.tol;
    hc.pair_mode = r.vec ? 1 : 0;
    return hc;
}

// q = A_c x_c for up to K columns: column i takes its values from src[field_i] (caller's numbering) and its scale from
// sp.c[i]; the control block is reset (no solve may be in flight).  Result in r.w.q, internal order.
template <int K>
int apply_columns(Run& r, const StartParams& sp, const double* d_src) {
    const if_mesh_s* h = r.h;
    int rc;
    Ctrl hc = fresh_ctrl(r);
    for (int c = 0; c < KMAX; ++c) { hc.c[c] = sp.c[c]; hc.field[c] = sp.field[c]; hc.rhs[c] = sp.rhs[c]; }
    hc.all_done = 0;
    IF_CUDA_TRY(cudaMemcpyAsync(r.w.ctrl, &hc, sizeof(Ctrl), cudaMemcpyHostToDevice, r.st));
    IF_CUDA_TRY(cudaStreamSynchronize(r.st));      // hc lives on this stack frame
    const unsigned eg = (unsigned)((h->n_vert * K + BLOCK - 1) / BLOCK);
    k_ingest<K><<<eg, BLOCK, 0, r.st>>>(r.m, sp, (1u << K) - 1u, d_src, r.w.x);
    IF_LAUNCH_CHECK();
    const double* v = r.w.x;
    if (r.order_n >= 2) {
        SpmmArgs a{r.w.x, nullptr, nullptr, r.w.t, nullptr, 1, 0};
        if ((rc = launch_spmm<K, MODE_PLAIN>(r, r.g.plain, a))) return rc;
        double* t = r.w.t;
        if ((rc = more_factors<K>(r, r.order_n - 2, &t))) return rc;
        v = t;
    }
    SpmmArgs b{v, r.w.x, nullptr, r.w.q, nullptr, 0, 0};
    return launch_spmm<K, MODE_CG2B>(r, r.g.cgb, b);
}

// Batches of right-hand sides for apply_columns: rhs[first ...] into columns (pairs of columns for the vector filter);
// src_by_rhs: the source field of a column is the right-hand side's own slot f * n_ells + j (the filtered fields in
// d_out) instead of field f.  Returns the number of columns in use.
template <int K>
size_t fill_columns(const Run& r, const std::vector<Rhs>& rhs, size_t first, int n_ells, bool src_by_rhs, StartParams* sp,
                    StartParams* orig) {
    const size_t step = r.vec ? 2 : 1, per_batch = K / step;
    const size_t count = std::min<size_t>(per_batch, rhs.size() - first) * step;
    memset(sp, 0, sizeof(*sp));
    for (int c = 0; c < KMAX; ++c) sp->field[c] = -1;
    if (orig) *orig = *sp;
    for (size_t i = 0; i < count; ++i) {
        const Rhs& q = rhs[first + i / step];
        const int f = r.vec ? 2 * q.f + (int)(i % step) : q.f;
        sp->c[i] = r.opt.gamma * std::pow(q.ell, 2.0 * r.order_n);
        sp->rhs[i] = f * n_ells + q.j;
        sp->field[i] = src_by_rhs ? sp->rhs[i] : f;
        if (orig) { orig->c[i] = sp->c[i]; orig->rhs[i] = sp->rhs[i]; orig->field[i] = f; }
    }
    return count;
}

// if_apply: out = A_c phi for every right-hand side, K at a time (no iteration).
template <int K>
int apply_all(Run& r, const double* d_fields, const std::vector<Rhs>& rhs, int n_ells, double* d_out) {
    const if_mesh_s* h = r.h;
    int rc;
    if ((rc = setup_grids<K>(r))) return rc;
    const size_t per_batch = K / (r.vec ? 2 : 1);
    for (size_t first = 0; first < rhs.size(); first += per_batch) {
        StartParams sp;
        fill_columns<K>(r, rhs, first, n_ells, false, &sp, nullptr);
        if ((rc = apply_columns<K>(r, sp, d_fields))) return rc;
        const int sgrid = (int)std::min<int64_t>((h->n_vert + 31) / 32, (int64_t)h->n_sm * 8);
        k_scatter<K><<<sgrid, BLOCK, 0, r.st>>>(r.m, r.w.ctrl, (1u << K) - 1u, r.w.q, r.w.p0, r.w.p1, 0, d_out, nullptr, 0);
        IF_LAUNCH_CHECK();
    }
    return IF_OK;
}

// IF_FLAG_TRUE_RESIDUAL after if_filter: ||M phi - A x|| / ||M phi|| of every returned field, into d_true[rhs]
template <int K>
int true_residuals(Run& r, const double* d_fields, const std::vector<Rhs>& rhs, int n_ells, const double* d_out,
                   double* d_true) {
    int rc;
    if ((rc = setup_grids<K>(r))) return rc;
    const size_t per_batch = K / (r.vec ? 2 : 1);
    for (size_t first = 0; first < rhs.size(); first += per_batch) {
        StartParams sp, orig;
        fill_columns<K>(r, rhs, first, n_ells, true, &sp, &orig);
        if ((rc = apply_columns<K>(r, sp, d_out))) return rc;
        k_true_res<K><<<r.g.stream, BLOCK, 0, r.st>>>(r.m, r.w.ctrl, r.w.partials, orig, d_fields, r.w.q, d_true);
        IF_LAUNCH_CHECK();
    }
    return IF_OK;
}

// Host view of the K columns: which right-hand side each one runs, and the epoch the device should report for it.
struct QueueState {
    int col_rhs[KMAX];
    int host_epoch[KMAX];
    size_t next = 0;     // next right-hand side of the queue
    int active = 0;      // columns running a right-hand side
};

// if_filter / if_spectrum: right-hand sides through K columns with refill.  With `first` the columns are started
// from the queue; otherwise the state comes from a wider phase (compact_columns).  Returns when every column has
// stopped, or -- if *compact_to is given -- when the queue is empty and at most K/2 columns are still running
// (*compact_to = 4 or 8: the survivors should move to that many columns).
template <int K>
int solve_phase(Run& r, Job job, const double* d_fields, const std::vector<Rhs>& rhs, int n_ells, double* d_out,
                PollState& poll, KernelTimes* times, QueueState& q, bool first, int* compact_to) {
    int rc;
    if ((rc = setup_grids<K>(r))) return rc;
    if (r.mg && (rc = mg_setup<K>(r))) return rc;
    const size_t R = rhs.size();
    if (compact_to) *compact_to = 0;
    auto assign = [&](unsigned mask, StartParams* sp, unsigned* started) {
        memset(sp, 0, sizeof(*sp));
        for (int c = 0; c < KMAX; ++c) sp->field[c] = -1;
        *started = 0;
        // vector filter: a right-hand side is a (u, v) pair (field index = pair index) and takes the columns (c, c + 1)
        const int step = r.vec ? 2 : 1;
        for (int c0 = 0; c0 < K; c0 += step) {
            if (!((mask >> c0) & 1u)) continue;
            const bool have = q.next < R;
            for (int c = c0; c < c0 + step; ++c) {
                if (have) {
                    const Rhs& s = rhs[q.next];
                    const int f = r.vec ? 2 * s.f + (c - c0) : s.f;
                    sp->c[c] = r.opt.gamma * std::pow(s.ell, 2.0 * r.order_n);
                    sp->c1[c] = r.order_n == 1 ? sp->c[c] : std::sqrt(sp->c[c]);   // K = M + sqrt(c) S (mg_solve.cuh)
                    sp->field[c] = f;
                    sp->rhs[c] = f * n_ells + s.j;
                    q.col_rhs[c] = (int)q.next;
                    ++q.active;
                } else {
                    q.col_rhs[c] = -1;
                }
                *started |= 1u << c;
                q.host_epoch[c] += 1;
            }
            if (have) ++q.next;
        }
    };
    StartParams sp;
    unsigned started = 0;
    if (first) {
        Ctrl hc = fresh_ctrl(r);
        IF_CUDA_TRY(cudaMemcpyAsync(r.w.ctrl, &hc, sizeof(Ctrl), cudaMemcpyHostToDevice, r.st));
        for (int c = 0; c < KMAX; ++c) { q.col_rhs[c] = -1; q.host_epoch[c] = 0; }
        assign((1u << K) - 1u, &sp, &started);          // empty columns are started too (zeroed, done at once)
        if ((rc = start_columns<K>(r, started, sp, d_fields))) return rc;
    }

    // the iteration loop: `check_every` iterations per CUDA graph launch, snapshot polled one launch behind
    // (a multigrid iteration is some forty launches and a thirtieth of a solve: one per graph)
    const int per_graph = r.mg ? 1 : r.opt.check_every;
    long long launches_per_graph = 0;
    GraphSet gs;
    rc = capture_graphs(r.st, gs, &launches_per_graph, [&](IterTimer* timer) {
        int rcc = IF_OK;
        const int timed_it = per_graph > 2 ? 2 : 0;
        for (int i = 0; i < per_graph && rcc == IF_OK; ++i) {
            IterTimer* tm = i == timed_it ? timer : nullptr;
            rcc = r.mg ? mg_enqueue_iteration<K>(r, tm) : enqueue_iteration<K>(r, tm);
        }
        return rcc;
    });
    if (rc != IF_OK) return rc;
    const bool use_graph = gs.exec[0] && gs.exec[1];
    const int64_t per_rhs = (r.opt.max_iter + per_graph - 1) / per_graph + 3;
    const int64_t max_loops = ((int64_t)(R + K - 1) / K + 1) * per_rhs + 8;
    unsigned free_cols = 0;   // stopped and finalised, waiting for a right-hand side
    for (int64_t it = 0; it < max_loops && q.active > 0; ++it) {
        if (use_graph) {
            IF_CUDA_TRY(cudaGraphLaunch(gs.exec[it & 1], r.st));
            g_launches += launches_per_graph;
        } else {
            for (int i = 0; i < per_graph; ++i)
                if ((rc = r.mg ? mg_enqueue_iteration<K>(r, nullptr) : enqueue_iteration<K>(r))) return rc;
        }
        const int slot = (int)(it & 3);
        IF_CUDA_TRY(cudaMemcpyAsync(&poll.snap[slot], reinterpret_cast<const char*>(r.w.ctrl) + offsetof(Ctrl, done),
                                    sizeof(Snapshot), cudaMemcpyDeviceToHost, r.st));
        IF_CUDA_TRY(cudaEventRecord(poll.ev[slot], r.st));
        if (it == 0) continue;
        const int prev = (int)((it - 1) & 3);
        IF_CUDA_TRY(cudaEventSynchronize(poll.ev[prev]));
        const Snapshot& s = poll.snap[prev];
        unsigned fin = 0;
        bool any_running = false;
        for (int c = 0; c < K; ++c) {
            if (q.col_rhs[c] < 0 || s.epoch[c] != q.host_epoch[c]) continue;
            if (s.done[c]) fin |= 1u << c; else any_running = true;
        }
        // launch it-1 did full work in every kernel: take its timing sample (graph (it-1)&1 is idle now)
        if (times && use_graph && any_running) add_timing_sample(*times, gs.tev[(it - 1) & 1]);
        if (fin) {
            // these columns stopped before launch it-1 ended and stayed frozen through launch it
            if ((rc = finalize_columns<K>(r, job, fin, d_out, d_fields))) return rc;
            for (int c = 0; c < K; ++c) if ((fin >> c) & 1u) --q.active;
            for (int c = 0; c < K; ++c) if ((fin >> c) & 1u) q.col_rhs[c] = -1;
            free_cols |= fin;
        }
        // refill as soon as MG_REFILL_MIN columns are free (1: at once, as the Jacobi path always does -- waiting for
        // company was measured and simulated on config 4: 156 batch iterations against 132)
        if (free_cols && q.next < R) {
            int nfree = 0;
            for (int c = 0; c < K; ++c) nfree += (free_cols >> c) & 1u;
            if (!r.mg || nfree >= MG_REFILL_MIN || q.active == 0 || (size_t)nfree >= R - q.next) {
                assign(free_cols, &sp, &started);
                if ((rc = start_columns<K>(r, started, sp, d_fields))) return rc;
                free_cols = 0;
            }
        }
        if (compact_to && !r.mg && K > 4 && q.next >= R && q.active > 0 && q.active <= K / 2) {
            *compact_to = (q.active <= 4) ? 4 : 8;
            return IF_OK;   // the graph launch already enqueued runs first; the caller repacks after it
        }
    }
    if (q.active > 0) return IF_ECUDA;   // cannot happen: every column stops at max_iter
    return IF_OK;
}

// Move the running columns of a KW-wide phase into a KN-wide layout (KN <= KW/2).  The narrow vectors live in the
// wide buffers that are dead at an iteration boundary: x, z -> the two halves of q; p0, p1 -> the halves of x;
// q, t -> the halves of z.
template <int KW, int KN>
int compact_columns(Run& r, QueueState& q) {
    static_assert(2 * KN <= KW, "compaction at least halves the width");
    ColMap map;
    QueueState nq = q;
    int j = 0;
    for (int c = 0; c < KMAX; ++c) { map.src[c] = -1; nq.col_rhs[c] = -1; nq.host_epoch[c] = 0; }
    for (int c = 0; c < KW; ++c)
        if (q.col_rhs[c] >= 0) {
            if (j >= KN) return IF_ECUDA;
            map.src[j] = c;
            nq.col_rhs[j] = q.col_rhs[c];
            nq.host_epoch[j] = q.host_epoch[c];
            ++j;
        }
    const int64_t nv = r.h->n_vert;
    const size_t vn = (size_t)nv * KN;   // doubles per narrow vector
    const unsigned g = (unsigned)((vn + BLOCK - 1) / BLOCK);
    Workspace& w = r.w;
    double* x2 = w.q;
    double* z2 = w.q + vn;
    k_repack<KW, KN><<<g, BLOCK, 0, r.st>>>(nv, map, w.x, x2);
    IF_LAUNCH_CHECK();
    k_repack<KW, KN><<<g, BLOCK, 0, r.st>>>(nv, map, w.z, z2);
    IF_LAUNCH_CHECK();
    double* p0_2 = w.x;
    double* p1_2 = w.x + vn;
    k_repack<KW, KN><<<g, BLOCK, 0, r.st>>>(nv, map, w.p0, p0_2);
    IF_LAUNCH_CHECK();
    k_repack<KW, KN><<<g, BLOCK, 0, r.st>>>(nv, map, w.p1, p1_2);
    IF_LAUNCH_CHECK();
    double* q2 = w.z;
    double* t2 = w.z + vn;
    k_compact_ctrl<<<1, KMAX, 0, r.st>>>(w.ctrl, map, KN);
    IF_LAUNCH_CHECK();
    double* t3 = w.p0;   // (the wide p0 is dead once repacked: room for the second factor buffer of n >= 3)
    w.x = x2; w.z = z2; w.p0 = p0_2; w.p1 = p1_2; w.q = q2;
    if (r.order_n >= 2) w.t = t2;
    if (r.order_n >= 3) w.t2 = t3;
    q = nq;
    return IF_OK;
}

template <int K>
int solve_from(Run& r, Job job, const double* d_fields, const std::vector<Rhs>& rhs, int n_ells, double* d_out,
               PollState& poll, KernelTimes* times, QueueState& q, bool first) {
    int to = 0;
    int rc = solve_phase<K>(r, job, d_fields, rhs, n_ells, d_out, poll, times, q, first, K > 4 ? &to : nullptr);
    if (rc != IF_OK || to == 0) return rc;
    if constexpr (K == 16) {
        if (to == 8) {
            if ((rc = compact_columns<16, 8>(r, q))) return rc;
            return solve_from<8>(r, job, d_fields, rhs, n_ells, d_out, poll, nullptr, q, false);
        }
        if ((rc = compact_columns<16, 4>(r, q))) return rc;
        return solve_from<4>(r, job, d_fields, rhs, n_ells, d_out, poll, nullptr, q, false);
    } else if constexpr (K == 8) {
        if ((rc = compact_columns<8, 4>(r, q))) return rc;
        return solve_from<4>(r, job, d_fields, rhs, n_ells, d_out, poll, nullptr, q, false);
    }
    return IF_ECUDA;
}

// End and start of columns inside the stream (multigrid path): what k_turn_plan decided is carried out by the same
// kernels the host-driven refill uses, with their masks read from the control block.
template <int K>
int mg_enqueue_turnover(const Run& r, Job job, double* d_out, const double* d_fields, bool first = false) {
    const if_mesh_s* h = r.h;
    const MgBuffers b = mg_buffers(r);
    k_turn_plan<<<1, 32, 0, r.st>>>(r.w.ctrl, r.w.queue, K, first ? 1 : 0, r.w.iters, r.w.status, r.w.relres);
    IF_LAUNCH_CHECK();
    if (job == JOB_SPECTRUM) {
        k_energy<K><<<r.g.stream, BLOCK, 0, r.st>>>(r.m, r.w.ctrl, r.w.partials, MASK_TURN_FIN, b.x, b.p[0], b.p[1],
                                                    h->total_area, r.w.energy);
    } else {
        const int sgrid = (int)std::min<int64_t>((h->n_vert + 31) / 32, (int64_t)h->n_sm * 8);
        k_scatter<K><<<sgrid, BLOCK, 0, r.st>>>(r.m, r.w.ctrl, MASK_TURN_FIN, b.x, b.p[0], b.p[1], 1, d_out, d_fields,
                                                  (r.opt.flags & IF_FLAG_HIGHPASS) ? 1 : 0);
    }
    IF_LAUNCH_CHECK();
    StartParams none;
    memset(&none, 0, sizeof(none));
    k_mg_start<K><<<r.g.stream, BLOCK, 0, r.st>>>(r.m, r.w.ctrl, r.w.partials, none, MASK_TURN_START, d_fields, b.x, b.zb,
                                                    b.r[0], b.r[1], b.p[0], b.p[1]);
    IF_LAUNCH_CHECK();
    const MgLevel& gl = h->mg[h->mg_levels - 1];
    if (gl.n <= MG_COARSEST) {
        k_mg_coarse_factor<<<K, 64, MG_FACTOR_SMEM, r.st>>>(mg_mat(gl), r.w.ctrl, MASK_TURN_START, b.coarse_inv);
        IF_LAUNCH_CHECK();
    }
    return IF_OK;
}

// The multigrid stream with the column turnover on the device: the queue of right-hand sides lives in the workspace,
// one CUDA graph = one iteration + the turnover, and the host only launches graphs and reads, one launch behind, how
// many columns still hold a right-hand side.  A stopped column runs its next right-hand side in the very next iteration
// (the host-driven refill of solve_phase, which sees a stop one launch late, loses an iteration per right-hand side).
// `first`: the queue and a fresh control block are set up and the first right-hand sides started; otherwise the state
// comes from a wider phase (mg_compact).  *compact_to (if given): set to 8 or 4 when the queue is empty and the columns
// still running fit that width -- the caller compacts after the launch already enqueued and goes on there.
template <int K>
int mg_stream_on_device(Run& r, Job job, const double* d_fields, const std::vector<Rhs>& rhs, int n_ells, double* d_out,
                        PollState& poll, KernelTimes* times, bool first, int* compact_to) {
    int rc;
    if (compact_to) *compact_to = 0;
    if ((rc = setup_grids<K>(r))) return rc;
    if ((rc = mg_setup<K>(r))) return rc;
    const size_t R = rhs.size();
    if (R == 0 || R > (size_t)MAX_RHS || !r.w.queue) return IF_EINVAL;
    std::vector<QEntry> hq(first ? R : 0);
    if (first) {
    for (size_t i = 0; i < R; ++i) {
        const Rhs& s = rhs[i];
        hq[i].c = r.opt.gamma * std::pow(s.ell, 2.0 * r.order_n);
        hq[i].c1 = r.order_n == 1 ? hq[i].c : std::sqrt(hq[i].c);   // K = M + sqrt(c) S (mg_solve.cuh)
        // (vector filter: s.f counts (u, v) pairs; the entry names the u field and slot, k_turn_plan derives v's)
        const int f = r.vec ? 2 * s.f : s.f;
        hq[i].field = f;
        hq[i].rhs = f * n_ells + s.j;
    }
    Ctrl hc = fresh_ctrl(r);
    hc.q_next = 0;
    hc.q_total = (int)R;
    hc.rhs_stride = n_ells;
    // (pageable sources: both copies are staged by the runtime before the call returns)
    IF_CUDA_TRY(cudaMemcpyAsync(r.w.ctrl, &hc, sizeof(Ctrl), cudaMemcpyHostToDevice, r.st));
    IF_CUDA_TRY(cudaMemcpyAsync(r.w.queue, hq.data(), R * sizeof(QEntry), cudaMemcpyHostToDevice, r.st));
    if ((rc = mg_enqueue_turnover<K>(r, job, d_out, d_fields, true))) return rc;      // the first K right-hand sides
    }

    long long launches_per_graph = 0;
    GraphSet gs;
    rc = capture_graphs(r.st, gs, &launches_per_graph, [&](IterTimer* timer) {
        const int rcc = mg_enqueue_iteration<K>(r, timer);
        return rcc != IF_OK ? rcc : mg_enqueue_turnover<K>(r, job, d_out, d_fields);
    });
    if (rc != IF_OK) return rc;
    const bool use_graph = gs.exec[0] && gs.exec[1];
    const int64_t slots = r.vec ? K / 2 : K;
    const int64_t max_loops = ((int64_t)(R + slots - 1) / slots + 1) * ((int64_t)r.opt.max_iter + 3) + 8;
    int* snap = reinterpret_cast<int*>(poll.snap);      // four slots of four ints in the pinned snapshot buffer
    bool finished = false;
    int running_before = 0;
    for (int64_t it = 0; it < max_loops && !finished; ++it) {
        if (use_graph) {
            IF_CUDA_TRY(cudaGraphLaunch(gs.exec[it & 1], r.st));
            g_launches += launches_per_graph;
        } else {
            if ((rc = mg_enqueue_iteration<K>(r, nullptr))) return rc;
            if ((rc = mg_enqueue_turnover<K>(r, job, d_out, d_fields))) return rc;
        }
        const int slot = (int)(it & 3);
        IF_CUDA_TRY(cudaMemcpyAsync(snap + 4 * slot, reinterpret_cast<const char*>(r.w.ctrl) + offsetof(Ctrl, snap),
                                    4 * sizeof(int), cudaMemcpyDeviceToHost, r.st));
        IF_CUDA_TRY(cudaEventRecord(poll.ev[slot], r.st));
        if (it == 0) continue;
        const int prev = (int)((it - 1) & 3);
        IF_CUDA_TRY(cudaEventSynchronize(poll.ev[prev]));
        const int occupied = snap[4 * prev], running = snap[4 * prev + 1];
        const bool worked = it == 1 || running_before > 0;     // columns were running when launch it-1 began
        running_before = running;
        // launch it-1 did full work in every kernel: take its timing sample (graph (it-1)&1 is idle now)
        if (times && use_graph && worked && running > 0) add_timing_sample(*times, gs.tev[(it - 1) & 1]);
        if (occupied == 0) finished = true;      // every right-hand side has been started, stopped and finalised
        // the tail: the queue is empty and the slots still occupied fit a narrower set of kernels
        const int occ_cols = occupied * (r.vec ? 2 : 1);
        if (!finished && compact_to && K > 4 && snap[4 * prev + 2] >= (int)R && occ_cols <= K / 2) {
            *compact_to = (occ_cols <= 4) ? 4 : 8;
            return IF_OK;   // the launch already enqueued runs first; the caller repacks after it
        }
    }
    if (!finished) return IF_ECUDA;   // cannot happen: every column stops at max_iter
    return IF_OK;
}

// The columns still running move from the KW-wide layout `b` to a KN-wide one (KN <= KW / 2), decided and done on the
// device at the iteration boundary this is enqueued at: x, the current r and p, and z are repacked into the halves of
// buffers that are dead there (q, za), the other narrow buffers take the halves of what the repacking freed.
template <int KW, int KN>
int mg_compact(const Run& r, const MgBuffers& b, MgBuffers* out) {
    static_assert(2 * KN <= KW, "compaction at least halves the width");
    const if_mesh_s* h = r.h;
    const int64_t nv = h->n_vert;
    const size_t vn = (size_t)nv * KN;      // doubles per narrow vector: two fit every buffer of the wide layout
    const unsigned g = (unsigned)((vn + BLOCK - 1) / BLOCK);
    MgBuffers n = b;
    n.x = b.q;          n.r[0] = b.q + vn;
    n.zb = b.za;        n.p[0] = b.za + vn;
    n.r[1] = b.t;       n.p[1] = b.t + vn;
    n.q = b.x;          n.za = b.x + vn;
    n.t = b.zb;
    k_mg_compact_plan<<<1, 32, 0, r.st>>>(r.w.ctrl, KW, KN);
    IF_LAUNCH_CHECK();
    k_mg_repack<KW, KN><<<g, BLOCK, 0, r.st>>>(nv, r.w.ctrl, 0, b.x, nullptr, n.x);
    IF_LAUNCH_CHECK();
    k_mg_repack<KW, KN><<<g, BLOCK, 0, r.st>>>(nv, r.w.ctrl, 1, b.r[0], b.r[1], n.r[0]);
    IF_LAUNCH_CHECK();
    k_mg_repack<KW, KN><<<g, BLOCK, 0, r.st>>>(nv, r.w.ctrl, 0, b.zb, nullptr, n.zb);
    IF_LAUNCH_CHECK();
    k_mg_repack<KW, KN><<<g, BLOCK, 0, r.st>>>(nv, r.w.ctrl, 2, b.p[0], b.p[1], n.p[0]);
    IF_LAUNCH_CHECK();
    k_mg_compact_ctrl<<<1, KMAX, 0, r.st>>>(r.w.ctrl, KN);
    IF_LAUNCH_CHECK();
    const MgLevel& gl = h->mg[h->mg_levels - 1];      // K^-1 of the coarsest level under the new column numbers
    if (gl.n <= MG_COARSEST) {
        IF_CUDA_TRY(cudaFuncSetAttribute(k_mg_coarse_factor, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)MG_FACTOR_SMEM));
        k_mg_coarse_factor<<<KN, 64, MG_FACTOR_SMEM, r.st>>>(mg_mat(gl), r.w.ctrl, (1u << KN) - 1u, n.coarse_inv);
        IF_LAUNCH_CHECK();
    }
    *out = n;
    return IF_OK;
}

template <int K>
int mg_stream_from(Run& r, Job job, const double* d_fields, const std::vector<Rhs>& rhs, int n_ells, double* d_out,
                   PollState& poll, KernelTimes* times, bool first) {
    int to = 0;
    int rc = mg_stream_on_device<K>(r, job, d_fields, rhs, n_ells, d_out, poll, times, first, K > 4 ? &to : nullptr);
    if (rc != IF_OK || to == 0) return rc;
    const MgBuffers cur = mg_buffers(r);
    MgBuffers narrow;
    const void* saved = r.mgb;
    if (const char* v = getenv("IF_VERBOSE"))
        if (atoi(v) >= 1) fprintf(stderr, "[implicit_filter] multigrid stream: tail moved from %d to %d columns\n", K, to);
    if constexpr (K == 16) {
        if (to == 8) {
            if ((rc = mg_compact<16, 8>(r, cur, &narrow))) return rc;
            r.mgb = &narrow;
            rc = mg_stream_from<8>(r, job, d_fields, rhs, n_ells, d_out, poll, nullptr, false);
        } else {
            if ((rc = mg_compact<16, 4>(r, cur, &narrow))) return rc;
            r.mgb = &narrow;
            rc = mg_stream_from<4>(r, job, d_fields, rhs, n_ells, d_out, poll, nullptr, false);
        }
    } else if constexpr (K == 8) {
        if ((rc = mg_compact<8, 4>(r, cur, &narrow))) return rc;
        r.mgb = &narrow;
        rc = mg_stream_from<4>(r, job, d_fields, rhs, n_ells, d_out, poll, nullptr, false);
    }
    r.mgb = saved;
    return rc;
}

template <int K>
int solve_all(Run& r, Job job, const double* d_fields, const std::vector<Rhs>& rhs, int n_ells, double* d_out,
              PollState& poll, KernelTimes* times, int64_t* batch_iters) {
    QueueState q;
    int rc = IF_OK;
    bool on_device = false;
    if (r.mg) {
        // multigrid stream: column turnover on the device where an iteration is long enough to pay for the four extra
        // graph nodes (about 12 us per iteration against one idle column-iteration per right-hand side: break-even
        // near 0.5 ms per iteration = 400 k rows for n = 1, a quarter of that for n = 2; measured on configs 2 and 4),
        // else the host-driven refill of solve_phase.  IF_MG_HOST_REFILL = 1 / 0 forces one or the other (tests).
        const char* env = getenv("IF_MG_HOST_REFILL");
        const bool big = r.h->n_vert * (r.order_n == 1 ? 1 : 4) >= MG_DEVICE_TURNOVER_ROWS;
        const bool host_refill = env != nullptr ? atoi(env) != 0 : !big;
        on_device = r.mg && !host_refill;
        if (on_device) rc = mg_stream_from<K>(r, job, d_fields, rhs, n_ells, d_out, poll, times, true);
    }
    if (!on_device) rc = solve_from<K>(r, job, d_fields, rhs, n_ells, d_out, poll, times, q, true);
    if (rc != IF_OK) return rc;
    long long total = 0;
    IF_CUDA_TRY(cudaMemcpyAsync(&total, &r.w.ctrl->total_iters, sizeof(long long), cudaMemcpyDeviceToHost, r.st));
    IF_CUDA_TRY(cudaStreamSynchronize(r.st));
    *batch_iters = (int64_t)total;
    return IF_OK;
}

int pick_k(int batch, size_t R) {
    int K = batch;
    while (K > 4 && R <= (size_t)K / 2) K /= 2;   // few right-hand sides: narrower columns, less wasted bandwidth
    return K;
}

int run_job_on_device(if_handle h, Job job, const double* d_fields, int n_fields, const double* ells, int n_ells, int order_n,
                      double* d_out, double* energy, double* k_mid, double* E, void* d_ws, size_t ws_bytes, void* stream,
                      const if_options* opt_in, if_stats* stats);

// The handle's device is made current for the call and the caller's device restored afterwards, whatever the outcome.
int run_job(if_handle h, Job job, const double* d_fields, int n_fields, const double* ells, int n_ells, int order_n,
            double* d_out, double* energy, double* k_mid, double* E, void* d_ws, size_t ws_bytes, void* stream,
            const if_options* opt_in, if_stats* stats) {
    if (!h) return IF_EINVAL;
    int prev = -1;
    if (cudaGetDevice(&prev) != cudaSuccess) { cudaGetLastError(); return IF_ECUDA; }
    if (prev != h->device) IF_CUDA_TRY(cudaSetDevice(h->device));
    const int rc = run_job_on_device(h, job, d_fields, n_fields, ells, n_ells, order_n, d_out, energy, k_mid, E, d_ws, ws_bytes,
                                     stream, opt_in, stats);
    if (prev != h->device) cudaSetDevice(prev);
    return rc;
}

int run_job_on_device(if_handle h, Job job, const double* d_fields, int n_fields, const double* ells, int n_ells, int order_n,
                      double* d_out, double* energy, double* k_mid, double* E, void* d_ws, size_t ws_bytes, void* stream,
                      const if_options* opt_in, if_stats* stats) {
    if (!h || !d_fields || !ells || n_fields < 1 || n_ells < 1 || order_n < 1 || order_n > 4 || !d_ws)
        return IF_EINVAL;
    if (job != JOB_SPECTRUM && !d_out) return IF_EINVAL;
    if (job == JOB_SPECTRUM && n_ells < 2) return IF_EINVAL;
    if (job == JOB_SPECTRUM && opt_in && (opt_in->flags & IF_FLAG_PAIRS) && n_fields % 2 != 0) return IF_EINVAL;
    const int64_t R = (int64_t)n_fields * n_ells;
    if (R > MAX_RHS) return IF_EINVAL;
    for (int j = 0; j < n_ells; ++j) {
        if (!(ells[j] > 0.0) || !std::isfinite(ells[j])) return IF_EINVAL;
        if (job == JOB_SPECTRUM && j > 0 && !(ells[j] > ells[j - 1])) return IF_EINVAL;
    }
    Run r;
    r.h = h;
    int rc = resolve_options(opt_in, &h->opt, &r.opt);
    if (rc != IF_OK) return rc;
    r.order_n = order_n;
    r.st = static_cast<cudaStream_t>(stream);
    r.vec = opt_in && (opt_in->flags & IF_FLAG_VECTOR);      // per call only: the handle's own flag just says "assembled"
    if (r.vec && (n_fields % 2 != 0 || order_n > 2 || !h->sell_dval)) return IF_EINVAL;
    const bool pairs = job == JOB_SPECTRUM && (r.opt.flags & IF_FLAG_PAIRS);
    const int n_out_fields = pairs ? n_fields / 2 : n_fields;
    r.w = layout_workspace(h, order_n, r.opt.batch, d_ws);
    if (ws_bytes < r.w.bytes) return IF_EWORKSPACE;
    int log2c = 0;
    while ((1 << log2c) < h->sell_c) ++log2c;
    // vector filter: D~ takes the place of S (entries, diagonal, Jacobi diagonal of n = 2), T rides beside it
    r.m = MeshView{h->chunk_ptr, h->sell_col, r.vec ? h->sell_dval : h->sell_val, r.vec ? h->sell_tval : nullptr, h->area,
                   h->inv_area, r.vec ? h->ddiag : h->sdiag, r.vec ? h->gdiag_vec : h->gdiag, h->gdiag3, h->gdiag4, h->perm,
                   h->sell_lcol, h->halo_rows, h->tile_desc, h->n_vert, h->n_chunks, log2c};

    PollState poll;
    int expected = 0;
    if (h->h_pinned && h->pinned_busy.compare_exchange_strong(expected, 1)) {
        poll.snap = static_cast<Snapshot*>(h->h_pinned);
        poll.h = h;
    } else {
        IF_CUDA_TRY(cudaHostAlloc((void**)&poll.snap, 4 * sizeof(Snapshot) + 512, cudaHostAllocDefault));
        poll.own_pinned = true;
    }
    for (auto& e : poll.ev) IF_CUDA_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    struct EvGuard {
        cudaEvent_t a = nullptr, b = nullptr;
        ~EvGuard() { if (a) cudaEventDestroy(a); if (b) cudaEventDestroy(b); }
    } evg;
    IF_CUDA_TRY(cudaEventCreate(&evg.a));
    IF_CUDA_TRY(cudaEventCreate(&evg.b));
    const cudaEvent_t t0 = evg.a, t1 = evg.b;
    // every way out of this function -- error returns included -- waits for what it has enqueued before the pinned
    // snapshot buffer, the events and this stack frame go away (declared last: runs first)
    struct SyncGuard { cudaStream_t s; ~SyncGuard() { cudaStreamSynchronize(s); } } sync_guard{r.st};
    IF_CUDA_TRY(cudaEventRecord(t0, r.st));

    // queue of right-hand sides: largest scale (most iterations) first, so that the short solves fill the tail
    std::vector<Rhs> rhs;
    rhs.reserve((size_t)R);
    for (int f = 0; f < (r.vec ? n_fields / 2 : n_fields); ++f)      // (vector filter: f counts (u, v) pairs)
        for (int j = 0; j < n_ells; ++j) rhs.push_back(Rhs{ells[j], f, j});
    if (job != JOB_APPLY)
        std::stable_sort(rhs.begin(), rhs.end(), [](const Rhs& a, const Rhs& b) { return a.ell > b.ell; });

    KernelTimes ktimes, mgtimes;
    int64_t batch_iters = 0, mg_batch_iters = 0;
    // large scales by multigrid-preconditioned CG (option solver = 1): a stream of right-hand sides through 16 columns
    // (vector filter: through the scalar hierarchy with the coupled operator on the mesh)
    if (job != JOB_APPLY && r.opt.solver == 1 && order_n <= 2 && r.opt.batch == MGK && r.w.mg_extra && h->mean_edge > 0.0) {
        // default split between the paths (option mg_min_ell = 0), in mean edge lengths: with 12 or more columns in
        // use the stream takes every scale from 0.5 up (tuned on configs 3-5); a call with fewer runs the 4- or
        // 8-column kernels, or leaves some of the 16 empty, and costs more per right-hand side and iteration, so
        // Jacobi-PCG keeps the smallest scales.  Measured on config 4's mesh, one field, 1 / 4 / 8 / 10 right-hand
        // sides: n = 1 breaks even near 2.5 / 2 / 1.5 / 1.3 edge lengths, n = 2 (whose Jacobi iterations grow with
        // l^2) near 1.2 / 1 / below 1 / below 1.
        const size_t cols = rhs.size() * (r.vec ? 2 : 1);
        const double dflt = cols >= 12 ? (order_n == 1 ? MG_MIN_ELL_N1 : MG_MIN_ELL_N2)
                          : order_n == 1 ? (cols > 4 ? 1.5 : 2.5)
                                         : 1.0;
        const double min_ell = (r.opt.mg_min_ell > 0.0 ? r.opt.mg_min_ell : dflt) * h->mean_edge;
        size_t n_big = 0;
        while (n_big < rhs.size() && rhs[n_big].ell >= min_ell) ++n_big;
        if (n_big > 0) {
            std::vector<Rhs> big(rhs.begin(), rhs.begin() + (ptrdiff_t)n_big);
            Run rm = r;
            rm.mg = true;
            // sweeps per side of the cycle: n = 1 (1, MG_NU_L1, MG_NU_COARSE) as tuned on config 4; n = 2 needs the
            // stronger smoother: what V leaves of a rough residual enters B = V M V squared
            rm.mg_nu[0] = order_n == 1 ? 1 : MG_NU0_N2;
            rm.mg_nu[1] = order_n == 1 ? MG_NU_L1 : MG_NU1_N2;
            rm.mg_nu[2] = MG_NU_COARSE;
            if (const char* e = getenv("IF_MG_NU")) {   // tuning runs: "nu0,nu1,nu2"
                int a0 = 0, a1 = 0, a2 = 0;
                if (sscanf(e, "%d,%d,%d", &a0, &a1, &a2) == 3 && a0 >= 1 && a1 >= 1 && a2 >= 1 && a0 <= MG_MAX_NU &&
                    a1 <= MG_MAX_NU && a2 <= MG_MAX_NU) { rm.mg_nu[0] = a0; rm.mg_nu[1] = a1; rm.mg_nu[2] = a2; }
            }
            // few right-hand sides: the 8- and 4-column variants of every kernel of the cycle (as on the Jacobi path)
            const int Kmg = pick_k(MGK, big.size() * (r.vec ? 2 : 1));
            rc = Kmg == 4 ? solve_all<4>(rm, job, d_fields, big, n_ells, d_out, poll, &mgtimes, &mg_batch_iters)
               : Kmg == 8 ? solve_all<8>(rm, job, d_fields, big, n_ells, d_out, poll, &mgtimes, &mg_batch_iters)
                          : solve_all<MGK>(rm, job, d_fields, big, n_ells, d_out, poll, &mgtimes, &mg_batch_iters);
            if (rc != IF_OK) { cudaStreamSynchronize(r.st); return rc; }
            rhs.erase(rhs.begin(), rhs.begin() + (ptrdiff_t)n_big);
            batch_iters += mg_batch_iters;
        }
    }
    const int K = pick_k(r.opt.batch, rhs.size() * (r.vec ? 2 : 1));
    if (job == JOB_APPLY) {
        rc = K == 4 ? apply_all<4>(r, d_fields, rhs, n_ells, d_out)
           : K == 8 ? apply_all<8>(r, d_fields, rhs, n_ells, d_out)
                    : apply_all<16>(r, d_fields, rhs, n_ells, d_out);
    } else if (!rhs.empty()) {
        int64_t jac_iters = 0;
        rc = K == 4 ? solve_all<4>(r, job, d_fields, rhs, n_ells, d_out, poll, &ktimes, &jac_iters)
           : K == 8 ? solve_all<8>(r, job, d_fields, rhs, n_ells, d_out, poll, &ktimes, &jac_iters)
                    : solve_all<16>(r, job, d_fields, rhs, n_ells, d_out, poll, &ktimes, &jac_iters);
        batch_iters += jac_iters;
    }
    if (rc != IF_OK) { cudaStreamSynchronize(r.st); return rc; }
    if (job == JOB_SPECTRUM) {
        IF_CUDA_TRY(cudaMemcpyAsync(r.w.ells, ells, (size_t)n_ells * sizeof(double), cudaMemcpyHostToDevice, r.st));
        const double* e_src = r.w.energy;
        if (pairs) {
            const int np = (n_fields / 2) * n_ells;
            k_pair_sum<<<(np + 127) / 128, 128, 0, r.st>>>(r.w.energy, n_fields / 2, n_ells, r.w.epair);
            IF_LAUNCH_CHECK();
            e_src = r.w.epair;
        }
        const int nb = n_out_fields * (n_ells - 1);
        k_spectrum<<<(nb + 127) / 128, 128, 0, r.st>>>(e_src, r.w.ells, n_out_fields, n_ells, r.w.k_mid, r.w.E);
        IF_LAUNCH_CHECK();
    }
    IF_CUDA_TRY(cudaEventRecord(t1, r.st));

    // IF_FLAG_TRUE_RESIDUAL (if_filter, low-pass output): one operator application per returned field, after the
    // timed part.  The workspace is laid out afresh (column compaction may have re-used buffers for narrower layouts).
    const bool want_true = job == JOB_FILTER && stats && stats->true_res && (r.opt.flags & IF_FLAG_TRUE_RESIDUAL) &&
                           !(r.opt.flags & IF_FLAG_HIGHPASS);
    std::vector<double> h_true;
    if (want_true) {
        r.w = layout_workspace(h, order_n, r.opt.batch, d_ws);
        r.mg = false;
        std::vector<Rhs> all;
        for (int f = 0; f < (r.vec ? n_fields / 2 : n_fields); ++f)
            for (int j = 0; j < n_ells; ++j) all.push_back(Rhs{ells[j], f, j});
        const int KB = r.opt.batch;
        rc = KB == 4 ? true_residuals<4>(r, d_fields, all, n_ells, d_out, r.w.E)
           : KB == 8 ? true_residuals<8>(r, d_fields, all, n_ells, d_out, r.w.E)
                     : true_residuals<16>(r, d_fields, all, n_ells, d_out, r.w.E);
        if (rc != IF_OK) return rc;
        h_true.resize((size_t)R);
        IF_CUDA_TRY(cudaMemcpyAsync(h_true.data(), r.w.E, (size_t)R * 8, cudaMemcpyDeviceToHost, r.st));
    }

    // results back to the host (small), then one synchronisation
    std::vector<int32_t> h_status((size_t)R, 0), h_iters((size_t)R, 0);
    std::vector<double> h_relres((size_t)R, 0.0);
    if (job != JOB_APPLY) {
        IF_CUDA_TRY(cudaMemcpyAsync(h_status.data(), r.w.status, (size_t)R * 4, cudaMemcpyDeviceToHost, r.st));
        IF_CUDA_TRY(cudaMemcpyAsync(h_iters.data(), r.w.iters, (size_t)R * 4, cudaMemcpyDeviceToHost, r.st));
        IF_CUDA_TRY(cudaMemcpyAsync(h_relres.data(), r.w.relres, (size_t)R * 8, cudaMemcpyDeviceToHost, r.st));
    }
    if (job == JOB_SPECTRUM) {
        if (energy) IF_CUDA_TRY(cudaMemcpyAsync(energy, pairs ? r.w.epair : r.w.energy, (size_t)n_out_fields * n_ells * 8, cudaMemcpyDeviceToHost, r.st));
        if (k_mid) IF_CUDA_TRY(cudaMemcpyAsync(k_mid, r.w.k_mid, (size_t)(n_ells - 1) * 8, cudaMemcpyDeviceToHost, r.st));
        if (E) IF_CUDA_TRY(cudaMemcpyAsync(E, r.w.E, (size_t)n_out_fields * (n_ells - 1) * 8, cudaMemcpyDeviceToHost, r.st));
    }
    IF_CUDA_TRY(cudaStreamSynchronize(r.st));
    int result = IF_OK;
    for (int64_t i = 0; i < R; ++i) if (h_status[(size_t)i] != 0) result = IF_WNOTCONVERGED;
    if (stats) {
        float ms = 0.f;
        IF_CUDA_TRY(cudaEventElapsedTime(&ms, t0, t1));
        stats->seconds = ms * 1e-3;
        stats->batch_iters = batch_iters;
        stats->rhs_iters = 0;
        stats->spmm_seconds = ktimes.samples ? 1e-3 * ktimes.ms[0] / (double)ktimes.samples : 0.0;
        stats->update_seconds = ktimes.samples ? 1e-3 * ktimes.ms[1] / (double)ktimes.samples : 0.0;
        stats->kernel_samples = ktimes.samples;
        for (int g = 0; g < 8; ++g)
            stats->mg_kernel_seconds[g] = mgtimes.samples && g < TIMER_GROUPS ? 1e-3 * mgtimes.ms[g] / (double)mgtimes.samples : 0.0;
        stats->mg_samples = mgtimes.samples;
        stats->mg_batch_iters = mg_batch_iters;
        for (int64_t i = 0; i < R; ++i) {
            stats->rhs_iters += h_iters[(size_t)i];
            if (stats->iters) stats->iters[i] = h_iters[(size_t)i];
            if (stats->status) stats->status[i] = h_status[(size_t)i];
            if (stats->rel_res) stats->rel_res[i] = h_relres[(size_t)i];
            if (want_true) stats->true_res[i] = h_true[(size_t)i];
        }
    }
    return result;
}

}  // namespace
}  // namespace ifl

using namespace ifl;

extern "C" int if_workspace_bytes(if_handle h, int order_n, int batch, size_t* bytes) {
    if (!h || !bytes || order_n < 1 || order_n > 4) return IF_EINVAL;
    if (batch == 0) batch = h->opt.batch;
    if (batch != 4 && batch != 8 && batch != 16) return IF_EINVAL;
    *bytes = layout_workspace(h, order_n, batch, nullptr).bytes;
    return IF_OK;
}

extern "C" int if_filter(if_handle h, const double* d_fields, int n_fields, const double* ells, int n_ells, int order_n,
                         double* d_out, void* d_workspace, size_t ws_bytes, void* cuda_stream, const if_options* opt,
                         if_stats* stats) {
    return run_job(h, JOB_FILTER, d_fields, n_fields, ells, n_ells, order_n, d_out, nullptr, nullptr, nullptr,
                   d_workspace, ws_bytes, cuda_stream, opt, stats);
}

extern "C" int if_spectrum(if_handle h, const double* d_fields, int n_fields, const double* ells, int n_ells,
                           int order_n, double* energy, double* k_mid, double* E, void* d_workspace, size_t ws_bytes,
                           void* cuda_stream, const if_options* opt, if_stats* stats) {
    return run_job(h, JOB_SPECTRUM, d_fields, n_fields, ells, n_ells, order_n, nullptr, energy, k_mid, E, d_workspace,
                   ws_bytes, cuda_stream, opt, stats);
}

extern "C" int if_spectrum_host(if_handle h, const double* h_fields, int n_fields, const double* ells, int n_ells,
                                int order_n, double* energy, double* k_mid, double* E, void* d_workspace,
                                size_t ws_bytes, void* cuda_stream, const if_options* opt, if_stats* stats) {
    if (!h || !h_fields || n_fields < 1 || !d_workspace || order_n < 1 || order_n > 4) return IF_EINVAL;
    Options o;
    int rc = resolve_options(opt, &h->opt, &o);
    if (rc != IF_OK) return rc;
    const size_t base = layout_workspace(h, order_n, o.batch, nullptr).bytes;
    const size_t fbytes = (size_t)n_fields * (size_t)h->n_vert * sizeof(double);
    if (ws_bytes < base + fbytes) return IF_EWORKSPACE;
    double* d_fields = reinterpret_cast<double*>(static_cast<char*>(d_workspace) + base);
    IF_CUDA_TRY(cudaMemcpyAsync(d_fields, h_fields, fbytes, cudaMemcpyHostToDevice,
                                static_cast<cudaStream_t>(cuda_stream)));
    return run_job(h, JOB_SPECTRUM, d_fields, n_fields, ells, n_ells, order_n, nullptr, energy, k_mid, E, d_workspace,
                   base, cuda_stream, opt, stats);
}

extern "C" int if_apply(if_handle h, const double* d_fields, int n_fields, const double* ells, int n_ells, int order_n,
                        double* d_out, void* d_workspace, size_t ws_bytes, void* cuda_stream, const if_options* opt) {
    return run_job(h, JOB_APPLY, d_fields, n_fields, ells, n_ells, order_n, d_out, nullptr, nullptr, nullptr,
                   d_workspace, ws_bytes, cuda_stream, opt, nullptr);
}

extern "C" int if_mesh_multigrid_info(if_handle h, int* n_levels, int64_t* rows, int64_t* nnz, int64_t* p_nnz,
                                      double* build_seconds, int* sweeps) {
    if (!h) return IF_EINVAL;
    if (n_levels) *n_levels = h->mg_levels;
    for (int l = 0; l < MG_MAX_LEVELS; ++l) {
        const bool on = l < h->mg_levels;
        if (rows) rows[l] = on ? h->mg[l].n : 0;
        if (nnz) nnz[l] = on ? h->mg[l].nnz : 0;
        if (p_nnz) p_nnz[l] = on ? h->mg[l].p_nnz : 0;
    }
    if (build_seconds) *build_seconds = h->mg_build_seconds;
    if (sweeps) {
        const int s[6] = {1, MG_NU_L1, MG_NU_COARSE, MG_NU0_N2, MG_NU1_N2, MG_NU_COARSE};
        for (int i = 0; i < 6; ++i) sweeps[i] = s[i];
    }
    return IF_OK;
}
