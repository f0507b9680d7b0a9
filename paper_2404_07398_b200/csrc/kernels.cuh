// Device code of the solving phase: batched multi-right-hand-side Jacobi-PCG on
//     A_c x_c = M phi_c,   A_c = M + c_c S (M^-1 S)^(n-1),   c_c = gamma l_c^(2n)
// for K = 4, 8 or 16 columns c at once, every column with its own scale l_c, field, alpha, beta and stop time.
//
// Layout: work vectors are [row][K] fp64 (K = 16: one 128-byte line per row), rows in the internal order.
// A row is handled by K/2 threads, each owning two adjacent columns (double2 = 16-byte accesses), so a warp
// covers 64/K rows and every gather of a neighbour row is one contiguous K*8-byte segment.
//
// CG is carried in the preconditioned residual z = r/d (d = diag(A_c), Jacobi):
//   kernel A (k_spmm, fused):  p' = z + beta p ;  x += alpha_prev p ;  q = A_c p' ;  partial p'.q
//   kernel B (k_update):       z -= alpha q/d ;  partial rho' = sum d z^2 = r.z  and  ||r||^2 = sum (d z)^2
// Per-column scalars (alpha, beta, rho, done flags) live in a device control block and are produced by the
// last block to finish each kernel (single-pass, fixed-order, deterministic grid reduction).
//
// Kernel A is tiled for sm_100a: a persistent CTA walks tiles of TILE_ROWS consecutive rows.  Per tile one thread
// issues bulk async copies (TMA, cp.async.bulk + mbarrier complete_tx) that land the tile of z and p, the tile's
// slice of the SELL matrix (with tile-local column ids built by if_prepare) and its diagonals in shared memory;
// meanwhile all threads fetch the tile's halo (the out-of-tile neighbour rows, listed by if_prepare) from L2
// into the same shared array and x into registers.  The CTA forms p' in place, hands it back with a bulk store,
// and the gather of the neighbours' p' is then branch-free shared-memory traffic (rows are in
// space-filling-curve order, so the halo is small).
#pragma once

#include "common.cuh"

namespace ifl {
namespace {

constexpr int KMAX = 16;
constexpr int BLOCK = 256;
constexpr int WCAP = 8;   // SELL slots per row that fit the shared-memory matrix slice (wider tiles read global)

struct MeshView {
    const int64_t* __restrict__ chunk_ptr;
    const int32_t* __restrict__ col;
    const double* __restrict__ val;
    const double* __restrict__ tval;        // vector filter: T entries beside val = D~ entries (null for scalar fields)
    const double* __restrict__ area;
    const double* __restrict__ inv_area;
    const double* __restrict__ sdiag;
    const double* __restrict__ gdiag;
    const double* __restrict__ gdiag3;
    const double* __restrict__ gdiag4;
    const int32_t* __restrict__ perm;
    const int32_t* __restrict__ lcol;       // tile-local column ids (tile row, or TILE_ROWS + halo slot)
    const int32_t* __restrict__ halo_rows;  // [tiles][HALO_CAP] out-of-tile rows each tile gathers from
    const int32_t* __restrict__ tile_desc;  // [tiles+1][16] first slot, slots, halo rows | -1, slice offsets
    int64_t nv;
    int64_t n_chunks;
    int log2c;
};

// diag(S (M^-1 S)^(n-1)) for the Jacobi preconditioner of order n
__device__ __forceinline__ const double* jacobi_diag(const MeshView& m, int order_n) {
    return order_n == 1 ? m.sdiag : order_n == 2 ? m.gdiag : order_n == 3 ? m.gdiag3 : m.gdiag4;
}

// per-column parameters of a (re)start, passed by value to k_init
struct StartParams {
    double c[KMAX];
    double c1[KMAX];      // multigrid path (see Ctrl::c1)
    int field[KMAX];
    int rhs[KMAX];
};

// one right-hand side of the device-side queue (multigrid stream with the column turnover on the device)
struct QEntry {
    double c, c1;
    int field, rhs;
};

struct Ctrl {
    double c[KMAX];       // gamma l^(2n)
    double alpha[KMAX];
    double beta[KMAX];
    double rho[KMAX];
    double bb[KMAX];      // ||M phi||^2
    double rr[KMAX];      // ||r||^2 (recursive)
    int field[KMAX];      // field of the column, -1 = empty column
    int rhs[KMAX];        // f * n_ells + j of the column
    int done[KMAX];
    int epoch[KMAX];      // bumped every time a column is (re)started: lets the host match a snapshot to a RHS
    int status[KMAX];
    int iters[KMAX];
    double c1[KMAX];      // multigrid path: coefficient of the cycle's operator K = M + c1 S (n = 1: c; n = 2: sqrt(c))
    int starting[KMAX];   // multigrid path: the column was (re)started (k_mg_start): its first iteration has alpha = 1
                          // (forms r0), then rho = r0.z0, beta = 0, nothing counted
    int cur_r;            // multigrid path: which residual buffer holds r (flipped with cur_p)
    int pair_mode;        // vector filter: columns (2i, 2i+1) are the (u, v) of ONE system: its dot products are the
                          // sums over both columns, so both share alpha, beta and the stop decision
    int all_done;
    int cur_p;            // which direction buffer holds the current direction (flipped at the end of every iteration)
    int max_iter;
    int pad_;
    double tol2;
    long long total_iters;   // fused iterations executed while some column was active
    unsigned int ticket[4];
    // column turnover on the device (multigrid stream, k_turn_plan): the queue position, which columns hold a
    // right-hand side, what this iteration's turnover finalises and starts, and what the host reads back
    int q_next, q_total;
    int rhs_stride;       // vector filter: output slot of the v component = that of u + rhs_stride (= n_ells)
    int pad2_;
    int occupied[KMAX];
    unsigned int turn_fin, turn_start;
    StartParams turn_sp;
    int snap[4];          // {slots holding a right-hand side, of those still running, q_next, 0} after the turnover
    int cmap[KMAX];       // compaction of the stream's tail (k_mg_compact_plan): new column j <- old column cmap[j], -1 = empty
};

// what the host reads back every check_every iterations
struct Snapshot {
    int done[KMAX];
    int epoch[KMAX];
};

// mask arguments of the start / end-of-column kernels: these values mean "what k_turn_plan left in the control block"
constexpr unsigned MASK_TURN_FIN = 0x80000000u;     // ctrl->turn_fin
constexpr unsigned MASK_TURN_START = 0x40000000u;   // ctrl->turn_start, parameters from ctrl->turn_sp

enum Mode { MODE_PLAIN = 0, MODE_CG1 = 1, MODE_CG2A = 2, MODE_CG2B = 3, MODE_AX = 4, MODE_MGR = 5, MODE_MGR0 = 6 };
// MODE_AX (multigrid path, level 0): v = in0 (gathered), r = in1 (own rows), K = M + c1 S per column (Ctrl::c1), and with
// SpmmArgs::scale_inv_area as the sub-mode:  0: out0 = K v ;  1: out0 = r - K v ;  2: out0 = v + omega (r - K v)/d
// (omega = SpmmArgs::omega, the Jacobi damping of the multigrid smoother on level 0);  3: as 2, the last sweep of
// the preconditioner z = B r, plus the CG bookkeeping of kernel B (rho' = r.z, ||r||^2, beta, stop test);
// 5 (n = 2, B = V M V): y = v + omega (r - K v)/d is the end of the first cycle, out0 = M y goes to the second one,
// and the bookkeeping uses rho' = y.M y = r.(V M V r) and ||r||^2.
// MODE_MGR0: MODE_MGR without the residual update (the second cycle of n = 2 starts from w = M y): e = omega w/d,
// t = w - K e; only one vector arrives by bulk copy.
// MODE_MGR (multigrid path, level 0): the residual update of CG, the first Jacobi sweep of the preconditioner (from a
// zero guess) and the residual of that sweep in one pass.  in0 = r, in1 = q (both gathered: tile by bulk copy, halo
// rows from L2), alpha from the control block:  r' = r - alpha q -> x ;  e = omega r'/d -> out1 (unless out1 is
// null: k_mg_prolong0 forms it again) ;  t = r' - A e -> out0.
// r' goes to a second buffer (x), not over r: other blocks still read r and q for their halo rows.

__device__ __forceinline__ double2 ld2(const double* __restrict__ p, int64_t i) {
    return *reinterpret_cast<const double2*>(p + i);
}
__device__ __forceinline__ void st2(double* __restrict__ p, int64_t i, double2 v) {
    *reinterpret_cast<double2*>(p + i) = v;
}

// 1/d for d > 0 in the normal range: hardware seed (2^-23) and two Newton steps (full fp64 precision, ~1 ulp).
// A fp64 division costs about five times as many instructions and made the streaming update kernel (kernel B) issue-bound.
__device__ __forceinline__ double rcp_pos(double d) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
    double e = fma(-d, r, 1.0);
    r = fma(r, e, r);
    e = fma(-d, r, 1.0);
    return fma(r, e, r);
}

// ---- bulk async copy (TMA) and mbarrier wrappers (PTX ISA: cp.async.bulk, mbarrier)
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    const uint32_t addr = smem_u32(bar);
    uint32_t ok;
    do {
        asm volatile(
            "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
            : "=r"(ok) : "r"(addr), "r"(parity) : "memory");
    } while (!ok);
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void bulk_load(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_store(void* dst_gmem, const void* src_smem, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst_gmem), "r"(smem_u32(src_smem)),
                 "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_prefetch_l2(const void* src_gmem, uint32_t bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src_gmem), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

// Fixed-order block reduction of NV double2 accumulators per thread over the threads owning the same column
// pair, then a ticket: the last block to arrive sums all blocks' partials in block order.
// Returns true in the last block, with the totals of value set j, column c in tot[j*KMAX + c] (shared memory).
template <int K, int NV, int NT = BLOCK>
__device__ __forceinline__ bool grid_reduce(const double2 (&acc)[NV], double* __restrict__ partials,
                                            unsigned int* ticket, double* tot /* shared [NV*KMAX] */) {
    constexpr int TPR = K / 2;
    __shared__ double2 red[NT];
    __shared__ bool is_last;
    const int tid = threadIdx.x;
    for (int j = 0; j < NV; ++j) {
        red[tid] = acc[j];
        __syncthreads();
        if (tid < TPR) {
            double2 s = red[tid];
            for (int i = tid + TPR; i < NT; i += TPR) { s.x += red[i].x; s.y += red[i].y; }
            partials[((size_t)j * gridDim.x + blockIdx.x) * K + 2 * tid] = s.x;
            partials[((size_t)j * gridDim.x + blockIdx.x) * K + 2 * tid + 1] = s.y;
        }
        __syncthreads();
    }
    if (tid == 0) {
        __threadfence();
        unsigned int t = atomicAdd(ticket, 1u);
        is_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return false;
    __threadfence();
    double* redd = reinterpret_cast<double*>(red);   // [NT] doubles (uses half of red)
    constexpr int LANES = NT / K;                  // threads per column
    for (int j = 0; j < NV; ++j) {
        const int c = tid % K, lane = tid / K;
        double s = 0.0;
        for (unsigned b = lane; b < gridDim.x; b += LANES)
            s += __ldcg(&partials[((size_t)j * gridDim.x + b) * K + c]);
        redd[tid] = s;
        __syncthreads();
        if (tid < K) {
            double t = 0.0;
            for (int i = 0; i < LANES; ++i) t += redd[i * K + tid];
            tot[j * KMAX + tid] = t;
        }
        __syncthreads();
    }
    if (tid == 0) *ticket = 0u;
    return true;
}

// Fixed-order grid reduction for the kernels in which a thread owns ROWS and carries one accumulator per column (the
// start and the end of a column: few columns of the K are touched, so threads are spread over rows, not over column
// pairs).  Per column in `mask`: xor tree inside a warp, the warps in order, partials[block][K], a ticket, and the last
// block adds the blocks' partial sums as grid_reduce does.  Returns true in the last block with the totals in tot[c].
template <int K, int NT = BLOCK>
__device__ __forceinline__ bool grid_reduce_cols(const double (&acc)[K], unsigned mask, double* __restrict__ partials,
                                                 unsigned int* ticket, double* tot /* shared [KMAX] */) {
    __shared__ double wsum[NT / 32][K];
    __shared__ double redd[NT];
    __shared__ bool is_last;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
#pragma unroll
    for (int c = 0; c < K; ++c) {
        if (!((mask >> c) & 1u)) continue;
        double s = acc[c];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (lane == 0) wsum[warp][c] = s;
    }
    __syncthreads();
    if (tid < K) {
        double s = 0.0;
        if ((mask >> tid) & 1u)
            for (int w = 0; w < NT / 32; ++w) s += wsum[w][tid];
        partials[(size_t)blockIdx.x * K + tid] = s;
    }
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        unsigned int t = atomicAdd(ticket, 1u);
        is_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return false;
    __threadfence();
    constexpr int LANES = NT / K;                  // threads per column
    const int c = tid % K, ln = tid / K;
    double s = 0.0;
    for (unsigned b = ln; b < gridDim.x; b += LANES) s += __ldcg(&partials[(size_t)b * K + c]);
    redd[tid] = s;
    __syncthreads();
    if (tid < K) {
        double t = 0.0;
        for (int i = 0; i < LANES; ++i) t += redd[i * K + tid];
        tot[tid] = t;
    }
    __syncthreads();
    if (tid == 0) *ticket = 0u;
    return true;
}

// Fixed-order grid reduction for k_mg_start: thread tid keeps column pair `pair` (slot tid % PP of the compacted pair
// list, PP a power of two, slots >= P idle).  Per slot the threads are added in thread order, partials[block][K], a
// ticket, and the last block adds the blocks' partial sums as grid_reduce does (columns of idle pairs come out as 0).
template <int K, int NT = BLOCK>
__device__ __forceinline__ bool grid_reduce_pairs(double2 acc, int PP, int P, int pair, double* __restrict__ partials,
                                                  unsigned int* ticket, double* tot /* shared [KMAX] */) {
    __shared__ double2 red[NT];
    __shared__ bool is_last;
    const int tid = threadIdx.x;
    red[tid] = acc;
    if (tid < K) partials[(size_t)blockIdx.x * K + tid] = 0.0;
    __syncthreads();
    if (tid < P) {
        double2 s = red[tid];
        for (int i = tid + PP; i < NT; i += PP) { s.x += red[i].x; s.y += red[i].y; }
        partials[(size_t)blockIdx.x * K + 2 * pair] = s.x;
        partials[(size_t)blockIdx.x * K + 2 * pair + 1] = s.y;
    }
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        unsigned int t = atomicAdd(ticket, 1u);
        is_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return false;
    __threadfence();
    double* redd = reinterpret_cast<double*>(red);
    constexpr int LANES = NT / K;                  // threads per column
    const int c = tid % K, ln = tid / K;
    double s = 0.0;
    for (unsigned b = ln; b < gridDim.x; b += LANES) s += __ldcg(&partials[(size_t)b * K + c]);
    __syncthreads();
    redd[tid] = s;
    __syncthreads();
    if (tid < K) {
        double t = 0.0;
        for (int i = 0; i < LANES; ++i) t += redd[i * K + tid];
        tot[tid] = t;
    }
    __syncthreads();
    if (tid == 0) *ticket = 0u;
    return true;
}

// CG bookkeeping after z = B r (run by the last block of a grid reduction; tot = rho' per column, then ||r||^2):
// beta = rho'/rho, stop test, iteration count -- the same rules as the tail of k_update.  A column that was
// (re)started (Ctrl::starting, k_mg_start) has just had r0 and z0 = B r0 formed: rho = rho', beta = 0, nothing counted.
template <int K>
__device__ __forceinline__ void cg_bookkeeping(Ctrl* __restrict__ ctrl, const double* tot) {
    __shared__ int any_active;
    const int tid = threadIdx.x;
    if (tid == 0) any_active = 0;
    __syncthreads();
    if (tid < K) {
        if (!ctrl->done[tid]) {
            const bool start = ctrl->starting[tid] != 0;
            // (vector filter: the two columns of a pair are one system -- its dot products are the sums over both)
            const int ta = ctrl->pair_mode ? (tid & ~1) : tid, tb = ctrl->pair_mode ? (tid | 1) : tid;
            const double w2 = ctrl->pair_mode ? 1.0 : 0.5;      // (ta == tb without pairs: the value itself)
            const double rho_new = w2 * (tot[ta] + tot[tb]), rr = w2 * (tot[KMAX + ta] + tot[KMAX + tb]);
            const int it = start ? 0 : ctrl->iters[tid] + 1;
            ctrl->iters[tid] = it;
            ctrl->rr[tid] = rr;
            double be = start ? 0.0 : rho_new / ctrl->rho[tid];
            ctrl->rho[tid] = rho_new;
            ctrl->starting[tid] = 0;
            int dn = 0;
            if (!isfinite(rr)) { dn = 1; ctrl->status[tid] = 2; }
            else if (rr <= ctrl->tol2 * ctrl->bb[tid]) { dn = 1; ctrl->status[tid] = 0; }
            else if (!isfinite(be) || !(rho_new > 0.0)) { dn = 1; ctrl->status[tid] = 2; }
            else if (it >= ctrl->max_iter) { dn = 1; ctrl->status[tid] = 1; }
            if (dn) { be = 0.0; ctrl->done[tid] = 1; }
            ctrl->beta[tid] = be;
            if (!dn) atomicOr(&any_active, 1);
        } else {
            ctrl->beta[tid] = 0.0;
        }
    }
    __syncthreads();
    if (tid == 0) {
        ctrl->all_done = !any_active;
        ctrl->total_iters += 1;
        ctrl->cur_p ^= 1;
        ctrl->cur_r ^= 1;
    }
}

// ------------------------------------------------------------------------------------------- kernel A
struct SpmmArgs {
    const double* in0;   // PLAIN: x        CG1/CG2A: z        CG2B: t            (the gathered vector)
    const double* in1;   //                 CG1/CG2A: p_old    CG2B: p (current)
    double* x;           //                 CG1/CG2A: x (in place)                        MGR: r' (new residual)
    double* out0;        // PLAIN: y        CG1: q             CG2A: t            CG2B: q
    double* out1;        //                 CG1/CG2A: p_new
    int scale_inv_area;  // PLAIN: multiply the row result by 1/A_v
    int p_select;        // CG1/CG2A/CG2B inside the iteration: in1 and out1 are the two direction buffers p[0], p[1] and
                         // the kernel picks old/new from ctrl->cur_p (the buffer holding the current direction), so a
                         // captured graph stays valid whatever iteration it resumes at
    double omega;        // AX, sub-mode 2: damping
    double omega2;       // MGR / MGR0 with two or more sweeps before the coarse correction: out0 = e + omega2 (r' - K e)/d
                         // (the second sweep) instead of the residual t = r' - K e; 0: the residual
    int r_select;        // multigrid path inside the iteration: the residual is double-buffered (r[0], r[1]) and picked on
                         // the device from ctrl->cur_r.  MGR: (in0, x) = (r[0], r[1]) -> reads r[cur_r], writes r[cur_r^1];
                         // AX: (in1, x) = (r[0], r[1]) -> reads r[cur_r^1] (the residual MGR has just written)
};

// One row of the staged SpMM: all column ids and values of the row first, then all W gathers from the shared
// tile, then the multiply-adds on two accumulators -- one shared-memory latency per phase instead of one per entry.
// VEC (vector filter): the thread's two columns are the (u, v) of one system and every entry carries the
// pair (D~_ij, T_ij):  s_u += D~ p_u + T p_v ;  s_v += D~ p_v - T p_u.
template <int W, int TPR, bool VEC>
__device__ __forceinline__ double2 gather_row(const int32_t* __restrict__ scol_row, const double* __restrict__ sval_row,
                                              const double* __restrict__ stval_row, const double2* __restrict__ sa, int l) {
    int2 cj[W / 2];
    double2 vj[W / 2], tj[VEC ? W / 2 : 1];
#pragma unroll
    for (int k = 0; k < W / 2; ++k) {
        cj[k] = reinterpret_cast<const int2*>(scol_row)[k];
        vj[k] = reinterpret_cast<const double2*>(sval_row)[k];
        if (VEC) tj[VEC ? k : 0] = reinterpret_cast<const double2*>(stval_row)[k];
    }
    double2 g[W];
#pragma unroll
    for (int k = 0; k < W / 2; ++k) {
        g[2 * k] = sa[cj[k].x * TPR + l];
        g[2 * k + 1] = sa[cj[k].y * TPR + l];
    }
    double2 s0 = {0.0, 0.0}, s1 = {0.0, 0.0};
#pragma unroll
    for (int k = 0; k < W / 2; ++k) {
        s0.x = fma(vj[k].x, g[2 * k].x, s0.x);     s0.y = fma(vj[k].x, g[2 * k].y, s0.y);
        s1.x = fma(vj[k].y, g[2 * k + 1].x, s1.x); s1.y = fma(vj[k].y, g[2 * k + 1].y, s1.y);
        if (VEC) {
            const double2 t = tj[VEC ? k : 0];
            s0.x = fma(t.x, g[2 * k].y, s0.x);      s0.y = fma(-t.x, g[2 * k].x, s0.y);
            s1.x = fma(t.y, g[2 * k + 1].y, s1.x);  s1.y = fma(-t.y, g[2 * k + 1].x, s1.y);
        }
    }
    s0.x += s1.x;
    s0.y += s1.y;
    return s0;
}

// dynamic shared memory of k_spmm: SpmmCfg<K>::STAGES stages of
//   [gathered vector: T tile rows + HALO_CAP halo rows][second vector: T rows][val slice][col slice][S_vv][A_v | 1/A_v]
// then a ring of four tile descriptors and one mbarrier per stage
#ifndef IF_SPMM_BLOCK
#define IF_SPMM_BLOCK 512
#endif
#ifndef IF_SPMM_STAGES
#define IF_SPMM_STAGES 3
#endif
#ifndef IF_SPMM_MINB
#define IF_SPMM_MINB 1
#endif
constexpr int SPMM_BLOCK = IF_SPMM_BLOCK;
constexpr int SPMM_STAGES = IF_SPMM_STAGES;
// Threads per CTA, CTAs per SM and pipeline stages of k_spmm.  The 16-column CG kernels fill an SM with one 512-thread
// CTA and three stages (186 KB).  The narrower layouts of the compacted tail have smaller stages and are bound by
// per-tile fixed costs, not by HBM: two 256-thread CTAs per SM overlap each other's stalls (K = 8 with two stages to
// fit shared memory).  The multigrid sweeps (AX, MGR0) move fewer bytes per tile than kernel A and were bound the
// same way as one CTA (0.57 of the copy bandwidth): their second vector -- needed for the tile's own rows only,
// never gathered -- goes through registers instead of a shared-memory region (REGB), the stage shrinks to 46 KB, and
// they run as two 256-thread CTAs per SM with two stages each (0.909 -> 0.776 ms per sweep on config 4).  MGR, which
// also reads q and stores r', lost by the same change in both forms tried (below) and stays as it was.
// MGR the same way (q by direct loads, r' stored from registers and read back by its thread): measured on config 4,
// 1.075 -> 1.235 ms (128 registers with spills at 256 threads x 2 CTAs) -- off.
#ifndef IF_MGR_REGB
#define IF_MGR_REGB 0
#endif
template <int K, int MODE> struct SpmmCfg {
    static constexpr bool REGB = (MODE == MODE_AX || MODE == MODE_MGR0 || (MODE == MODE_MGR && IF_MGR_REGB));
    static constexpr bool WIDE1 = (K == 16) && !REGB;              // one 512-thread CTA per SM
    static constexpr int NT = WIDE1 ? SPMM_BLOCK : 256;
    static constexpr int MINB = WIDE1 ? IF_SPMM_MINB : 2;
    static constexpr int STAGES = (K == 8 || (K == 16 && REGB)) ? 2 : SPMM_STAGES;
};

template <int K, int MODE, bool VEC = false> struct TileSmem {
    static constexpr int T = TILE_ROWS;
    // tile-sized vector regions of a stage: the gathered vector (+ halo), and the second vector unless it goes
    // through registers
    static constexpr int NVEC = (MODE == MODE_PLAIN || SpmmCfg<K, MODE>::REGB) ? 1 : 2;   // (MGR0 as non-REGB would keep 2)
    static constexpr int NLOAD = (MODE == MODE_PLAIN || MODE == MODE_MGR0 || SpmmCfg<K, MODE>::REGB) ? 1 : 2;   // vectors that arrive by bulk copy
    static constexpr size_t vec_bytes = (size_t)T * K * sizeof(double);
    static constexpr size_t off_b = (size_t)(T + HALO_CAP) * K * sizeof(double);
    static constexpr size_t off_val = off_b + (NVEC - 1) * vec_bytes;
    static constexpr size_t off_tval = off_val + (size_t)T * WCAP * sizeof(double);   // vector filter: T entries
    static constexpr size_t off_col = off_tval + (VEC ? (size_t)T * WCAP * sizeof(double) : 0);
    static constexpr size_t off_dg = off_col + (size_t)T * WCAP * sizeof(int32_t);   // S_vv of the tile's rows
    static constexpr size_t off_ar = off_dg + (size_t)T * sizeof(double);            // A_v or 1/A_v
    static constexpr size_t stage_bytes = off_ar + (size_t)T * sizeof(double);
    static constexpr size_t off_desc = SpmmCfg<K, MODE>::STAGES * stage_bytes;
    static constexpr size_t off_bar = off_desc + 4 * 16 * sizeof(int32_t);
    static constexpr size_t bytes = off_bar + 8 * SpmmCfg<K, MODE>::STAGES + 8;
};

// What one thread needs to issue the bulk copies of a tile (kept in registers by the issuing thread).
struct TileIssue { int64_t cp_first; int slots; int nh; };
__device__ __forceinline__ TileIssue load_issue(const int32_t* __restrict__ desc, int64_t tile) {
    const int4 v = *reinterpret_cast<const int4*>(desc + tile * 16);
    TileIssue t;
    t.cp_first = (int64_t)(uint32_t)v.x | ((int64_t)v.y << 32);
    t.slots = v.z;
    t.nh = v.w;
    return t;
}

// Software pipeline of one persistent CTA per SM (tile i being computed):
//   bulk copies (TMA) of tiles i+1 and i+2 are in flight into the other two stages,
//   x and the halo rows of tile i+1 are in flight into registers,
//   descriptors and halo row ids are fetched two tiles ahead.
// About 130 KB of loads per SM are outstanding at all times, which is what the loaded HBM latency of B200 needs.
template <int K, int MODE, bool VEC = false>
__global__ void __launch_bounds__(SpmmCfg<K, MODE>::NT, SpmmCfg<K, MODE>::MINB) k_spmm(MeshView m, Ctrl* __restrict__ ctrl,
                                                        double* __restrict__ partials, SpmmArgs a_in) {
    using SM = TileSmem<K, MODE, VEC>;
    constexpr int T = SM::T;
    constexpr int NT = SpmmCfg<K, MODE>::NT;
    constexpr int NS = SpmmCfg<K, MODE>::STAGES;         // pipeline stages
    constexpr bool REGB = SpmmCfg<K, MODE>::REGB;        // second vector through registers (bq / bcur below)
    constexpr int LA = NS - 1;                           // tiles the bulk copies run ahead of the gather
    constexpr int TPR = K / 2;
    constexpr int ROWS = NT / TPR;
    constexpr int XPT = (T * TPR + NT - 1) / NT;         // double2 elements of a tile vector per thread
    constexpr int HPT = (HALO_CAP + ROWS - 1) / ROWS;    // halo rows per thread group
    constexpr bool CG_A = (MODE == MODE_CG1 || MODE == MODE_CG2A);
    constexpr bool MGR = (MODE == MODE_MGR || MODE == MODE_MGR0);
    constexpr bool MGQ = (MODE == MODE_MGR);                      // with the residual update r' = r - alpha q
    constexpr bool AXE = (MODE == MODE_AX || MGR);                // epilogue with K = M + c1 S
    if (MODE != MODE_PLAIN && ctrl->all_done) return;
    SpmmArgs a = a_in;
    if ((CG_A || MODE == MODE_CG2B) && a.p_select) {
        // direction buffers by the device-side index: p[cur_p] is the current direction, kernel A writes the other one
        // (cur_p flips at the end of the iteration, in the last block of k_update / cg_bookkeeping)
        double* const pb[2] = {const_cast<double*>(a_in.in1), a_in.out1};
        const int cp = ctrl->cur_p;
        a.in1 = pb[CG_A ? cp : cp ^ 1];
        a.out1 = CG_A ? pb[cp ^ 1] : nullptr;
    }
    if (AXE && a.r_select) {
        const int cr = ctrl->cur_r;
        if (MGQ) {
            double* const rb[2] = {const_cast<double*>(a_in.in0), a_in.x};
            a.in0 = rb[cr];
            a.x = rb[cr ^ 1];
        } else if (MODE == MODE_AX) {
            double* const rb[2] = {const_cast<double*>(a_in.in1), a_in.x};
            a.in1 = rb[cr ^ 1];
        }
    }
    extern __shared__ __align__(128) unsigned char smem[];
    int32_t* sdesc = reinterpret_cast<int32_t*>(smem + SM::off_desc);   // [4][16] tile descriptors (ring)
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + SM::off_bar);   // one per stage
    // the per-row factor next to S_vv: A_v for q = A_v p + c S v, 1/A_v for t = M^-1 S v
    const double* __restrict__ rowfac =
        (MODE == MODE_CG2A || (MODE == MODE_PLAIN && a.scale_inv_area)) ? m.inv_area : m.area;

    const int tid = threadIdx.x;
    const int l = tid % TPR;
    const int rg = tid / TPR;                            // row group of the thread
    double2 beta = {0.0, 0.0}, alpha = {0.0, 0.0}, cc = {0.0, 0.0};
    if (MODE != MODE_PLAIN) {
        beta = ld2(ctrl->beta, 2 * l);
        alpha = ld2(ctrl->alpha, 2 * l);
        cc = ld2(AXE ? ctrl->c1 : ctrl->c, 2 * l);
    }
    const int C = 1 << m.log2c;
    const int64_t ntiles = (m.nv + T - 1) / T;
    const int64_t G = gridDim.x;
    const int64_t tile0 = blockIdx.x;

    auto issue = [&](int64_t tile, int stage, const TileIssue& ti) {   // thread 0 only
        unsigned char* st = smem + (size_t)stage * SM::stage_bytes;
        const int64_t row0 = tile * T;
        const int nrows = (int)min((int64_t)T, m.nv - row0);
        const uint32_t vbytes = (uint32_t)nrows * K * sizeof(double);
        const uint32_t dbytes = ((uint32_t)nrows * 8u + 15u) & ~15u;   // the arrays are padded by 16 bytes
        const bool staged = ti.nh >= 0 && ti.slots <= T * WCAP;
        uint64_t* bar = &bars[stage];
        mbar_expect_tx(bar, vbytes * SM::NLOAD + 2u * dbytes + (staged ? (uint32_t)ti.slots * (VEC ? 20u : 12u) : 0u));
        bulk_load(st, a.in0 + row0 * K, vbytes, bar);
        if (SM::NLOAD >= 2) bulk_load(st + SM::off_b, a.in1 + row0 * K, vbytes, bar);
        if (REGB && (MODE == MODE_AX || MODE == MODE_MGR) && a.in1) bulk_prefetch_l2(a.in1 + row0 * K, vbytes);
        bulk_load(st + SM::off_dg, m.sdiag + row0, dbytes, bar);
        bulk_load(st + SM::off_ar, rowfac + row0, dbytes, bar);
        if (staged) {
            bulk_load(st + SM::off_val, m.val + ti.cp_first, (uint32_t)ti.slots * 8u, bar);
            if (VEC) bulk_load(st + SM::off_tval, m.tval + ti.cp_first, (uint32_t)ti.slots * 8u, bar);
            bulk_load(st + SM::off_col, m.lcol + ti.cp_first, (uint32_t)ti.slots * 4u, bar);
        }
    };
    double2 hd[MGR ? HPT : 1];   // MGR: (S_vv, A_v) of the halo rows in flight
    auto load_halo = [&](const int (&idx)[HPT], int nh, double2 (&h0)[HPT], double2 (&h1)[HPT]) {
#pragma unroll
        for (int i = 0; i < HPT; ++i) {
            if (rg + i * ROWS < nh) {
                const int64_t j = idx[i];
                h0[i] = ld2(a.in0, j * K + 2 * l);
                if (CG_A || MGQ) h1[i] = ld2(a.in1, j * K + 2 * l);
                if (MGR) hd[MGR ? i : 0] = make_double2(m.sdiag[j], m.area[j]);
            }
        }
    };
    auto load_hidx = [&](int64_t tile, int (&idx)[HPT]) {
#pragma unroll
        for (int i = 0; i < HPT; ++i) {
            const int hh = rg + i * ROWS;
            idx[i] = (tile < ntiles && hh < HALO_CAP) ? m.halo_rows[tile * HALO_CAP + hh] : 0;
        }
    };
    auto load_x = [&](int64_t tile, double2 (&xv)[XPT]) {
        if (tile >= ntiles) return;
        const int64_t row0 = tile * T;
        const int nrows = (int)min((int64_t)T, m.nv - row0);
#pragma unroll
        for (int i = 0; i < XPT; ++i) {
            const int e = tid + i * NT;
            if (e < nrows * TPR) xv[i] = ld2(a.x, row0 * K + 2 * (int64_t)e);
        }
    };
    // stage views
    auto stage_ptr = [&](int64_t it) { return smem + (size_t)(it % NS) * SM::stage_bytes; };
    // halo of a tile: registers -> shared memory behind the tile rows (p' = z + beta p for the CG passes)
    auto halo_to_smem = [&](unsigned char* st, int nh, const double2 (&h0)[HPT], const double2 (&h1)[HPT]) {
        double2* sa = reinterpret_cast<double2*>(st);
#pragma unroll
        for (int i = 0; i < HPT; ++i) {
            const int hh = rg + i * ROWS;
            if (hh < nh) {
                double2 g = h0[i];
                if (CG_A) { g.x = fma(beta.x, h1[i].x, g.x); g.y = fma(beta.y, h1[i].y, g.y); }
                if (MGR) {   // e = omega (r - alpha q) / d of the halo row
                    const double2 dd = hd[MGR ? i : 0];
                    if (MGQ) { g.x = fma(-alpha.x, h1[i].x, g.x); g.y = fma(-alpha.y, h1[i].y, g.y); }
                    g.x = a.omega * g.x * rcp_pos(fma(cc.x, dd.x, dd.y));
                    g.y = a.omega * g.y * rcp_pos(fma(cc.y, dd.x, dd.y));
                }
                sa[(T + hh) * TPR + l] = g;
            }
        }
    };
    // p' = z + beta p in place over the z tile ; x += alpha_prev p (x comes from and goes to global memory)
    auto elementwise = [&](unsigned char* st, int64_t tile, double2 (&xv)[XPT]) {
        double2* sa = reinterpret_cast<double2*>(st);
        const double2* sb = reinterpret_cast<const double2*>(st + SM::off_b);
        const int64_t row0 = tile * T;
        const int nrows = (int)min((int64_t)T, m.nv - row0);
#pragma unroll
        for (int i = 0; i < XPT; ++i) {
            const int e = tid + i * NT;
            if (e < nrows * TPR) {
                const double2 zv = sa[e], pv = sb[e];
                double2 own;
                own.x = fma(beta.x, pv.x, zv.x);
                own.y = fma(beta.y, pv.y, zv.y);
                xv[i].x = fma(alpha.x, pv.x, xv[i].x);
                xv[i].y = fma(alpha.y, pv.y, xv[i].y);
                sa[e] = own;
                st2(a.x, row0 * K + 2 * (int64_t)e, xv[i]);
            }
        }
    };
    // MGR: r' = r - alpha q over the q tile, e = omega r'/d over the r tile.  (REGB, i.e. MGR0: there is no q and no
    // second region; the epilogue reads its own rows of w = r' again from global memory, an L2 hit)
    auto elementwise_mgr = [&](unsigned char* st, int64_t tile) {
        double2* sa = reinterpret_cast<double2*>(st);
        double2* sb = reinterpret_cast<double2*>(st + SM::off_b);
        const double* sdg = reinterpret_cast<const double*>(st + SM::off_dg);
        const double* sar = reinterpret_cast<const double*>(st + SM::off_ar);
        const int64_t row0 = tile * T;
        const int nrows = (int)min((int64_t)T, m.nv - row0);
        double2 qg[XPT];
        if (MGQ && REGB) {      // q of the tile's own rows straight from global memory (L2: prefetched with the tile)
#pragma unroll
            for (int i = 0; i < XPT; ++i) {
                const int e = tid + i * NT;
                if (e < nrows * TPR) qg[i] = ld2(a.in1, row0 * K + 2 * (int64_t)e);
            }
        }
#pragma unroll
        for (int i = 0; i < XPT; ++i) {
            const int e = tid + i * NT;
            if (e < nrows * TPR) {
                const int rr = e / TPR;
                const double2 rv = sa[e];
                const double sd = sdg[rr], av = sar[rr];
                double2 rn = rv;
                if (MGQ) {
                    const double2 qv = REGB ? qg[i] : sb[e];
                    rn.x = fma(-alpha.x, qv.x, rv.x);
                    rn.y = fma(-alpha.y, qv.y, rv.y);
                    // (REGB: r' goes out from registers; the same thread reads it back in the tile's epilogue)
                    if (REGB) st2(a.x, row0 * K + 2 * (int64_t)e, rn);
                }
                if (!REGB) sb[e] = rn;
                sa[e] = make_double2(a.omega * rn.x * rcp_pos(fma(cc.x, sd, av)), a.omega * rn.y * rcp_pos(fma(cc.y, sd, av)));
            }
        }
    };
    auto is_staged = [&](const int32_t* d) { return d[3] >= 0 && d[2] <= T * WCAP; };

    if (tid == 0) {
        for (int s = 0; s < NS; ++s) mbar_init(&bars[s], 1);
        fence_proxy_async();
    }
    // ---- prologue: descriptors of tiles 0..2, bulk copies of the first LA tiles, tile 0 made ready for its gather
    if (tid < 48) {
        const int64_t t = tile0 + (tid / 16) * G;
        sdesc[tid] = t < ntiles ? m.tile_desc[t * 16 + tid % 16] : 0;
    }
    __syncthreads();
    TileIssue tq{0, 0, -1};   // thread 0: what it needs to issue the tile two ahead
    if (tid == 0) {
        for (int k = 0; k < LA; ++k) {
            const int64_t t = tile0 + k * G;
            if (t < ntiles) issue(t, k, load_issue(m.tile_desc, t));
        }
        if (tile0 + LA * G < ntiles) tq = load_issue(m.tile_desc, tile0 + LA * G);
    }
    int hid_n[HPT];
    double2 h0[HPT], h1[HPT], xv[XPT];
    int dnext = 0;
    if (tile0 < ntiles) {
        load_hidx(tile0, hid_n);
        if (is_staged(sdesc)) load_halo(hid_n, sdesc[3], h0, h1);
        if (CG_A) load_x(tile0, xv);
        if (is_staged(sdesc)) halo_to_smem(smem, sdesc[3], h0, h1);
        load_hidx(tile0 + G, hid_n);
        if (tile0 + G < ntiles && is_staged(sdesc + 16)) load_halo(hid_n, sdesc[16 + 3], h0, h1);
        load_hidx(tile0 + 2 * G, hid_n);
        if (tid < 16) dnext = tile0 + 3 * G < ntiles ? m.tile_desc[(tile0 + 3 * G) * 16 + tid] : 0;
        mbar_wait(&bars[0], 0u);
        if (CG_A) {
            elementwise(smem, tile0, xv);
            load_x(tile0 + G, xv);
            fence_proxy_async();
        }
        if (MGR) {
            elementwise_mgr(smem, tile0);
            fence_proxy_async();
        }
    }
    double2 acc[MODE == MODE_AX ? 2 : 1] = {};
    int64_t tile = tile0;
    // ---- main loop.  Iteration `it` gathers tile it (made ready one iteration earlier) and then makes tile it+1
    // ready; one block barrier per tile.
    for (int64_t it = 0; tile < ntiles; ++it, tile += G) {
        unsigned char* st = stage_ptr(it);
        const double2* sa = reinterpret_cast<const double2*>(st);          // gathered vector: tile + halo
        const double2* sb = reinterpret_cast<const double2*>(st + SM::off_b);   // own p' (CG2B)
        const double* sval = reinterpret_cast<const double*>(st + SM::off_val);
        const double* stval = reinterpret_cast<const double*>(st + SM::off_tval);
        const int32_t* scol = reinterpret_cast<const int32_t*>(st + SM::off_col);
        const double* sdg = reinterpret_cast<const double*>(st + SM::off_dg);
        const double* sar = reinterpret_cast<const double*>(st + SM::off_ar);
        const int64_t row0 = tile * T;
        const int nrows = (int)min((int64_t)T, m.nv - row0);
        __syncthreads();   // tile it is ready in its stage; tile it-1 is fully consumed
        const int32_t* d = sdesc + (it & 3) * 16;
        const int64_t cp_first = (int64_t)(uint32_t)d[0] | ((int64_t)d[1] << 32);
        const int32_t* scp = d + 4;
        const bool staged = is_staged(d);
        if (tid == 0) {
            const int64_t t2 = tile + LA * G;
            bulk_wait_read0();   // the stage of tile it-1 is free once its bulk store has been read
            if (t2 < ntiles) issue(t2, (int)((it + LA) % NS), tq);
            if (CG_A || MGR) {
                // (MGR with out1 == nullptr: e is not stored, the prolongation kernel forms it again from r')
                if (!MGR || a.out1) bulk_store(a.out1 + row0 * K, sa, (uint32_t)nrows * K * sizeof(double));
                if (MGQ && !REGB) bulk_store(a.x + row0 * K, sb, (uint32_t)nrows * K * sizeof(double));
                bulk_commit();
            }
            if (t2 + G < ntiles) tq = load_issue(m.tile_desc, t2 + G);
        }
        if (tid < 16) {   // descriptor ring: tile it+3 in, tile it+4 on its way
            sdesc[((it + 3) & 3) * 16 + tid] = dnext;
            dnext = tile + 4 * G < ntiles ? m.tile_desc[(tile + 4 * G) * 16 + tid] : 0;
        }

        for (int r = rg; r < nrows; r += ROWS) {
            const int64_t row = row0 + r;
            // REGB: the row's own entry of the second vector straight from global memory, asked for before the gather
            // (thread 0 prefetched the tile into L2 when it issued the tile's bulk copies)
            double2 rv_g = {0.0, 0.0};
            if (REGB) {
                if (MODE == MODE_MGR) {     // r', written by this very thread when it prepared the tile: a coherent (L2) load
                    rv_g = __ldcg(reinterpret_cast<const double2*>(a.x + row * K + 2 * l));
                } else {
                    const double* __restrict__ src = (MODE == MODE_MGR0) ? a.in0 : a.in1;
                    if (src) rv_g = ld2(src, row * K + 2 * l);
                }
            }
            const int chl = r >> m.log2c;
            const int cpr = scp[chl];
            const int w = (scp[chl + 1] - cpr) >> m.log2c;
            const int o = cpr + (r & (C - 1)) * w;
            const double2 own = sa[r * TPR + l];
            double2 s = {0.0, 0.0};
            if (staged) {
                // every neighbour (tile or halo) is in shared memory under its tile-local index
                // the width is the same for all rows of a SELL slice, hence warp-uniform: fully unrolled rows
                switch (w) {
                    case 2: s = gather_row<2, TPR, VEC>(scol + o, sval + o, stval + o, sa, l); break;
                    case 4: s = gather_row<4, TPR, VEC>(scol + o, sval + o, stval + o, sa, l); break;
                    case 6: s = gather_row<6, TPR, VEC>(scol + o, sval + o, stval + o, sa, l); break;
                    case 8: s = gather_row<8, TPR, VEC>(scol + o, sval + o, stval + o, sa, l); break;
                    default:
                        // a slice wider than 8 (a vertex of valence 9 or more in its 32 rows): the tile's slots still
                        // fit the shared slice (is_staged checks the total), so the same gather as a plain loop
                        for (int k = 0; k < w; k += 2) {
                            const int2 cj = *reinterpret_cast<const int2*>(scol + o + k);
                            const double2 vj = *reinterpret_cast<const double2*>(sval + o + k);
                            const double2 g0 = sa[cj.x * TPR + l], g1 = sa[cj.y * TPR + l];
                            s.x = fma(vj.x, g0.x, s.x); s.y = fma(vj.x, g0.y, s.y);
                            s.x = fma(vj.y, g1.x, s.x); s.y = fma(vj.y, g1.y, s.y);
                            if (VEC) {
                                const double2 tj = *reinterpret_cast<const double2*>(stval + o + k);
                                s.x = fma(tj.x, g0.y, s.x); s.y = fma(-tj.x, g0.x, s.y);
                                s.x = fma(tj.y, g1.y, s.x); s.y = fma(-tj.y, g1.x, s.y);
                            }
                        }
                        break;
                }
            } else {
                // fallback (wide rows or a halo beyond HALO_CAP): global column ids, out-of-tile rows from L2
                for (int k = 0; k < w; k += 2) {
                    const int2 cj = *reinterpret_cast<const int2*>(m.col + cp_first + o + k);
                    const double2 vj = ld2(m.val, cp_first + o + k);
                    double2 g0, g1;
                    const unsigned j0 = (unsigned)(cj.x - (int)row0), j1 = (unsigned)(cj.y - (int)row0);
                    if (j0 < (unsigned)nrows) {
                        g0 = sa[j0 * TPR + l];
                    } else {
                        g0 = ld2(a.in0, (int64_t)cj.x * K + 2 * l);
                        if (CG_A) {
                            const double2 p0 = ld2(a.in1, (int64_t)cj.x * K + 2 * l);
                            g0.x = fma(beta.x, p0.x, g0.x); g0.y = fma(beta.y, p0.y, g0.y);
                        }
                        if (MGR) {
                            if (MGQ) {
                                const double2 p0 = ld2(a.in1, (int64_t)cj.x * K + 2 * l);
                                g0.x = fma(-alpha.x, p0.x, g0.x); g0.y = fma(-alpha.y, p0.y, g0.y);
                            }
                            const double sj = m.sdiag[cj.x], aj = m.area[cj.x];
                            g0.x = a.omega * g0.x * rcp_pos(fma(cc.x, sj, aj));
                            g0.y = a.omega * g0.y * rcp_pos(fma(cc.y, sj, aj));
                        }
                    }
                    if (j1 < (unsigned)nrows) {
                        g1 = sa[j1 * TPR + l];
                    } else {
                        g1 = ld2(a.in0, (int64_t)cj.y * K + 2 * l);
                        if (CG_A) {
                            const double2 p1 = ld2(a.in1, (int64_t)cj.y * K + 2 * l);
                            g1.x = fma(beta.x, p1.x, g1.x); g1.y = fma(beta.y, p1.y, g1.y);
                        }
                        if (MGR) {
                            if (MGQ) {
                                const double2 p1 = ld2(a.in1, (int64_t)cj.y * K + 2 * l);
                                g1.x = fma(-alpha.x, p1.x, g1.x); g1.y = fma(-alpha.y, p1.y, g1.y);
                            }
                            const double sj = m.sdiag[cj.y], aj = m.area[cj.y];
                            g1.x = a.omega * g1.x * rcp_pos(fma(cc.x, sj, aj));
                            g1.y = a.omega * g1.y * rcp_pos(fma(cc.y, sj, aj));
                        }
                    }
                    s.x = fma(vj.x, g0.x, s.x); s.y = fma(vj.x, g0.y, s.y);
                    s.x = fma(vj.y, g1.x, s.x); s.y = fma(vj.y, g1.y, s.y);
                    if (VEC) {
                        const double2 tj = ld2(m.tval, cp_first + o + k);
                        s.x = fma(tj.x, g0.y, s.x); s.y = fma(-tj.x, g0.x, s.y);
                        s.x = fma(tj.y, g1.y, s.x); s.y = fma(-tj.y, g1.x, s.y);
                    }
                }
            }
            const double sd = sdg[r];
            s.x = fma(sd, own.x, s.x);
            s.y = fma(sd, own.y, s.y);          // s = (S v)_row
            const int64_t ri = row * K + 2 * l;
            if (MODE == MODE_PLAIN) {
                if (a.scale_inv_area) { const double ia = sar[r]; s.x *= ia; s.y *= ia; }
                st2(a.out0, ri, s);
            } else if (MODE == MODE_CG2A) {
                const double ia = sar[r];
                s.x *= ia; s.y *= ia;            // t = M^-1 S p'
                st2(a.out0, ri, s);
            } else if (AXE) {
                const int sub = MGR ? 1 : a.scale_inv_area;
                const double av = sar[r];
                double2 o = {fma(cc.x, s.x, av * own.x), fma(cc.y, s.y, av * own.y)};   // A v
                if (sub >= 1) {
                    const double2 rv = REGB ? rv_g : sb[r * TPR + l];
                    o.x = rv.x - o.x; o.y = rv.y - o.y;                                  // r - A v
                    if (MGR && a.omega2 != 0.0) {      // second sweep: e2 = e1 + omega2 (r' - K e1)/d
                        o.x = fma(a.omega2 * o.x, rcp_pos(fma(cc.x, sd, av)), own.x);
                        o.y = fma(a.omega2 * o.y, rcp_pos(fma(cc.y, sd, av)), own.y);
                    }
                    if (sub >= 2) {
                        // (rcp_pos as in the first sweep: the same D^-1 on both sides of the cycle, and a fifth of
                        // this kernel's instructions less than two fp64 divisions)
                        o.x = fma(a.omega * o.x, rcp_pos(fma(cc.x, sd, av)), own.x);
                        o.y = fma(a.omega * o.y, rcp_pos(fma(cc.y, sd, av)), own.y);
                        if (sub == 5) {     // y = V r ends the first cycle of B = V M V: rho' = y.M y, w = M y goes on
                            const double2 wv = {av * o.x, av * o.y};
                            acc[0].x = fma(wv.x, o.x, acc[0].x);  acc[0].y = fma(wv.y, o.y, acc[0].y);
                            o = wv;
                        } else {
                            acc[0].x = fma(rv.x, o.x, acc[0].x);  acc[0].y = fma(rv.y, o.y, acc[0].y);     // r.z
                        }
                        acc[MODE == MODE_AX ? 1 : 0].x = fma(rv.x, rv.x, acc[MODE == MODE_AX ? 1 : 0].x);
                        acc[MODE == MODE_AX ? 1 : 0].y = fma(rv.y, rv.y, acc[MODE == MODE_AX ? 1 : 0].y);
                    }
                }
                st2(a.out0, ri, o);
            } else {
                // q = A_v p + c (S v)_row ; v = p (n = 1) or t (n = 2)
                const double av = sar[r];
                const double2 pv = (MODE == MODE_CG1) ? own : sb[r * TPR + l];
                double2 q;
                q.x = fma(cc.x, s.x, av * pv.x);
                q.y = fma(cc.y, s.y, av * pv.y);
                st2(a.out0, ri, q);
                acc[0].x = fma(pv.x, q.x, acc[0].x);
                acc[0].y = fma(pv.y, q.y, acc[0].y);
            }
        }
        // ---- make tile it+1 ready: halo into its stage, wait for its bulk copies, form p', update x
        if (tile + G < ntiles) {
            unsigned char* st1 = stage_ptr(it + 1);
            const int32_t* d1 = sdesc + ((it + 1) & 3) * 16;
            const int32_t* d2 = sdesc + ((it + 2) & 3) * 16;
            if (is_staged(d1)) halo_to_smem(st1, d1[3], h0, h1);
            if (tile + 2 * G < ntiles && is_staged(d2)) load_halo(hid_n, d2[3], h0, h1);
            load_hidx(tile + 3 * G, hid_n);
            mbar_wait(&bars[(it + 1) % NS], (uint32_t)((it + 1) / NS) & 1u);
            if (CG_A) {
                elementwise(st1, tile + G, xv);
                load_x(tile + 2 * G, xv);
                fence_proxy_async();
            }
            if (MGR) {
                elementwise_mgr(st1, tile + G);
                fence_proxy_async();
            }
        }
    }
    if ((CG_A || MGR) && tid == 0) bulk_wait0();
    if (MODE == MODE_CG1 || MODE == MODE_CG2B) {
        __shared__ double tot[KMAX];
        const double2 acc1[1] = {acc[0]};
        if (grid_reduce<K, 1, NT>(acc1, partials, &ctrl->ticket[0], tot)) {
            if (tid < K) {
                const double pq = ctrl->pair_mode ? tot[tid & ~1] + tot[tid | 1] : tot[tid];
                double al = 0.0;
                if (!ctrl->done[tid]) {
                    if (ctrl->starting[tid]) al = 1.0;     // p' = phi, q = A phi: the next kernel forms r0 = M phi - A phi
                    else if (pq > 0.0 && isfinite(pq)) al = ctrl->rho[tid] / pq;
                    else { ctrl->done[tid] = 1; ctrl->status[tid] = 2; }
                }
                ctrl->alpha[tid] = al;
            }
        }
    }
    if (MODE == MODE_AX && a.scale_inv_area >= 3) {
        __shared__ double tot2[2 * KMAX];
        const double2 acc2[2] = {acc[0], acc[MODE == MODE_AX ? 1 : 0]};
        if (grid_reduce<K, 2, NT>(acc2, partials, &ctrl->ticket[2], tot2))
            cg_bookkeeping<K>(ctrl, tot2);
    }
}

// ------------------------------------------------------------------------------------------- start of a column
// x[row][c] = field_c[perm[row]] for the columns in `mask`  (H0 ingest: gather through the permutation, transpose)
template <int K>
__global__ void __launch_bounds__(BLOCK) k_ingest(MeshView m, StartParams sp, unsigned mask,
                                                  const double* __restrict__ fields, double* __restrict__ x) {
    const int64_t i = (int64_t)blockIdx.x * BLOCK + threadIdx.x;
    if (i >= m.nv * K) return;
    const int64_t row = i / K;
    const int c = (int)(i % K);
    if (!((mask >> c) & 1u)) return;
    const int f = sp.field[c];
    x[i] = f >= 0 ? fields[(int64_t)f * m.nv + m.perm[row]] : 0.0;
}

// Start of CG from x0 = phi for the columns in `mask`: y = S (M^-1 S)^(n-1) phi is given;
// r0 = M phi - A_c phi = -c y ;  z0 = r0/d ;  p = 0 ;  rho0 = r0.z0 ;  ||r0||^2 ;  ||M phi||^2.
template <int K>
__global__ void __launch_bounds__(BLOCK) k_init(MeshView m, Ctrl* __restrict__ ctrl, double* __restrict__ partials,
                                                StartParams sp, unsigned mask, const double* __restrict__ x,
                                                const double* __restrict__ y, double* __restrict__ z_,
                                                double* __restrict__ p0, double* __restrict__ p1, int order_n) {
    double* __restrict__ z = z_;
    constexpr int TPR = K / 2;
    constexpr int ROWS = BLOCK / TPR;
    const int tid = threadIdx.x, l = tid % TPR;
    const bool on0 = (mask >> (2 * l)) & 1u, on1 = (mask >> (2 * l + 1)) & 1u;
    const double2 cc = {sp.c[2 * l], sp.c[2 * l + 1]};
    const double* __restrict__ dg = jacobi_diag(m, order_n);
    double2 acc[3] = {{0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}};
    if (on0 || on1) {
        for (int64_t row = (int64_t)blockIdx.x * ROWS + tid / TPR; row < m.nv; row += (int64_t)gridDim.x * ROWS) {
            const int64_t ri = row * K + 2 * l;
            const double av = m.area[row], dv = dg[row];
            const double2 d = {fma(cc.x, dv, av), fma(cc.y, dv, av)};
            const double2 xv = ld2(x, ri), yv = ld2(y, ri);
            double2 zv = ld2(z, ri), pa = ld2(p0, ri), pb = ld2(p1, ri);
            const double2 r = {-cc.x * yv.x, -cc.y * yv.y};
            const double2 b = {av * xv.x, av * xv.y};
            if (on0) {
                zv.x = r.x / d.x; pa.x = 0.0; pb.x = 0.0;
                acc[0].x = fma(r.x, zv.x, acc[0].x); acc[1].x = fma(r.x, r.x, acc[1].x); acc[2].x = fma(b.x, b.x, acc[2].x);
            }
            if (on1) {
                zv.y = r.y / d.y; pa.y = 0.0; pb.y = 0.0;
                acc[0].y = fma(r.y, zv.y, acc[0].y); acc[1].y = fma(r.y, r.y, acc[1].y); acc[2].y = fma(b.y, b.y, acc[2].y);
            }
            st2(z, ri, zv);
            st2(p0, ri, pa);
            st2(p1, ri, pb);
        }
    }
    __shared__ double tot[3 * KMAX];
    if (grid_reduce<K, 3>(acc, partials, &ctrl->ticket[1], tot)) {
        if (tid < K && ((mask >> tid) & 1u)) {
            const int ta = ctrl->pair_mode ? (tid & ~1) : tid, tb = ctrl->pair_mode ? (tid | 1) : tid;
            const double w2 = ctrl->pair_mode ? 1.0 : 0.5;      // (ta == tb without pairs: the value itself)
            const double rho = w2 * (tot[ta] + tot[tb]), rr = w2 * (tot[KMAX + ta] + tot[KMAX + tb]),
                         bb = w2 * (tot[2 * KMAX + ta] + tot[2 * KMAX + tb]);
            ctrl->c[tid] = sp.c[tid]; ctrl->c1[tid] = sp.c1[tid]; ctrl->field[tid] = sp.field[tid]; ctrl->rhs[tid] = sp.rhs[tid];
            ctrl->starting[tid] = 0;
            ctrl->rho[tid] = rho; ctrl->rr[tid] = rr; ctrl->bb[tid] = bb;
            ctrl->alpha[tid] = 0.0; ctrl->beta[tid] = 0.0; ctrl->iters[tid] = 0;
            int st = 0;
            int dn = (sp.field[tid] < 0) || (rr <= ctrl->tol2 * bb);
            if (!isfinite(rr) || !isfinite(bb)) { dn = 1; st = 2; }
            ctrl->status[tid] = st;
            ctrl->epoch[tid] = ctrl->epoch[tid] + 1;
            ctrl->done[tid] = dn;
        }
        __syncthreads();
        if (tid == 0) {
            int any = 0;
            for (int c = 0; c < K; ++c) any |= !ctrl->done[c];
            ctrl->all_done = !any;
        }
    }
}

// Start of multigrid-preconditioned CG for the columns in `mask` (mg_solve.cuh), from x0 = phi without a
// pass of its own over the matrix: the column joins the stream with
//     x = 0 ,  z = phi ,  p = 0 ,  r = M phi ,  beta = 0 ,  starting = 1,
// and its first iteration -- the same launch sequence as every other -- does the rest: kernel A forms p' = z = phi and
// q = A phi and sets alpha = 1 for a starting column, the fused residual kernel forms r0 = r - alpha q = M phi - A phi,
// the cycle gives z0 = B r0, the bookkeeping sets rho = r0.z0, beta = 0 and counts nothing; the next kernel A applies
// the pending x += alpha p' = phi.  (Jacobi path: k_init, with r0 = -c S (M^-1 S)^(n-1) phi from a plain SpMM.)
// fields are gathered through the permutation; r goes to the residual buffer in use (Ctrl::cur_r).
template <int K>
__global__ void __launch_bounds__(BLOCK) k_mg_start(MeshView m, Ctrl* __restrict__ ctrl, double* __restrict__ partials,
                                                    StartParams sp, unsigned mask, const double* __restrict__ fields,
                                                    double* __restrict__ x, double* __restrict__ z,
                                                    double* __restrict__ r0, double* __restrict__ r1,
                                                    double* __restrict__ p0, double* __restrict__ p1) {
    // Mostly one to four of the K columns start at a time.  Measured on B200 (7.3 M rows, four vectors): 8-byte stores
    // that miss in L2 are not merged -- each becomes its own 32-byte read-modify-write in DRAM (0.72 ms for one
    // column, 4.7 ms for sixteen) -- while 16-byte updates of lines loaded first cost about 1.1 ms for any mask when only
    // the lanes of the masked pairs work.  So: 16-byte read-modify-write with the masked column PAIRS compacted, P of
    // them padded to a power of two PP: a thread keeps one pair and walks rows, every thread works; pairs with both
    // columns starting are stored without a load; of the two direction buffers only p[cur_p] -- the one kernel A reads
    // as the old direction -- is cleared (kernel A writes the other one in full).
    constexpr int TPR = K / 2;
    constexpr int U = 2;
    __shared__ int s_pair[TPR];
    __shared__ int s_np;
    const int tid = threadIdx.x;
    const bool dev = mask == MASK_TURN_START;      // turnover on the device: mask and parameters from k_turn_plan
    if (dev) mask = ctrl->turn_start;
    if (mask == 0u) return;
    if (tid == 0) {
        int n = 0;
        for (int l = 0; l < TPR; ++l)
            if ((mask >> (2 * l)) & 3u) s_pair[n++] = l;
        s_np = n;
    }
    __syncthreads();
    const int P = s_np;
    const int PP = P <= 1 ? 1 : P <= 2 ? 2 : P <= 4 ? 4 : P <= 8 ? 8 : TPR;
    const int j = tid & (PP - 1);
    const bool active = j < P;
    const int l = active ? s_pair[j] : 0;
    const bool on0 = active && ((mask >> (2 * l)) & 1u), on1 = active && ((mask >> (2 * l + 1)) & 1u);
    const int f0 = dev ? ctrl->turn_sp.field[2 * l] : sp.field[2 * l];
    const int f1 = dev ? ctrl->turn_sp.field[2 * l + 1] : sp.field[2 * l + 1];
    double* __restrict__ r = ctrl->cur_r ? r1 : r0;
    double* __restrict__ p = ctrl->cur_p ? p1 : p0;
    double2 acc = {0.0, 0.0};
    if (active) {
        const int rows_blk = BLOCK / PP;
        const int64_t stride = (int64_t)gridDim.x * rows_blk;
        const bool both = on0 && on1;
        for (int64_t base = (int64_t)blockIdx.x * rows_blk + tid / PP; base < m.nv; base += U * stride) {
            double2 xv[U], zv[U], rv[U], pv[U];
            double av[U], ph0[U], ph1[U];
#pragma unroll
            for (int i = 0; i < U; ++i) {
                const int64_t row = base + i * stride;
                if (row >= m.nv) continue;
                const int64_t ri = row * K + 2 * l;
                if (!both) { xv[i] = ld2(x, ri); zv[i] = ld2(z, ri); rv[i] = ld2(r, ri); pv[i] = ld2(p, ri); }
                av[i] = m.area[row];
                const int64_t u = m.perm[row];
                ph0[i] = (on0 && f0 >= 0) ? fields[(int64_t)f0 * m.nv + u] : 0.0;
                ph1[i] = (on1 && f1 >= 0) ? fields[(int64_t)f1 * m.nv + u] : 0.0;
            }
#pragma unroll
            for (int i = 0; i < U; ++i) {
                const int64_t row = base + i * stride;
                if (row >= m.nv) continue;
                const int64_t ri = row * K + 2 * l;
                if (on0) {
                    xv[i].x = 0.0; zv[i].x = ph0[i]; rv[i].x = av[i] * ph0[i]; pv[i].x = 0.0;
                    acc.x = fma(rv[i].x, rv[i].x, acc.x);
                }
                if (on1) {
                    xv[i].y = 0.0; zv[i].y = ph1[i]; rv[i].y = av[i] * ph1[i]; pv[i].y = 0.0;
                    acc.y = fma(rv[i].y, rv[i].y, acc.y);
                }
                st2(x, ri, xv[i]); st2(z, ri, zv[i]); st2(r, ri, rv[i]); st2(p, ri, pv[i]);
            }
        }
    }
    __shared__ double tot[KMAX];
    if (grid_reduce_pairs<K>(acc, PP, P, l, partials, &ctrl->ticket[1], tot)) {
        if (tid < K && ((mask >> tid) & 1u)) {
            const int ta = ctrl->pair_mode ? (tid & ~1) : tid, tb = ctrl->pair_mode ? (tid | 1) : tid;
            const double bb = (ctrl->pair_mode ? 1.0 : 0.5) * (tot[ta] + tot[tb]);
            const int fld = dev ? ctrl->turn_sp.field[tid] : sp.field[tid];
            ctrl->c[tid] = dev ? ctrl->turn_sp.c[tid] : sp.c[tid];
            ctrl->c1[tid] = dev ? ctrl->turn_sp.c1[tid] : sp.c1[tid];
            ctrl->field[tid] = fld;
            ctrl->rhs[tid] = dev ? ctrl->turn_sp.rhs[tid] : sp.rhs[tid];
            ctrl->rho[tid] = 0.0; ctrl->rr[tid] = bb; ctrl->bb[tid] = bb;
            ctrl->alpha[tid] = 0.0; ctrl->beta[tid] = 0.0; ctrl->iters[tid] = 0;
            ctrl->status[tid] = isfinite(bb) ? 0 : 2;
            ctrl->epoch[tid] = ctrl->epoch[tid] + 1;
            ctrl->done[tid] = (fld < 0 || !isfinite(bb)) ? 1 : 0;
            ctrl->starting[tid] = ctrl->done[tid] ? 0 : 1;
        }
        __syncthreads();
        if (tid == 0) {
            int any = 0;
            for (int c = 0; c < K; ++c) any |= !ctrl->done[c];
            ctrl->all_done = !any;
        }
    }
}

// ------------------------------------------------------------------------------------------- kernel B
// z -= alpha q/d ; rho' = sum d z^2 ; ||r||^2 = sum (d z)^2 ; then (last block) beta, stop tests.
// Pure streaming: every thread keeps U = 8 rows (16 independent 16-byte loads) in flight, two blocks per SM --
// measured on B200 this reaches the copy bandwidth, while more resident warps with fewer loads each do not.
template <int K>
__global__ void __launch_bounds__(BLOCK, 2) k_update(MeshView m, Ctrl* __restrict__ ctrl, double* __restrict__ partials,
                                                     double* __restrict__ z, const double* __restrict__ q, int order_n) {
    constexpr int TPR = K / 2;
    constexpr int ROWS = BLOCK / TPR;
    constexpr int U = 8;
    if (ctrl->all_done) return;
    const int tid = threadIdx.x, l = tid % TPR;
    const double2 cc = ld2(ctrl->c, 2 * l);
    const double2 alpha = ld2(ctrl->alpha, 2 * l);
    const double* __restrict__ dg = jacobi_diag(m, order_n);
    double2 acc[2] = {{0.0, 0.0}, {0.0, 0.0}};
    const int64_t stride = (int64_t)gridDim.x * ROWS;
    for (int64_t base = (int64_t)blockIdx.x * ROWS + tid / TPR; base < m.nv; base += U * stride) {
        double2 zv[U], qv[U];
        double av[U], dv[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int64_t row = base + u * stride;
            if (row < m.nv) {
                zv[u] = ld2(z, row * K + 2 * l);
                qv[u] = ld2(q, row * K + 2 * l);
                av[u] = m.area[row];
                dv[u] = dg[row];
            }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int64_t row = base + u * stride;
            if (row < m.nv) {
                const double2 d = {fma(cc.x, dv[u], av[u]), fma(cc.y, dv[u], av[u])};
                zv[u].x = fma(-alpha.x * qv[u].x, rcp_pos(d.x), zv[u].x);
                zv[u].y = fma(-alpha.y * qv[u].y, rcp_pos(d.y), zv[u].y);
                st2(z, row * K + 2 * l, zv[u]);
                const double2 r = {d.x * zv[u].x, d.y * zv[u].y};
                acc[0].x = fma(r.x, zv[u].x, acc[0].x); acc[0].y = fma(r.y, zv[u].y, acc[0].y);
                acc[1].x = fma(r.x, r.x, acc[1].x);     acc[1].y = fma(r.y, r.y, acc[1].y);
            }
        }
    }
    __shared__ double tot[2 * KMAX];
    if (grid_reduce<K, 2>(acc, partials, &ctrl->ticket[2], tot)) {
        __shared__ int any_active;
        if (tid == 0) any_active = 0;
        __syncthreads();
        if (tid < K) {
            if (!ctrl->done[tid]) {
                const bool pr = ctrl->pair_mode != 0;
                const double rho_new = pr ? tot[tid & ~1] + tot[tid | 1] : tot[tid];
                const double rr = pr ? tot[KMAX + (tid & ~1)] + tot[KMAX + (tid | 1)] : tot[KMAX + tid];
                const int it = ctrl->iters[tid] + 1;
                ctrl->iters[tid] = it;
                ctrl->rr[tid] = rr;
                double be = rho_new / ctrl->rho[tid];
                ctrl->rho[tid] = rho_new;
                int dn = 0;
                if (!isfinite(rr)) { dn = 1; ctrl->status[tid] = 2; }
                else if (rr <= ctrl->tol2 * ctrl->bb[tid]) { dn = 1; ctrl->status[tid] = 0; }
                else if (!isfinite(be)) { dn = 1; ctrl->status[tid] = 2; }
                else if (it >= ctrl->max_iter) { dn = 1; ctrl->status[tid] = 1; }
                if (dn) { be = 0.0; ctrl->done[tid] = 1; }
                ctrl->beta[tid] = be;
                if (!dn) atomicOr(&any_active, 1);
            } else {
                ctrl->beta[tid] = 0.0;
            }
        }
        __syncthreads();
        if (tid == 0) { ctrl->all_done = !any_active; ctrl->total_iters += 1; ctrl->cur_p ^= 1; }
    }
}

// ------------------------------------------------------------------------------------------- end of a column
// H6b for the columns in `mask`: x_final = x + alpha p (the update still pending, alpha = 0 once applied),
// e_c = 1/2 sum_v A_v x_v^2 / sum_v A_v
template <int K>
__global__ void __launch_bounds__(BLOCK) k_energy(MeshView m, Ctrl* __restrict__ ctrl, double* __restrict__ partials,
                                                  unsigned mask, const double* __restrict__ x,
                                                  const double* __restrict__ pa, const double* __restrict__ pb,
                                                  double total_area, double* __restrict__ energy) {
    // as k_mg_start: a thread owns rows and loops over the columns in `mask`
    constexpr int U = 2;
    const int tid = threadIdx.x;
    if (mask == MASK_TURN_FIN) mask = ctrl->turn_fin;
    if (mask == 0u) return;
    const double* __restrict__ p = ctrl->cur_p ? pb : pa;
    __shared__ double s_alpha[KMAX];
    if (tid < KMAX) s_alpha[tid] = ctrl->alpha[tid];
    __syncthreads();
    double acc[K];
#pragma unroll
    for (int c = 0; c < K; ++c) acc[c] = 0.0;
    const int64_t stride = (int64_t)gridDim.x * BLOCK;
    for (int64_t base = (int64_t)blockIdx.x * BLOCK + tid; base < m.nv; base += U * stride) {
        double av[U];
#pragma unroll
        for (int i = 0; i < U; ++i) av[i] = base + i * stride < m.nv ? m.area[base + i * stride] : 0.0;
#pragma unroll
        for (int c = 0; c < K; ++c) {
            if (!((mask >> c) & 1u)) continue;
            double xv[U], pv[U];
#pragma unroll
            for (int i = 0; i < U; ++i) {
                const int64_t row = base + i * stride;
                const bool ok = row < m.nv;
                xv[i] = ok ? x[row * K + c] : 0.0;
                pv[i] = ok ? p[row * K + c] : 0.0;
            }
#pragma unroll
            for (int i = 0; i < U; ++i) {
                const double xf = fma(s_alpha[c], pv[i], xv[i]);
                acc[c] = fma(av[i] * xf, xf, acc[c]);
            }
        }
    }
    __shared__ double tot[KMAX];
    if (grid_reduce_cols<K>(acc, mask, partials, &ctrl->ticket[3], tot)) {
        if (tid < K && ((mask >> tid) & 1u) && ctrl->field[tid] >= 0)
            energy[ctrl->rhs[tid]] = 0.5 * tot[tid] / total_area;
    }
}

// H6a for the columns in `mask`: x_final scattered back to the caller's numbering: out[rhs][perm[row]]
// (or the high-pass field phi - x_final)
template <int K>
__global__ void __launch_bounds__(BLOCK) k_scatter(MeshView m, const Ctrl* __restrict__ ctrl, unsigned mask,
                                                   const double* __restrict__ x, const double* __restrict__ pa,
                                                   const double* __restrict__ pb, int use_p, double* __restrict__ out,
                                                   const double* __restrict__ fields, int highpass) {
    __shared__ double tile[K][33];
    __shared__ int32_t dst[32];
    const int tid = threadIdx.x;
    if (mask == MASK_TURN_FIN) mask = ctrl->turn_fin;
    if (mask == 0u) return;
    const double* __restrict__ p = ctrl->cur_p ? pb : pa;
    // BLOCK threads move 32 rows x K columns per step
    for (int64_t base = (int64_t)blockIdx.x * 32; base < m.nv; base += (int64_t)gridDim.x * 32) {
        for (int e = tid; e < 32 * K; e += BLOCK) {
            const int r = e / K, c = e % K;
            const int64_t row = base + r;
            double v = 0.0;
            if (row < m.nv && ((mask >> c) & 1u)) {
                v = x[row * K + c];
                if (use_p) v = fma(ctrl->alpha[c], p[row * K + c], v);
            }
            tile[c][r] = v;
        }
        if (tid < 32) dst[tid] = base + tid < m.nv ? m.perm[base + tid] : -1;
        __syncthreads();
        for (int e = tid; e < 32 * K; e += BLOCK) {
            const int c = e / 32, r = e % 32;
            if (((mask >> c) & 1u) && ctrl->field[c] >= 0 && dst[r] >= 0) {
                double v = tile[c][r];
                if (highpass) v = fields[(int64_t)ctrl->field[c] * m.nv + dst[r]] - v;   // phi - phibar
                out[(int64_t)ctrl->rhs[c] * m.nv + dst[r]] = v;
            }
        }
        __syncthreads();
    }
}

// True residual of returned solutions (IF_FLAG_TRUE_RESIDUAL): q = A_c x_c is given for the K columns (x = the filtered
// fields as the caller received them); per column ||M phi - q||_2 / ||M phi||_2 with phi gathered from the caller's
// fields through the permutation (sp.field = field of the column, sp.rhs = where the result goes; pairs of the vector
// filter share one norm over both components).
template <int K>
__global__ void __launch_bounds__(BLOCK) k_true_res(MeshView m, Ctrl* __restrict__ ctrl, double* __restrict__ partials,
                                                    StartParams sp, const double* __restrict__ fields,
                                                    const double* __restrict__ q, double* __restrict__ out) {
    constexpr int TPR = K / 2;
    constexpr int ROWS = BLOCK / TPR;
    const int tid = threadIdx.x, l = tid % TPR;
    const int f0 = sp.field[2 * l], f1 = sp.field[2 * l + 1];
    double2 acc[2] = {{0.0, 0.0}, {0.0, 0.0}};
    for (int64_t row = (int64_t)blockIdx.x * ROWS + tid / TPR; row < m.nv; row += (int64_t)gridDim.x * ROWS) {
        const double av = m.area[row];
        const int64_t u = m.perm[row];
        const double2 qv = ld2(q, row * K + 2 * l);
        const double b0 = f0 >= 0 ? av * fields[(int64_t)f0 * m.nv + u] : 0.0;
        const double b1 = f1 >= 0 ? av * fields[(int64_t)f1 * m.nv + u] : 0.0;
        const double d0 = f0 >= 0 ? b0 - qv.x : 0.0, d1 = f1 >= 0 ? b1 - qv.y : 0.0;
        acc[0].x = fma(d0, d0, acc[0].x); acc[0].y = fma(d1, d1, acc[0].y);
        acc[1].x = fma(b0, b0, acc[1].x); acc[1].y = fma(b1, b1, acc[1].y);
    }
    __shared__ double tot[2 * KMAX];
    if (grid_reduce<K, 2>(acc, partials, &ctrl->ticket[1], tot)) {
        if (tid < K && sp.field[tid] >= 0) {
            const int ta = ctrl->pair_mode ? (tid & ~1) : tid, tb = ctrl->pair_mode ? (tid | 1) : tid;
            const double w2 = ctrl->pair_mode ? 1.0 : 0.5;
            const double rr = w2 * (tot[ta] + tot[tb]), bb = w2 * (tot[KMAX + ta] + tot[KMAX + tb]);
            out[sp.rhs[tid]] = bb > 0.0 ? sqrt(rr / bb) : 0.0;
        }
    }
}

// per-right-hand-side results of the columns in `mask`
__global__ void k_stats(const Ctrl* __restrict__ ctrl, int K, unsigned mask, int32_t* __restrict__ iters,
                        int32_t* __restrict__ status, double* __restrict__ relres) {
    const int c = threadIdx.x;
    if (c < K && ((mask >> c) & 1u) && ctrl->field[c] >= 0) {
        const int r = ctrl->rhs[c];
        iters[r] = ctrl->iters[c];
        status[r] = ctrl->status[c];
        relres[r] = ctrl->bb[c] > 0.0 ? sqrt(ctrl->rr[c] / ctrl->bb[c]) : 0.0;
    }
}

// Column turnover on the device (multigrid stream; one thread, at the end of every iteration's graph): the columns that
// hold a right-hand side and have stopped are to be finalised (turn_fin); every free column takes the next entry of
// the queue (turn_start, turn_sp).  The kernels that follow in the same graph -- k_energy or k_scatter,
// k_mg_start, k_mg_coarse_factor -- read these masks and return at once when they are empty, so a stopped column is
// running its next right-hand side in the very next iteration and the host only watches `snap`.
// `first` (before the first iteration): every column is started -- those the queue has nothing for as empty columns
// (zeroed, stopped at once), so that no kernel ever reads what the workspace held before.
__global__ void k_turn_plan(Ctrl* __restrict__ ctrl, const QEntry* __restrict__ queue, int K, int first,
                            int32_t* __restrict__ iters, int32_t* __restrict__ status, double* __restrict__ relres) {
    // one warp, lane s = slot s: a column, or with the vector filter (pair_mode) the column pair (2s, 2s+1) of one
    // coupled system, whose queue entry names the u field and output slot; v follows at field + 1, slot + rhs_stride.
    // Masks by ballot, the queue position of a free slot = its rank among the free ones.
    const unsigned full = 0xffffffffu;
    const int s = threadIdx.x;
    const int step = ctrl->pair_mode ? 2 : 1;
    const unsigned bits = step == 2 ? 3u : 1u;
    const bool in = s < K / step;
    const int c0 = in ? s * step : 0;
    const int occ0 = in ? ctrl->occupied[c0] : 0;
    const int dn = in ? ctrl->done[c0] : 1;            // (the columns of a pair share every decision)
    const int next = ctrl->q_next, total = ctrl->q_total;
    const bool fin_s = occ0 && dn;
    if (fin_s) {                                 // the per-right-hand-side results (k_stats of the host-driven refill)
        for (int c = c0; c < c0 + step; ++c) {
            const int r = ctrl->rhs[c];
            iters[r] = ctrl->iters[c];
            status[r] = ctrl->status[c];
            relres[r] = ctrl->bb[c] > 0.0 ? sqrt(ctrl->rr[c] / ctrl->bb[c]) : 0.0;
        }
    }
    const bool free_s = in && (!occ0 || fin_s);
    const unsigned finm = __ballot_sync(full, fin_s);
    const unsigned freem = __ballot_sync(full, free_s);
    const int rank = __popc(freem & ((1u << s) - 1u));
    const bool take = free_s && next + rank < total;
    const bool occ = (occ0 && !fin_s) || take;
    if (in) {
        QEntry e = {0.0, 0.0, -1, 0};
        if (take) e = queue[next + rank];
        for (int i = 0; i < step; ++i) {
            const int c = c0 + i;
            ctrl->turn_sp.c[c] = e.c; ctrl->turn_sp.c1[c] = e.c1;
            ctrl->turn_sp.field[c] = e.field < 0 ? -1 : e.field + i;
            ctrl->turn_sp.rhs[c] = e.rhs + i * ctrl->rhs_stride;
            ctrl->occupied[c] = occ ? 1 : 0;
        }
    }
    const unsigned startm = __ballot_sync(full, take || (first && free_s));
    const unsigned occm = __ballot_sync(full, occ);
    const unsigned runm = __ballot_sync(full, occ && (take || !dn));
    const unsigned takem = __ballot_sync(full, take);
    if (s == 0) {
        // slot masks -> column masks
        unsigned fin = 0u, start = 0u;
        for (int i = 0; i < K / step; ++i) {
            if ((finm >> i) & 1u) fin |= bits << (i * step);
            if ((startm >> i) & 1u) start |= bits << (i * step);
        }
        ctrl->q_next = next + __popc(takem);
        ctrl->turn_fin = fin;
        ctrl->turn_start = start;
        ctrl->snap[0] = __popc(occm); ctrl->snap[1] = __popc(runm); ctrl->snap[2] = next + __popc(takem); ctrl->snap[3] = 0;
    }
}

// velocity pairs (IF_FLAG_PAIRS): e_pair[i][j] = e[2i][j] + e[2i+1][j]   (1/2 <u^2 + v^2>: the two spectra add)
__global__ void k_pair_sum(const double* __restrict__ energy, int n_pairs, int n_ells, double* __restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_pairs * n_ells) return;
    const int p = i / n_ells, j = i % n_ells;
    out[i] = energy[(2 * p) * n_ells + j] + energy[(2 * p + 1) * n_ells + j];
}

// H7: k_j = 1/l_j ; E_j = (e_j - e_j+1)/(k_j - k_j+1) ; k_mid_j = sqrt(k_j k_j+1)
__global__ void k_spectrum(const double* __restrict__ energy, const double* __restrict__ ells, int n_fields, int n_ells,
                           double* __restrict__ k_mid, double* __restrict__ E) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int nb = n_ells - 1;
    if (i >= n_fields * nb) return;
    const int f = i / nb, j = i % nb;
    const double k0 = 1.0 / ells[j], k1 = 1.0 / ells[j + 1];
    E[i] = (energy[f * n_ells + j] - energy[f * n_ells + j + 1]) / (k0 - k1);
    if (f == 0) k_mid[j] = sqrt(k0 * k1);
}

// ------------------------------------------------------------------------------------------- column compaction (H5)
// When the queue is empty and at most half of the columns are still running, the survivors move to a narrower
// layout ([row][KN] instead of [row][KW]) so that finished columns stop costing bandwidth.
struct ColMap { int src[KMAX]; };   // new column j <- old column src[j]; -1 = empty

template <int KW, int KN>
__global__ void __launch_bounds__(BLOCK) k_repack(int64_t nv, ColMap map, const double* __restrict__ src,
                                                  double* __restrict__ dst) {
    const int64_t i = (int64_t)blockIdx.x * BLOCK + threadIdx.x;
    if (i >= nv * KN) return;
    const int64_t row = i / KN;
    const int s = map.src[i % KN];
    dst[i] = s >= 0 ? src[row * KW + s] : 0.0;
}

__global__ void k_compact_ctrl(Ctrl* __restrict__ ctrl, ColMap map, int KN) {
    const int j = threadIdx.x;   // one block of KMAX threads
    const int s = j < KN ? map.src[j] : -1;
    double c = 0.0, c1 = 0.0, al = 0.0, be = 0.0, rho = 0.0, bb = 0.0, rr = 0.0;
    int field = -1, rhs = 0, done = 1, epoch = 0, status = 0, iters = 0;
    if (s >= 0) {
        c = ctrl->c[s]; c1 = ctrl->c1[s]; al = ctrl->alpha[s]; be = ctrl->beta[s]; rho = ctrl->rho[s]; bb = ctrl->bb[s]; rr = ctrl->rr[s];
        field = ctrl->field[s]; rhs = ctrl->rhs[s]; done = ctrl->done[s]; epoch = ctrl->epoch[s];
        status = ctrl->status[s]; iters = ctrl->iters[s];
    }
    __syncthreads();
    ctrl->c[j] = c; ctrl->c1[j] = c1; ctrl->starting[j] = 0; ctrl->alpha[j] = al; ctrl->beta[j] = be; ctrl->rho[j] = rho; ctrl->bb[j] = bb; ctrl->rr[j] = rr;
    ctrl->field[j] = field; ctrl->rhs[j] = rhs; ctrl->done[j] = done; ctrl->epoch[j] = epoch;
    ctrl->status[j] = status; ctrl->iters[j] = iters;
    __syncthreads();
    if (j == 0) {
        int any = 0;
        for (int k = 0; k < KMAX; ++k) any |= !ctrl->done[k];
        ctrl->all_done = !any;
    }
}

// ---- tail of the multigrid stream: when the queue is empty and at most half of the columns still run, the survivors
// move to the narrower kernels.  Everything is decided on the device, at the iteration boundary the host enqueues it at.
// k_mg_compact_plan: the column map, occupied slots first in their order (a slot = a column, or a (u, v) pair).
__global__ void k_mg_compact_plan(Ctrl* __restrict__ ctrl, int KW, int KN) {
    const unsigned full = 0xffffffffu;
    const int s = threadIdx.x;
    const int step = ctrl->pair_mode ? 2 : 1;
    const bool in = s < KW / step;
    const bool occ = in && ctrl->occupied[s * step] != 0;
    const unsigned occm = __ballot_sync(full, occ);
    if (s < KMAX) ctrl->cmap[s] = -1;
    __syncwarp();
    if (occ) {
        const int rank = __popc(occm & ((1u << s) - 1u));
        for (int i = 0; i < step; ++i)
            if (rank * step + i < KN) ctrl->cmap[rank * step + i] = s * step + i;
    }
}

// one state vector [nv][KW] -> [nv][KN] through ctrl->cmap; `sel` picks the source of a double-buffered one:
// 0: src0 ;  1: (src0, src1)[ctrl->cur_r] ;  2: (src0, src1)[ctrl->cur_p]
template <int KW, int KN>
__global__ void __launch_bounds__(BLOCK) k_mg_repack(int64_t nv, const Ctrl* __restrict__ ctrl, int sel,
                                                     const double* __restrict__ src0, const double* __restrict__ src1,
                                                     double* __restrict__ dst) {
    const int64_t i = (int64_t)blockIdx.x * BLOCK + threadIdx.x;
    if (i >= nv * KN) return;
    const double* __restrict__ src = sel == 1 ? (ctrl->cur_r ? src1 : src0) : sel == 2 ? (ctrl->cur_p ? src1 : src0) : src0;
    const int64_t row = i / KN;
    const int s = ctrl->cmap[i % KN];
    dst[i] = s >= 0 ? src[row * KW + s] : 0.0;
}

// the control block through the same map; the current buffers of the narrow layout are r'[0] and p'[0]
__global__ void k_mg_compact_ctrl(Ctrl* __restrict__ ctrl, int KN) {
    const int j = threadIdx.x;   // one block of KMAX threads
    const int s = j < KN ? ctrl->cmap[j] : -1;
    double c = 0.0, c1 = 0.0, al = 0.0, be = 0.0, rho = 0.0, bb = 0.0, rr = 0.0;
    int field = -1, rhs = 0, done = 1, epoch = 0, status = 0, iters = 0, starting = 0, occupied = 0;
    if (s >= 0) {
        c = ctrl->c[s]; c1 = ctrl->c1[s]; al = ctrl->alpha[s]; be = ctrl->beta[s]; rho = ctrl->rho[s]; bb = ctrl->bb[s]; rr = ctrl->rr[s];
        field = ctrl->field[s]; rhs = ctrl->rhs[s]; done = ctrl->done[s]; epoch = ctrl->epoch[s];
        status = ctrl->status[s]; iters = ctrl->iters[s]; starting = ctrl->starting[s]; occupied = ctrl->occupied[s];
    }
    __syncthreads();
    ctrl->c[j] = c; ctrl->c1[j] = c1; ctrl->starting[j] = starting; ctrl->alpha[j] = al; ctrl->beta[j] = be; ctrl->rho[j] = rho;
    ctrl->bb[j] = bb; ctrl->rr[j] = rr; ctrl->field[j] = field; ctrl->rhs[j] = rhs; ctrl->done[j] = done; ctrl->epoch[j] = epoch;
    ctrl->status[j] = status; ctrl->iters[j] = iters; ctrl->occupied[j] = occupied;
    __syncthreads();
    if (j == 0) {
        int any = 0;
        for (int k = 0; k < KMAX; ++k) any |= !ctrl->done[k];
        ctrl->all_done = !any;
        ctrl->cur_r = 0;
        ctrl->cur_p = 0;
    }
}

}  // namespace
}  // namespace ifl
