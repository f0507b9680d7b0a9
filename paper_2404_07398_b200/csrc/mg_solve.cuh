// Multigrid-preconditioned CG for large scales (included by solve.cu).
//
//   n = 1:  PCG on (M + c S) x = M phi, x0 = phi, preconditioner B = V = one V cycle of the smoothed-
//           aggregation hierarchy of mg.cu for K = M + c S: damped Jacobi smoothing (one sweep on the mesh, MG_NU_L1 on
//           level 1, MG_NU_COARSE on the coarser levels), dense Cholesky solve on the coarsest level.
//   n = 2:  PCG on (M + c S M^-1 S) x = M phi with the product preconditioner B = V M V, V = the same V cycle for
//           K = M + mu S, mu = sqrt(c):  K M^-1 K = M + 2 mu S + c S M^-1 S, and for every eigenvalue lambda of M^-1 S
//           1 <= (1 + mu lambda)^2 / (1 + c lambda^2) <= 2, so with exact inner solves the condition number is <= 2
//           (PAPER.md:207 names the loss of convergence of the biharmonic filter at large l as the open problem).
//   V is a fixed symmetric positive definite operator per column (fixed sweep counts, the same damping before and
//   after the coarse correction), hence so are B = V and B = V M V, and plain PCG applies.
// K = 16 columns at a time (8 or 4 when a call has no more right-hand sides than that, and for the tail of the stream:
// every kernel here takes the width as a template parameter), every column with its own c, alpha, beta and stop time;
// all per-column scalars live in the device control block (Ctrl), so ONE iteration is a fixed launch sequence, captured
// in a CUDA graph by solve.cu (written for K = 16):
//       k_spmm<16, CG1>  (n = 2: CG2A, CG2B)   p' = z + beta p ; x += alpha p ; q = A p' ; alpha' = rho / p'.q
//       k_spmm<16, MGR>      r' = r - alpha' q ; e = omega r'/d ; t = r' - K e    (residual update, first sweep of V on
//                            level 0 and its residual in one pass), then restriction, coarse levels, prolongation
//       k_spmm<16, AX> sub 3 z = last sweep ; rho' = r'.z ; ||r'||^2 ; beta ; stop test      (CG bookkeeping)
//   n = 2: the last sweep of the first cycle is sub 5 (y = V r', w = M y, rho' = y.w, bookkeeping), then a second
//   cycle on w (k_spmm<16, MGR0>, transfers, coarse levels, sub 2) gives z = V w.
// A (re)started column (Ctrl::starting, set by k_mg_start) joins at an iteration boundary with x = 0, z = phi, r = M phi:
// its first iteration has alpha = 1, which makes kernel A and the fused residual kernel form r0 = M phi - A phi on the
// way (no pass of its own over the matrix), and ends with rho = r0.z0, beta = 0 -- the start of PCG from x0 = phi -- so
// columns are refilled from the queue as in the Jacobi path and the host never waits inside the loop (on large meshes
// the ending and starting of columns is itself part of every iteration's graph: k_turn_plan, solve.cu).
// With IF_FLAG_VECTOR the level-0 kernels are the VEC variants (coupled operator D_2 with the metric terms), the levels
// below work per component.
// The stop test is the same as in the Jacobi path: recursive ||r||_2 <= tol ||M phi||_2.
#pragma once

namespace ifl {
namespace {

constexpr int MGK = 16;               // columns of the multigrid path at full width (buffers are sized for it)
constexpr size_t MG_FACTOR_SMEM = 2 * (size_t)MG_COARSEST * (MG_COARSEST + 1) * sizeof(double);   // k_mg_coarse_factor
constexpr int MG_REFILL_MIN = 1;      // stopped columns are restarted as soon as this many are free (solve.cu)
// right-hand sides below this many mean edge lengths stay on the Jacobi path (option mg_min_ell = 0)
constexpr double MG_MIN_ELL_N1 = 0.5;
constexpr double MG_MIN_ELL_N2 = 0.5;
// n = 2: sweeps per side of the cycle on the mesh and on level 1 (Chebyshev-root dampings, mg_omegas)
constexpr int MG_NU0_N2 = 4;
constexpr int MG_NU1_N2 = 2;
constexpr int MG_UB = 4;              // matrix entries a thread has in flight in the CSR kernels of the hierarchy
#ifndef IF_MG_BPS
#define IF_MG_BPS 6                   // blocks per SM of the CSR kernels (what their registers allow: one full wave)
#endif
#ifndef IF_MG_MINB
#define IF_MG_MINB 6
#endif
#ifndef IF_MG_WIDE
#define IF_MG_WIDE 24                 // mean row length from which a row is split over four entry slices
#endif

struct MgMat {                        // one level's (S, M) pair
    const int64_t* __restrict__ rowptr;
    const int32_t* __restrict__ col;
    const double2* __restrict__ sm;
    const double2* __restrict__ diag;
    int64_t n;
    double omega;                     // Jacobi damping of the smoother on this level
};

// A row is handled by TPR * SL threads (TPR = K / 2): column pair l = tid % TPR, entry slice sl = (tid / TPR) % SL.  SL = 1 for the
// short rows of the fine levels; SL = 4 (one row per warp, slices added with two shuffles) for the coarse levels
// whose rows have hundreds of entries and would otherwise be walked serially.
// MODE 0: y = A x ;  MODE 1: y = r - A x ;  MODE 2: y = x + omega (r - A x) / d        with A = M + c S per column
template <int MODE, int SL, int K = MGK>
__global__ void __launch_bounds__(BLOCK, IF_MG_MINB) k_mg_apply(MgMat g, const Ctrl* __restrict__ ctrl, const double* __restrict__ x,
                                                    const double* __restrict__ r, double* __restrict__ y) {
    constexpr int TPR = K / 2, RPW = 32 / TPR;         // lanes per row (one column pair each), rows per warp at SL = 1
    constexpr int WPB = BLOCK / (TPR * SL);
    const int l = threadIdx.x % TPR, sl = (threadIdx.x / TPR) % SL;
    if (ctrl->all_done) return;
    const double2 cc = ld2(ctrl->c1, 2 * l);
    // (rows are padded to whole warps by the loop bound: every lane of a warp takes part in the shuffles)
    // a block walks a contiguous range of rows, WPB at a time: neighbouring rows gather the same rows of x, which
    // the L1 then serves (a grid-stride assignment sends every gather to the L2)
    const int64_t per_block = ((g.n + gridDim.x - 1) / gridDim.x + WPB - 1) / WPB * WPB;
    const int64_t row_end = min((int64_t)(blockIdx.x + 1) * per_block, (g.n + RPW - 1) / RPW * RPW);
    for (int64_t row = (int64_t)blockIdx.x * per_block + threadIdx.x / (TPR * SL); row < row_end; row += WPB) {
        double2 s = {0.0, 0.0};
        const bool live = row < g.n;
        const int64_t k1 = live ? g.rowptr[row + 1] : 0;
        // MG_UB entries at a time: their column ids and values first, then the gathers, then the multiply-adds
        for (int64_t k = live ? g.rowptr[row] + sl : 0; k < k1; k += MG_UB * SL) {
            double2 w[MG_UB], v[MG_UB];
            int32_t cj[MG_UB];
#pragma unroll
            for (int j = 0; j < MG_UB; ++j) {
                const int64_t kk = k + j * SL < k1 ? k + j * SL : k;
                cj[j] = g.col[kk];
                w[j] = g.sm[kk];
            }
#pragma unroll
            for (int j = 0; j < MG_UB; ++j) v[j] = ld2(x, (int64_t)cj[j] * K + 2 * l);
#pragma unroll
            for (int j = 0; j < MG_UB; ++j)
                if (k + j * SL < k1) {
                    s.x = fma(fma(cc.x, w[j].x, w[j].y), v[j].x, s.x);
                    s.y = fma(fma(cc.y, w[j].x, w[j].y), v[j].y, s.y);
                }
        }
        if (SL >= 2) { s.x += __shfl_xor_sync(0xffffffffu, s.x, TPR);  s.y += __shfl_xor_sync(0xffffffffu, s.y, TPR); }
        if (SL >= 4) { s.x += __shfl_xor_sync(0xffffffffu, s.x, 2 * TPR); s.y += __shfl_xor_sync(0xffffffffu, s.y, 2 * TPR); }
        if (sl != 0 || !live) continue;
        const int64_t ri = row * K + 2 * l;
        if (MODE == 0) {
            st2(y, ri, s);
        } else {
            const double2 rv = ld2(r, ri);
            double2 t = {rv.x - s.x, rv.y - s.y};
            if (MODE == 2) {
                const double2 d = g.diag[row];
                const double2 xv = ld2(x, ri);
                t.x = fma(g.omega * t.x, 1.0 / fma(cc.x, d.x, d.y), xv.x);
                t.y = fma(g.omega * t.y, 1.0 / fma(cc.y, d.x, d.y), xv.y);
            }
            st2(y, ri, t);
        }
    }
}

// e = omega r / d  (Jacobi sweep from a zero initial guess)
template <int K = MGK>
__global__ void __launch_bounds__(BLOCK) k_mg_jacobi0(MgMat g, const Ctrl* __restrict__ ctrl, const double* __restrict__ r,
                                                      double* __restrict__ e) {
    constexpr int TPR = K / 2;
    constexpr int ROWS = BLOCK / TPR;
    const int l = threadIdx.x % TPR;
    if (ctrl->all_done) return;
    const double2 cc = ld2(ctrl->c1, 2 * l);
    for (int64_t row = (int64_t)blockIdx.x * ROWS + threadIdx.x / TPR; row < g.n; row += (int64_t)gridDim.x * ROWS) {
        const int64_t ri = row * K + 2 * l;
        const double2 d = g.diag[row];
        const double2 rv = ld2(r, ri);
        st2(e, ri, make_double2(g.omega * rv.x / fma(cc.x, d.x, d.y), g.omega * rv.y / fma(cc.y, d.x, d.y)));
    }
}

// y (+)= B x for a scalar CSR matrix (restriction R, prolongation P); thread mapping as above
template <int ACC, int SL, int K = MGK>
__global__ void __launch_bounds__(BLOCK, IF_MG_MINB) k_mg_csr(const int64_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                                                  const double* __restrict__ val, int64_t n,
                                                  const Ctrl* __restrict__ ctrl, const double* __restrict__ x,
                                                  double* __restrict__ y) {
    constexpr int TPR = K / 2, RPW = 32 / TPR;
    constexpr int WPB = BLOCK / (TPR * SL);
    if (ctrl->all_done) return;
    const int l = threadIdx.x % TPR, sl = (threadIdx.x / TPR) % SL;
    const int64_t per_block = ((n + gridDim.x - 1) / gridDim.x + WPB - 1) / WPB * WPB;   // contiguous rows per block
    const int64_t row_end = min((int64_t)(blockIdx.x + 1) * per_block, (n + RPW - 1) / RPW * RPW);
    for (int64_t row = (int64_t)blockIdx.x * per_block + threadIdx.x / (TPR * SL); row < row_end; row += WPB) {
        double2 s = {0.0, 0.0};
        const bool live = row < n;
        const int64_t k1 = live ? rowptr[row + 1] : 0;
        for (int64_t k = live ? rowptr[row] + sl : 0; k < k1; k += MG_UB * SL) {
            double w[MG_UB];
            double2 v[MG_UB];
            int32_t cj[MG_UB];
#pragma unroll
            for (int j = 0; j < MG_UB; ++j) {
                const int64_t kk = k + j * SL < k1 ? k + j * SL : k;
                cj[j] = col[kk];
                w[j] = val[kk];
            }
#pragma unroll
            for (int j = 0; j < MG_UB; ++j) v[j] = ld2(x, (int64_t)cj[j] * K + 2 * l);
#pragma unroll
            for (int j = 0; j < MG_UB; ++j)
                if (k + j * SL < k1) {
                    s.x = fma(w[j], v[j].x, s.x);
                    s.y = fma(w[j], v[j].y, s.y);
                }
        }
        if (SL >= 2) { s.x += __shfl_xor_sync(0xffffffffu, s.x, TPR);  s.y += __shfl_xor_sync(0xffffffffu, s.y, TPR); }
        if (SL >= 4) { s.x += __shfl_xor_sync(0xffffffffu, s.x, 2 * TPR); s.y += __shfl_xor_sync(0xffffffffu, s.y, 2 * TPR); }
        if (sl != 0 || !live) continue;
        const int64_t ri = row * K + 2 * l;
        if (ACC) { const double2 o = ld2(y, ri); s.x += o.x; s.y += o.y; }
        st2(y, ri, s);
    }
}

// Prolongation onto the mesh fused with the first sweep:  e = omega r / d + P e_c  (8 threads per row as above; the
// prolongator has 2.6 entries per row).  k_spmm<16, MGR> then does not store its e = omega r'/d, and this kernel
// reads r' where k_mg_csr<1, 1> would read e back: one pass over a [V][16] vector less per iteration.
template <int K = MGK>
__global__ void __launch_bounds__(BLOCK, IF_MG_MINB) k_mg_prolong0(const int64_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                                                       const double* __restrict__ val, MgMat g, const Ctrl* __restrict__ ctrl,
                                                       const double* __restrict__ x, const double* __restrict__ r0,
                                                       const double* __restrict__ r1, int r_select,
                                                       double* __restrict__ y) {
    constexpr int TPR = K / 2;
    constexpr int WPB = BLOCK / TPR;
    // r_select: the residual k_spmm<16, MGR> has just written, r[cur_r ^ 1] of the double buffer (r0, r1); else r0
    const double* __restrict__ r = r_select ? (ctrl->cur_r ? r0 : r1) : r0;
    const int l = threadIdx.x % TPR;
    if (ctrl->all_done) return;
    const double2 cc = ld2(ctrl->c1, 2 * l);
    const int64_t n = g.n;
    const int64_t per_block = ((n + gridDim.x - 1) / gridDim.x + WPB - 1) / WPB * WPB;   // contiguous rows per block
    const int64_t row_end = min((int64_t)(blockIdx.x + 1) * per_block, n);
    for (int64_t row = (int64_t)blockIdx.x * per_block + threadIdx.x / TPR; row < row_end; row += WPB) {
        const int64_t ri = row * K + 2 * l;
        const double2 rv = ld2(r, ri);
        const double2 d = g.diag[row];
        double2 s = {0.0, 0.0};
        const int64_t k1 = rowptr[row + 1];
        for (int64_t k = rowptr[row]; k < k1; k += MG_UB) {
            double w[MG_UB];
            double2 v[MG_UB];
            int32_t cj[MG_UB];
#pragma unroll
            for (int j = 0; j < MG_UB; ++j) {
                const int64_t kk = k + j < k1 ? k + j : k;
                cj[j] = col[kk];
                w[j] = val[kk];
            }
#pragma unroll
            for (int j = 0; j < MG_UB; ++j) v[j] = ld2(x, (int64_t)cj[j] * K + 2 * l);
#pragma unroll
            for (int j = 0; j < MG_UB; ++j)
                if (k + j < k1) {
                    s.x = fma(w[j], v[j].x, s.x);
                    s.y = fma(w[j], v[j].y, s.y);
                }
        }
        // the same arithmetic as the e of k_spmm<16, MGR> (rcp_pos, this order of the products)
        s.x += g.omega * rv.x * rcp_pos(fma(cc.x, d.x, d.y));
        s.y += g.omega * rv.y * rcp_pos(fma(cc.y, d.x, d.y));
        st2(y, ri, s);
    }
}

// ---- row-block kernels of the cycle (round 2).  The CSR kernels above walk a dependent chain per row -- row pointer ->
// entries -> gathered rows of x, three trips to memory, the first two to lines nobody has touched -- and are bound by
// exactly that chain: 9 latencies per group of four rows on level 1 (12.5 entries per row in batches of four) give
// 0.20 ms for its 815 k rows on config 4 (measured 0.216), 3 latencies give 0.64 ms for the prolongation onto the mesh
// (measured 0.64).  Here a persistent CTA walks tiles of MG_TILE consecutive rows through a ring of shared-memory
// stages: one thread issues bulk async copies (TMA, mbarrier complete_tx) of the tile's row pointers, its contiguous
// range of entries (columns, values) and its own rows of the per-row operands two tiles ahead, and the only trip to
// memory left in a row's chain is the gather itself, eight entries in flight per thread.  Same sums in the same order
// as the CSR kernels (entry by entry), so the results are bit-identical.
// (First form tried: a persistent CTA with a ring of stages that also held the own-row vectors -- 16 warps per SM and
// a block barrier per 64 rows: restriction 0.34 -> 0.93 ms, level 1 0.62 -> 1.06 ms.  Rejected.)
enum RowsKind { ROWS_RES = 0, ROWS_SWEEP = 1, ROWS_SET = 2, ROWS_ACC = 3, ROWS_PROLONG0 = 4 };
//   ROWS_RES      y = r - K x                      K = M + c1 S, (S, M) pairs per entry
//   ROWS_SWEEP    y = x + omega (r - K x) / d
//   ROWS_SET      y = B x                          scalar entries (restriction)
//   ROWS_ACC      y += B x                         (prolongation)
//   ROWS_PROLONG0 y = omega r / d + B x            (prolongation onto the mesh fused with the first sweep, as k_mg_prolong0)
struct RowsArgs {
    const int64_t* rowptr;
    const int32_t* col;
    const void* val;          // double2 (S, M) for RES / SWEEP, double for the others
    const double2* diag;      // SWEEP, PROLONG0: (S_ii, M_ii)
    int64_t n;                // rows
    const double* x;          // the gathered vector
    const double* own0;       // RES, SWEEP, PROLONG0: r ;  ACC: y (read)
    const double* own1;       // SWEEP: x (own rows) ;  PROLONG0 with r_select: the second residual buffer
    double* y;
    double omega;
    int r_select;             // PROLONG0: r = (own0, own1)[cur_r ^ 1] (see SpmmArgs::r_select)
    int cap;                  // entries a stage holds (MgLevel::cap_*)
    int stages;
};

constexpr int ROWS_PER_CTA = 2 * MG_TILE;      // rows of one CTA (MgLevel::cap_* bounds the entries of MG_TILE rows)

struct RowsLayout { uint32_t col, val, bytes; };      // offsets inside the CTA's shared memory
template <int KIND>
__host__ __device__ inline RowsLayout rows_layout(int cap) {
    constexpr bool PAIR = KIND <= ROWS_SWEEP;
    const uint32_t ce = (uint32_t)cap * (ROWS_PER_CTA / MG_TILE);      // entries of the CTA's rows, at most
    RowsLayout L;
    L.col = (uint32_t)((ROWS_PER_CTA + 2) * 8);
    L.val = L.col + (((ce + 4u) * 4u + 15u) & ~15u);
    L.bytes = L.val + (PAIR ? ce * 16u : (((ce + 2u) * 8u + 15u) & ~15u)) + 16u;     // + the mbarrier
    return L;
}

// One CTA = ROWS_PER_CTA consecutive rows: thread 0 asks for the two row pointers that bound the CTA's entries and
// issues three bulk copies (row pointers, columns, values); meanwhile every thread loads the own-row operands of its
// rows; after the mbarrier the rows are walked with the gathers as the only trips to memory.  Several CTAs are
// resident per SM, so one CTA's copy phase hides behind the others' gathers (no block barrier inside the loop).
#ifndef IF_ROWS_UB_PAIR
#define IF_ROWS_UB_PAIR 8
#endif
#ifndef IF_ROWS_MINB_PAIR
#define IF_ROWS_MINB_PAIR 2
#endif
template <int KIND, int K = MGK>
__global__ void __launch_bounds__(BLOCK, KIND <= 1 ? IF_ROWS_MINB_PAIR : 4) k_mg_rows(RowsArgs a, const Ctrl* __restrict__ ctrl) {
    constexpr int TPR = K / 2;
    constexpr bool PAIR = KIND <= ROWS_SWEEP;
    // gathers a thread has in flight: rows of the level matrices have a dozen entries and more, prolongator rows 2-5
    constexpr int ROWS_UB = (KIND == ROWS_ACC || KIND == ROWS_PROLONG0) ? 4 : (KIND <= ROWS_SWEEP ? IF_ROWS_UB_PAIR : 8);
    constexpr bool OWN0 = KIND != ROWS_SET, OWN1 = KIND == ROWS_SWEEP, DIAG = KIND == ROWS_SWEEP || KIND == ROWS_PROLONG0;
    constexpr int RPT = ROWS_PER_CTA / (BLOCK / TPR);      // rows per thread group
    if (ctrl->all_done) return;
    extern __shared__ __align__(128) unsigned char smem[];
    const RowsLayout L = rows_layout<KIND>(a.cap);
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem + L.bytes - 16);
    const int tid = threadIdx.x, l = tid % TPR, g = tid / TPR;
    const int64_t r0 = (int64_t)blockIdx.x * ROWS_PER_CTA;
    const int nr = (int)min((int64_t)ROWS_PER_CTA, a.n - r0);
    if (tid == 0) {
        mbar_init(bar, 1);
        fence_proxy_async();
        const int64_t k0 = a.rowptr[r0], k1 = a.rowptr[r0 + nr];
        const uint32_t rp_bytes = ((uint32_t)(nr + 1) * 8u + 15u) & ~15u;
        const int64_t kA = k0 & ~3LL;
        const uint32_t col_bytes = ((uint32_t)(k1 - kA) * 4u + 15u) & ~15u;
        const int64_t kB = PAIR ? k0 : (k0 & ~1LL);
        const uint32_t val_bytes = PAIR ? (uint32_t)(k1 - k0) * 16u : (((uint32_t)(k1 - kB) * 8u + 15u) & ~15u);
        mbar_expect_tx(bar, rp_bytes + col_bytes + val_bytes);
        bulk_load(smem, a.rowptr + r0, rp_bytes, bar);
        bulk_load(smem + L.col, a.col + kA, col_bytes, bar);
        if (PAIR) bulk_load(smem + L.val, static_cast<const double2*>(a.val) + k0, val_bytes, bar);
        else bulk_load(smem + L.val, static_cast<const double*>(a.val) + kB, val_bytes, bar);
    }
    double2 cc = {0.0, 0.0};
    if (PAIR || KIND == ROWS_PROLONG0) cc = ld2(ctrl->c1, 2 * l);
    const double* own0 = a.own0;
    if (KIND == ROWS_PROLONG0 && a.r_select) own0 = ctrl->cur_r ? a.own0 : a.own1;
    // own-row operands: those of the thread's first row are in flight while the bulk copies land, those of row i + 1
    // while row i is gathered
    double2 o0n = {0.0, 0.0}, o1n = {0.0, 0.0}, dgn = {0.0, 0.0};
    auto load_own = [&](int r) {
        if (r < nr) {
            const int64_t ri = (r0 + r) * K + 2 * l;
            if (OWN0) o0n = ld2(own0, ri);
            if (OWN1) o1n = ld2(a.own1, ri);
            if (DIAG) dgn = a.diag[r0 + r];
        }
    };
    load_own(g);
    __syncthreads();            // the mbarrier is initialised
    mbar_wait(bar, 0u);
    const int64_t* srp = reinterpret_cast<const int64_t*>(smem);
    const int32_t* scol = reinterpret_cast<const int32_t*>(smem + L.col);
    const double2* sval2 = reinterpret_cast<const double2*>(smem + L.val);
    const double* sval1 = reinterpret_cast<const double*>(smem + L.val);
    const int64_t k0 = srp[0];
    const int64_t kA = k0 & ~3LL, kB = PAIR ? k0 : (k0 & ~1LL);
#pragma unroll
    for (int i = 0; i < RPT; ++i) {
        const int r = g + i * (BLOCK / TPR);
        if (r >= nr) break;
        const double2 o0c = o0n, o1c = o1n, dgc = dgn;
        load_own(r + BLOCK / TPR);
        const int64_t kb = srp[r], ke = srp[r + 1];
        double2 s = {0.0, 0.0};
        for (int64_t k = kb; k < ke; k += ROWS_UB) {
            int32_t cj[ROWS_UB];
            double2 v[ROWS_UB];
#pragma unroll
            for (int j = 0; j < ROWS_UB; ++j) cj[j] = scol[(k + j < ke ? k + j : k) - kA];
#pragma unroll
            for (int j = 0; j < ROWS_UB; ++j) v[j] = ld2(a.x, (int64_t)cj[j] * K + 2 * l);
#pragma unroll
            for (int j = 0; j < ROWS_UB; ++j)
                if (k + j < ke) {
                    if (PAIR) {
                        const double2 w = sval2[k + j - k0];
                        s.x = fma(fma(cc.x, w.x, w.y), v[j].x, s.x);
                        s.y = fma(fma(cc.y, w.x, w.y), v[j].y, s.y);
                    } else {
                        const double w = sval1[k + j - kB];
                        s.x = fma(w, v[j].x, s.x);
                        s.y = fma(w, v[j].y, s.y);
                    }
                }
        }
        const int64_t ri = (r0 + r) * K + 2 * l;
        if (KIND == ROWS_SET) {
            st2(a.y, ri, s);
        } else if (KIND == ROWS_ACC) {
            st2(a.y, ri, make_double2(s.x + o0c.x, s.y + o0c.y));
        } else if (KIND == ROWS_PROLONG0) {
            const double2 rv = o0c, d = dgc;
            s.x += a.omega * rv.x * rcp_pos(fma(cc.x, d.x, d.y));       // the arithmetic of k_mg_prolong0
            s.y += a.omega * rv.y * rcp_pos(fma(cc.y, d.x, d.y));
            st2(a.y, ri, s);
        } else {
            const double2 rv = o0c;
            double2 t = {rv.x - s.x, rv.y - s.y};
            if (KIND == ROWS_SWEEP) {
                const double2 d = dgc, xv = o1c;
                t.x = fma(a.omega * t.x, 1.0 / fma(cc.x, d.x, d.y), xv.x);   // the arithmetic of k_mg_apply<2, *>
                t.y = fma(a.omega * t.y, 1.0 / fma(cc.y, d.x, d.y), xv.y);
            }
            st2(a.y, ri, t);
        }
    }
}

// Coarsest level (n <= MG_COARSEST unknowns).  K = M + c1 S depends on the column only through c1, which changes when
// the column is (re)started -- not from cycle to cycle -- so its inverse is formed once per column start
// (k_mg_coarse_factor: dense Cholesky K = L L^T in shared memory, L^-1 by forward substitution on the unit vectors,
// K^-1 = L^-T L^-1, symmetric by construction; one block per column) and a cycle only multiplies by it.  Round 1
// factorised in every cycle: 118 us of the 385 us the levels >= 2 took per cycle on config 4.
// inv: [MGK][MG_COARSEST][MG_COARSEST] in the workspace.
__global__ void __launch_bounds__(64) k_mg_coarse_factor(MgMat g, const Ctrl* __restrict__ ctrl, unsigned mask,
                                                         double* __restrict__ inv) {
    extern __shared__ double coarse_sm[];            // two [MG_COARSEST][MG_COARSEST + 1] arrays (65 KB: opt-in)
    double (*a)[MG_COARSEST + 1] = reinterpret_cast<double (*)[MG_COARSEST + 1]>(coarse_sm);
    double (*li)[MG_COARSEST + 1] = reinterpret_cast<double (*)[MG_COARSEST + 1]>(coarse_sm + MG_COARSEST * (MG_COARSEST + 1));
    const int c = blockIdx.x, t = threadIdx.x, n = (int)g.n;
    if (mask == MASK_TURN_START) mask = ctrl->turn_start;
    if (!((mask >> c) & 1u)) return;
    const double cc = ctrl->c1[c];
    for (int i = t; i < n; i += 64)
        for (int j = 0; j < n; ++j) { a[i][j] = 0.0; li[i][j] = 0.0; }
    __syncthreads();
    for (int i = t; i < n; i += 64)
        for (int64_t k = g.rowptr[i]; k < g.rowptr[i + 1]; ++k) a[i][g.col[k]] += fma(cc, g.sm[k].x, g.sm[k].y);
    __syncthreads();
    for (int k = 0; k < n; ++k) {                 // right-looking Cholesky, lower triangle
        if (t == 0) a[k][k] = sqrt(a[k][k]);
        __syncthreads();
        for (int i = k + 1 + t; i < n; i += 64) a[i][k] /= a[k][k];
        __syncthreads();
        for (int i = k + 1 + t; i < n; i += 64)
            for (int j = k + 1; j <= i; ++j) a[i][j] -= a[i][k] * a[j][k];
        __syncthreads();
    }
    // column j of L^-1 (thread j): L y = e_j by forward substitution; y_i = 0 for i < j
    for (int j = t; j < n; j += 64)
        for (int i = j; i < n; ++i) {
            double s = i == j ? 1.0 : 0.0;
            for (int k = j; k < i; ++k) s -= a[i][k] * li[k][j];
            li[i][j] = s / a[i][i];
        }
    __syncthreads();
    // K^-1 = L^-T L^-1: entry (i, j) = sum_k li[k][i] li[k][j], k >= max(i, j); thread i fills row i
    double* out = inv + (size_t)c * MG_COARSEST * MG_COARSEST;
    for (int i = t; i < n; i += 64)
        for (int j = 0; j < n; ++j) {
            double s = 0.0;
            for (int k = (i > j ? i : j); k < n; ++k) s = fma(li[k][i], li[k][j], s);
            out[i * MG_COARSEST + j] = s;
        }
}

// e = K^-1 r on the coarsest level, one block per column
template <int K = MGK>
__global__ void __launch_bounds__(64) k_mg_coarse(MgMat g, const Ctrl* __restrict__ ctrl, const double* __restrict__ inv,
                                                  const double* __restrict__ r, double* __restrict__ e) {
    __shared__ double v[MG_COARSEST];
    const int c = blockIdx.x, t = threadIdx.x, n = (int)g.n;
    if (ctrl->all_done) return;
    for (int i = t; i < n; i += 64) v[i] = r[(int64_t)i * K + c];
    __syncthreads();
    const double* a = inv + (size_t)c * MG_COARSEST * MG_COARSEST;
    for (int i = t; i < n; i += 64) {
        double s = 0.0;
        for (int j = 0; j < n; ++j) s = fma(a[i * MG_COARSEST + j], v[j], s);
        e[(int64_t)i * K + c] = s;
    }
}

// ------------------------------------------------------------------------------------------- host side
struct MgBuffers {
    double *x, *r[2], *p[2], *q, *za, *zb, *t;  // level 0, [n][16]; r is double-buffered (k_spmm<16, MGR>)
    double* lev[MG_MAX_LEVELS][4];              // levels >= 1: R, E, T, E2
    double* coarse_inv;                         // [MGK][MG_COARSEST][MG_COARSEST]: K^-1 of the coarsest level per column
};

// level-0 vectors beyond the Jacobi workspace: za (e), zb (z), the second r; for n = 1 also t (the n = 2 workspace has one)
inline size_t mg_extra_bytes(const if_mesh_s* h, int order_n) {
    if (h->mg_levels < 2) return 0;
    size_t b = (order_n == 1 ? 4 : 3) * align_up((size_t)h->n_vert * MGK * sizeof(double));
    for (int l = 1; l < h->mg_levels; ++l) b += 4 * align_up((size_t)h->mg[l].n * MGK * sizeof(double));
    b += align_up((size_t)MGK * MG_COARSEST * MG_COARSEST * sizeof(double));
    return b;
}

inline MgBuffers mg_layout(const if_mesh_s* h, const Workspace& w, int order_n) {
    MgBuffers m{};
    m.x = w.x; m.r[0] = w.z; m.p[0] = w.p0; m.p[1] = w.p1; m.q = w.q;
    char* p = static_cast<char*>(w.mg_extra);
    size_t off = 0;
    auto take = [&](size_t bytes) { void* r = p + off; off += align_up(bytes); return r; };
    m.za = (double*)take((size_t)h->n_vert * MGK * sizeof(double));
    m.zb = (double*)take((size_t)h->n_vert * MGK * sizeof(double));
    m.r[1] = (double*)take((size_t)h->n_vert * MGK * sizeof(double));
    m.t = order_n == 1 ? (double*)take((size_t)h->n_vert * MGK * sizeof(double)) : w.t;
    for (int l = 1; l < h->mg_levels; ++l)
        for (int k = 0; k < 4; ++k) m.lev[l][k] = (double*)take((size_t)h->mg[l].n * MGK * sizeof(double));
    m.coarse_inv = (double*)take((size_t)MGK * MG_COARSEST * MG_COARSEST * sizeof(double));
    return m;
}

// the buffers of the phase in progress: the layout of the workspace, or what a compaction of the tail made of it
inline MgBuffers mg_buffers(const Run& r) {
    return r.mgb ? *static_cast<const MgBuffers*>(r.mgb) : mg_layout(r.h, r.w, r.order_n);
}

// level 0: the prolongation kernel can form e = omega r'/d itself (short prolongator rows only)
inline bool mg_fused_prolongation(const MgLevel& g) { return g.p_nnz < IF_MG_WIDE * g.n; }
inline MgMat mg_mat(const MgLevel& g) { return MgMat{g.rowptr, g.col, g.sm, g.diag, g.n, g.omega}; }
inline int mg_grid(const if_mesh_s* h, int64_t n, int tpr, int sl = 1) {
    const int64_t rows = BLOCK / (tpr * sl);
    return (int)std::max<int64_t>(1, std::min<int64_t>((n + rows - 1) / rows, (int64_t)h->n_sm * IF_MG_BPS));
}

// groups of the per-kernel timing (if_stats.mg_kernel_seconds)
enum { MGT_A = 0, MGT_MGR = 1, MGT_RESTRICT0 = 2, MGT_LEVEL1 = 3, MGT_COARSE = 4, MGT_PROLONG0 = 5, MGT_LAST = 6 };

#ifndef IF_MG_ROWS
#define IF_MG_ROWS 1                 // 0: the CSR kernels everywhere (A/B measurements)
#endif
constexpr size_t ROWS_SMEM_MAX = 200 * 1024;      // dynamic shared memory a k_mg_rows CTA may ask for
constexpr size_t ROWS_SMEM_SM = 220 * 1024;       // what the CTAs of one SM share

// Launch k_mg_rows<KIND> if the entries of a CTA's rows fit its shared memory; *done = false means "use the CSR kernel".
template <int KIND, int K>
int launch_rows(const Run& r, RowsArgs a, int cap, bool* done) {
    *done = false;
    if (!IF_MG_ROWS || cap <= 0 || a.n < 4 * ROWS_PER_CTA) return IF_OK;
    const RowsLayout L = rows_layout<KIND>(cap);
    if (L.bytes > ROWS_SMEM_MAX / 3) return IF_OK;          // fewer than three CTAs per SM: the copy phases would show
    a.cap = cap;
    a.stages = 1;
    const unsigned grid = (unsigned)((a.n + ROWS_PER_CTA - 1) / ROWS_PER_CTA);
    k_mg_rows<KIND, K><<<grid, BLOCK, L.bytes, r.st>>>(a, r.w.ctrl);
    IF_LAUNCH_CHECK();
    *done = true;
    return IF_OK;
}

template <int K>
int mg_setup(Run& r) {
    const if_mesh_s* h = r.h;
    IF_CUDA_TRY(cudaFuncSetAttribute(k_mg_rows<ROWS_RES, K>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ROWS_SMEM_MAX));
    IF_CUDA_TRY(cudaFuncSetAttribute(k_mg_rows<ROWS_SWEEP, K>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ROWS_SMEM_MAX));
    IF_CUDA_TRY(cudaFuncSetAttribute(k_mg_rows<ROWS_SET, K>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ROWS_SMEM_MAX));
    IF_CUDA_TRY(cudaFuncSetAttribute(k_mg_rows<ROWS_ACC, K>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ROWS_SMEM_MAX));
    IF_CUDA_TRY(cudaFuncSetAttribute(k_mg_rows<ROWS_PROLONG0, K>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ROWS_SMEM_MAX));
    IF_CUDA_TRY(cudaFuncSetAttribute(k_mg_coarse_factor, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)MG_FACTOR_SMEM));
    const int64_t tiles = (h->n_vert + TILE_ROWS - 1) / TILE_ROWS;
    int rc;
    if (r.vec) {      // vector filter: the coupled operator in the level-0 kernels of the cycle
        if ((rc = resident_grid(k_spmm<K, MODE_AX, true>, TileSmem<K, MODE_AX, true>::bytes, h->n_sm, tiles, &r.mgg.ax, SpmmCfg<K, MODE_AX>::NT))) return rc;
        if ((rc = resident_grid(k_spmm<K, MODE_MGR, true>, TileSmem<K, MODE_MGR, true>::bytes, h->n_sm, tiles, &r.mgg.mgr, SpmmCfg<K, MODE_MGR>::NT))) return rc;
        if (r.order_n == 2 &&
            (rc = resident_grid(k_spmm<K, MODE_MGR0, true>, TileSmem<K, MODE_MGR0, true>::bytes, h->n_sm, tiles, &r.mgg.mgr0, SpmmCfg<K, MODE_MGR0>::NT))) return rc;
        return IF_OK;
    }
    if ((rc = resident_grid(k_spmm<K, MODE_AX>, TileSmem<K, MODE_AX>::bytes, h->n_sm, tiles, &r.mgg.ax, SpmmCfg<K, MODE_AX>::NT))) return rc;
    if ((rc = resident_grid(k_spmm<K, MODE_MGR>, TileSmem<K, MODE_MGR>::bytes, h->n_sm, tiles, &r.mgg.mgr, SpmmCfg<K, MODE_MGR>::NT))) return rc;
    if (r.order_n == 2 &&
        (rc = resident_grid(k_spmm<K, MODE_MGR0>, TileSmem<K, MODE_MGR0>::bytes, h->n_sm, tiles, &r.mgg.mgr0, SpmmCfg<K, MODE_MGR0>::NT))) return rc;
    return IF_OK;
}

// y = R x (restriction of level l, rows = the coarse level) and y += P x (prolongation, rows = level l)
template <int K>
int mg_restrict(const Run& r, const MgLevel& g, const double* x, double* y) {
    const if_mesh_s* h = r.h;
    const bool wide_r = g.p_nnz >= IF_MG_WIDE * g.n_coarse;
    bool done = false;
    int rc;
    if (!wide_r) {
        RowsArgs a{g.r_rowptr, g.r_col, g.r_val, nullptr, g.n_coarse, x, nullptr, nullptr, y, 0.0, 0, 0, 0};
        if ((rc = launch_rows<ROWS_SET, K>(r, a, g.cap_r, &done))) return rc;
        if (done) return IF_OK;
    }
    if (wide_r) k_mg_csr<0, 4, K><<<mg_grid(h, g.n_coarse, K / 2, 4), BLOCK, 0, r.st>>>(g.r_rowptr, g.r_col, g.r_val, g.n_coarse, r.w.ctrl, x, y);
    else k_mg_csr<0, 1, K><<<mg_grid(h, g.n_coarse, K / 2), BLOCK, 0, r.st>>>(g.r_rowptr, g.r_col, g.r_val, g.n_coarse, r.w.ctrl, x, y);
    IF_LAUNCH_CHECK();
    return IF_OK;
}
template <int K>
int mg_prolong_add(const Run& r, const MgLevel& g, const double* x, double* y) {
    const if_mesh_s* h = r.h;
    const bool wide_p = g.p_nnz >= IF_MG_WIDE * g.n;
    bool done = false;
    int rc;
    if (!wide_p) {
        RowsArgs a{g.p_rowptr, g.p_col, g.p_val, nullptr, g.n, x, y, nullptr, y, 0.0, 0, 0, 0};
        if ((rc = launch_rows<ROWS_ACC, K>(r, a, g.cap_p, &done))) return rc;
        if (done) return IF_OK;
    }
    if (wide_p) k_mg_csr<1, 4, K><<<mg_grid(h, g.n, K / 2, 4), BLOCK, 0, r.st>>>(g.p_rowptr, g.p_col, g.p_val, g.n, r.w.ctrl, x, y);
    else k_mg_csr<1, 1, K><<<mg_grid(h, g.n, K / 2), BLOCK, 0, r.st>>>(g.p_rowptr, g.p_col, g.p_val, g.n, r.w.ctrl, x, y);
    IF_LAUNCH_CHECK();
    return IF_OK;
}

// Damping of the Jacobi sweeps of a level.  One sweep: omega = min(MG_OMEGA_MAX, 1.6 / rho), rho = max(rho(D_S^-1 S),
// rho(D_M^-1 M)) (mg.cu).  k >= 2 sweeps: the reciprocals of the roots of the Chebyshev polynomial of degree k on
// [rho / 4, rho] -- the same number of passes, but the product of the k factors (1 - omega_j t) is 1 / T_k(5/3) on the
// upper three quarters of the spectrum (0.22, 0.074, 0.025 for k = 2, 3, 4) where k equal sweeps give 0.6^k, and stays
// below 1 in modulus on (0, rho]: the smoother contracts, the cycle stays symmetric positive definite.
inline void mg_omegas(const MgLevel& g, int k, double* om) {
    if (k <= 1) { om[0] = g.omega; return; }
    const double rho = std::max(g.rho, g.rho_m), lo = rho / 4.0;
    const double c = 0.5 * (rho + lo), hw = 0.5 * (rho - lo);
    for (int j = 0; j < k; ++j) om[j] = 1.0 / (c + hw * std::cos(M_PI * (2 * j + 1) / (2.0 * k)));
}
constexpr int MG_MAX_NU = 8;

// Levels >= 1 of a V cycle: e = V_l r.  nu Jacobi sweeps (the first from a zero guess), coarse correction, nu sweeps;
// nu = r.mg_nu[1] on level 1 and r.mg_nu[2] below.  R holds r and is not changed; E, T, E2 are work buffers of the
// level; *result is the one that holds e.
template <int K>
int mg_vcycle(const Run& r, const MgBuffers& b, int l, double* R, double* E, double* T, double* E2, double** result,
              IterTimer* tm) {
    const if_mesh_s* h = r.h;
    const MgLevel& g = h->mg[l];
    MgMat gm = mg_mat(g);
    const Ctrl* ctrl = r.w.ctrl;
    const bool last = l == h->mg_levels - 1;
    int rc;
    if (last && g.n <= MG_COARSEST) {
        k_mg_coarse<K><<<K, 64, 0, r.st>>>(gm, ctrl, b.coarse_inv, R, E);
        IF_LAUNCH_CHECK();
        if (l == 1 && tm && (rc = tm->mark(r.st, MGT_LEVEL1))) return rc;
        *result = E;
        return IF_OK;
    }
    // rows with many entries (coarse levels, restriction) are split over four entry slices
    const bool wide = g.nnz >= IF_MG_WIDE * g.n;
    const int grid1 = mg_grid(h, g.n, K / 2);
    const int grid = mg_grid(h, g.n, K / 2, wide ? 4 : 1);
    // sub 1: out = R - K v ;  sub 2: out = v + omega (R - K v) / d
    auto apply = [&](int sub, double omega, const double* v, double* out) -> int {
        gm.omega = omega;
        if (!wide) {       // the row-block kernel, if a stage for this level's tiles fits
            bool done = false;
            int rcc;
            RowsArgs a{g.rowptr, g.col, g.sm, g.diag, g.n, v, R, v, out, omega, 0, 0, 0};
            if (sub == 1) rcc = launch_rows<ROWS_RES, K>(r, a, g.cap_a, &done);
            else rcc = launch_rows<ROWS_SWEEP, K>(r, a, g.cap_a, &done);
            if (rcc != IF_OK || done) return rcc;
        }
        if (sub == 1) {
            if (wide) k_mg_apply<1, 4, K><<<grid, BLOCK, 0, r.st>>>(gm, ctrl, v, R, out);
            else k_mg_apply<1, 1, K><<<grid, BLOCK, 0, r.st>>>(gm, ctrl, v, R, out);
        } else {
            if (wide) k_mg_apply<2, 4, K><<<grid, BLOCK, 0, r.st>>>(gm, ctrl, v, R, out);
            else k_mg_apply<2, 1, K><<<grid, BLOCK, 0, r.st>>>(gm, ctrl, v, R, out);
        }
        IF_LAUNCH_CHECK();
        return IF_OK;
    };
    // a coarsest level too large for the dense solve (coarsening stalled): smoothing only
    const int nu = std::min(MG_MAX_NU, last ? 4 * r.mg_nu[2] : r.mg_nu[l == 1 ? 1 : 2]);
    double om[MG_MAX_NU];
    mg_omegas(g, nu, om);
    if (nu >= 2 && nu == r.mg_nu[l == 1 ? 1 : 2] && r.order_n == 1)
        for (int j = 0; j < nu; ++j) om[j] = g.omega;      // n = 1: equal sweeps, as tuned
    double* cur = E;
    double* spare[2] = {E2, T};
    gm.omega = om[0];
    k_mg_jacobi0<K><<<grid1, BLOCK, 0, r.st>>>(gm, ctrl, R, cur);
    IF_LAUNCH_CHECK();
    for (int k = 1; k < nu; ++k) {
        if ((rc = apply(2, om[k], cur, spare[0]))) return rc;
        std::swap(cur, spare[0]);
    }
    if (last) {
        if (l == 1 && tm && (rc = tm->mark(r.st, MGT_LEVEL1))) return rc;
        *result = cur;
        return IF_OK;
    }
    if ((rc = apply(1, 0.0, cur, spare[1]))) return rc;                // residual of the level
    double* const* nb = b.lev[l + 1];
    if ((rc = mg_restrict<K>(r, g, spare[1], nb[0]))) return rc;
    if (l == 1 && tm && (rc = tm->mark(r.st, MGT_LEVEL1))) return rc;
    double* ec = nullptr;
    if ((rc = mg_vcycle<K>(r, b, l + 1, nb[0], nb[1], nb[2], nb[3], &ec, tm))) return rc;
    if (l == 1 && tm && (rc = tm->mark(r.st, MGT_COARSE))) return rc;
    if ((rc = mg_prolong_add<K>(r, g, ec, cur))) return rc;
    for (int k = 0; k < nu; ++k) {
        if ((rc = apply(2, om[nu - 1 - k], cur, spare[k & 1]))) return rc;
        std::swap(cur, spare[k & 1]);
    }
    if (l == 1 && tm && (rc = tm->mark(r.st, MGT_LEVEL1))) return rc;
    *result = cur;
    return IF_OK;
}

// Level 0 of one V cycle.  `first` (k_spmm<16, MGR | MGR0>) has done the first sweep from a zero guess on the way:
//   one sweep per side (nu0 = 1): it left t = R - K e in b.t and did not store e = omega R/d -- the prolongation
//       kernel forms it again (unless the prolongator is too wide for that kernel; then e is in b.za);
//   nu0 >= 2: it left the SECOND sweep e2 in b.za; the other sweeps and the residual follow here.
// Then restriction, coarse levels, prolongation, nu0 sweeps, the last one with sub-mode `final_sub` into `out`.
// R is (R0, R1) picked on the device (r_select, see SpmmArgs) or R0.  Work buffers: b.za, b.zb, b.t (and out, which
// is only written by the last sweep).
template <int K>
int mg_cycle_level0(const Run& r, const MgBuffers& b, const double* R0, const double* R1, int r_select, double* out,
                    int final_sub, IterTimer* tm) {
    const if_mesh_s* h = r.h;
    const MgLevel& g = h->mg[0];
    const Ctrl* ctrl = r.w.ctrl;
    const int nu = r.mg_nu[0];
    double om[MG_MAX_NU];
    mg_omegas(g, nu, om);
    int rc;
    auto sweep = [&](int sub, double omega, const double* v, double* dst) -> int {
        SpmmArgs a{v, R0, const_cast<double*>(R1), dst, nullptr, sub, 0, omega, 0.0, r_select};
        return launch_spmm<K, MODE_AX>(r, r.mgg.ax, a);
    };
    double* cur = b.za;
    if (nu >= 2) {
        double* other = b.zb;
        for (int k = 2; k < nu; ++k) {
            if ((rc = sweep(2, om[k], cur, other))) return rc;
            std::swap(cur, other);
        }
        if ((rc = sweep(1, 0.0, cur, b.t))) return rc;                 // residual after the sweeps
        if (tm && (rc = tm->mark(r.st, MGT_LAST))) return rc;
    }
    double* const* nb = b.lev[1];
    if ((rc = mg_restrict<K>(r, g, b.t, nb[0]))) return rc;
    if (tm && (rc = tm->mark(r.st, MGT_RESTRICT0))) return rc;
    double* ec = nullptr;
    if ((rc = mg_vcycle<K>(r, b, 1, nb[0], nb[1], nb[2], nb[3], &ec, tm))) return rc;
    if (nu == 1 && mg_fused_prolongation(g) && !r.vec) {    // e = omega R/d formed again here: it has not been stored
        bool done = false;
        RowsArgs a{g.p_rowptr, g.p_col, g.p_val, g.diag, g.n, ec, R0, R1, cur, g.omega, r_select, 0, 0};
        if ((rc = launch_rows<ROWS_PROLONG0, K>(r, a, g.cap_p, &done))) return rc;
        if (!done) {
            k_mg_prolong0<K><<<mg_grid(h, g.n, K / 2), BLOCK, 0, r.st>>>(g.p_rowptr, g.p_col, g.p_val, mg_mat(g), ctrl, ec, R0, R1, r_select, cur);
            IF_LAUNCH_CHECK();
        }
    } else if ((rc = mg_prolong_add<K>(r, g, ec, cur))) {
        return rc;
    }
    if (tm && (rc = tm->mark(r.st, MGT_PROLONG0))) return rc;
    // sweeps after the correction, dampings in reverse order (the cycle is symmetric); scratch: za, zb, t minus `out`
    for (int k = 0; k < nu - 1; ++k) {
        double* dst = nullptr;
        for (double* cand : {b.za, b.t, b.zb})
            if (cand != cur && cand != out) { dst = cand; break; }
        if ((rc = sweep(2, om[nu - 1 - k], cur, dst))) return rc;
        cur = dst;
    }
    if ((rc = sweep(final_sub, om[0], cur, out))) return rc;
    if (tm && (rc = tm->mark(r.st, MGT_LAST))) return rc;
    return IF_OK;
}

// ONE iteration of multigrid-preconditioned CG for the 16 columns (see the head of this file); every pointer that
// alternates between iterations is picked on the device, so the sequence is the same every time (CUDA graph).
template <int K>
int mg_enqueue_iteration(const Run& r, IterTimer* tm) {
    const if_mesh_s* h = r.h;
    const MgBuffers b = mg_buffers(r);
    const int nu = r.mg_nu[0];
    double om[MG_MAX_NU];
    mg_omegas(h->mg[0], nu, om);
    // what the fused first-sweep kernel leaves behind (see mg_cycle_level0)
    // (vector filter: the first sweep divides by the diagonal of D~, which the prolongation kernel does not have: stored)
    double* e_store = (nu == 1 && (r.vec || !mg_fused_prolongation(h->mg[0]))) ? b.za : nullptr;
    double* first_out = nu >= 2 ? b.za : b.t;
    const double omega2 = nu >= 2 ? om[1] : 0.0;
    int rc;
    if (tm && (rc = tm->mark(r.st, -1))) return rc;
    if (r.order_n == 1) {
        SpmmArgs a{b.zb, b.p[0], b.x, b.q, b.p[1], 0, 1, 0.0, 0.0, 0};          // kernel A of the Jacobi path
        if ((rc = launch_spmm<K, MODE_CG1>(r, r.g.cga, a))) return rc;
    } else {
        SpmmArgs a{b.zb, b.p[0], b.x, b.t, b.p[1], 0, 1, 0.0, 0.0, 0};
        if ((rc = launch_spmm<K, MODE_CG2A>(r, r.g.cga, a))) return rc;
        SpmmArgs c{b.t, b.p[0], nullptr, b.q, b.p[1], 0, 1, 0.0, 0.0, 0};
        if ((rc = launch_spmm<K, MODE_CG2B>(r, r.g.cgb, c))) return rc;
    }
    if (tm && (rc = tm->mark(r.st, MGT_A))) return rc;
    {
        SpmmArgs a{b.r[0], b.q, b.r[1], first_out, e_store, 0, 0, om[0], omega2, 1};
        if ((rc = launch_spmm<K, MODE_MGR>(r, r.mgg.mgr, a))) return rc;
    }
    if (tm && (rc = tm->mark(r.st, MGT_MGR))) return rc;
    if (r.order_n == 1) return mg_cycle_level0<K>(r, b, b.r[0], b.r[1], 1, b.zb, 3, tm);
    // n = 2: y = V r', w = M y (into q, dead by now), bookkeeping with rho' = y.w; then z = V w
    if ((rc = mg_cycle_level0<K>(r, b, b.r[0], b.r[1], 1, b.q, 5, tm))) return rc;
    {
        SpmmArgs a{b.q, nullptr, nullptr, first_out, e_store, 0, 0, om[0], omega2, 0};
        if ((rc = launch_spmm<K, MODE_MGR0>(r, r.mgg.mgr0, a))) return rc;
    }
    if (tm && (rc = tm->mark(r.st, MGT_MGR))) return rc;
    return mg_cycle_level0<K>(r, b, b.q, nullptr, 0, b.zb, 2, tm);
}

}  // namespace
}  // namespace ifl
