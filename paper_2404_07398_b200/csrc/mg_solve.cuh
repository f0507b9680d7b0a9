// Multigrid-preconditioned CG for the n = 1 systems at large scales (included by solve.cu).
//
//   PCG on (M + c S) x = M phi, x0 = phi, preconditioner B = one V cycle of the smoothed-
//   aggregation hierarchy of mg.cu with damped Jacobi smoothing (one sweep on the mesh, MG_NU_L1 on level 1,
//   MG_NU_COARSE on the coarser levels) and a dense Cholesky solve on the coarsest level.
//   B is symmetric positive definite and fixed per column, so plain PCG applies.  16 columns at a time, every
//   column with its own c, alpha, beta and stop time.  As in the Jacobi path all CG scalars live in the device
//   control block: the iteration is
//       k_spmm<16, CG1>      p' = z + beta p ; x += alpha p ; q = A p' ; alpha' = rho / p'.q         (kernel A)
//       k_spmm<16, MGR>      r' = r - alpha' q ; e = omega r'/d ; t = r' - A e     (residual update, first sweep of B
//                            on level 0 and its residual in one pass), then restriction, coarse levels, prolongation
//       k_spmm<16, AX> sub 3 z = last sweep ; rho' = r.z ; ||r||^2 ; beta ; stop test        (CG bookkeeping)
//   and the host reads the control block once per iteration to see whether every column has stopped.
// The stop test is the same as in the Jacobi path: recursive ||r||_2 <= tol ||M phi||_2.
#pragma once

namespace ifl {
namespace {

constexpr int MGK = 16;               // columns of the multigrid path
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

struct MgCols {                       // per-column scalars, passed by value
    double c[MGK];
    double a[MGK];
    double b[MGK];
};

struct MgMat {                        // one level's (S, M) pair
    const int64_t* __restrict__ rowptr;
    const int32_t* __restrict__ col;
    const double2* __restrict__ sm;
    const double2* __restrict__ diag;
    int64_t n;
    double omega;                     // Jacobi damping of the smoother on this level
};

// A row is handled by 8 * SL threads: column pair l = tid % 8, entry slice sl = (tid / 8) % SL.  SL = 1 for the
// short rows of the fine levels; SL = 4 (one row per warp, slices added with two shuffles) for the coarse levels
// whose rows have hundreds of entries and would otherwise be walked serially.
// MODE 0: y = A x ;  MODE 1: y = r - A x ;  MODE 2: y = x + omega (r - A x) / d        with A = M + c S per column
template <int MODE, int SL>
__global__ void __launch_bounds__(BLOCK, IF_MG_MINB) k_mg_apply(MgMat g, MgCols cs, const double* __restrict__ x,
                                                    const double* __restrict__ r, double* __restrict__ y) {
    constexpr int WPB = BLOCK / (8 * SL);
    const int l = threadIdx.x % 8, sl = (threadIdx.x / 8) % SL;
    const double2 cc = {cs.c[2 * l], cs.c[2 * l + 1]};
    // (rows are padded to whole warps by the loop bound: every lane of a warp takes part in the shuffles)
    // a block walks a contiguous range of rows, WPB at a time: neighbouring rows gather the same rows of x, which
    // the L1 then serves (a grid-stride assignment sends every gather to the L2)
    const int64_t per_block = ((g.n + gridDim.x - 1) / gridDim.x + WPB - 1) / WPB * WPB;
    const int64_t row_end = min((int64_t)(blockIdx.x + 1) * per_block, (g.n + 3) / 4 * 4);
    for (int64_t row = (int64_t)blockIdx.x * per_block + threadIdx.x / (8 * SL); row < row_end; row += WPB) {
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
            for (int j = 0; j < MG_UB; ++j) v[j] = ld2(x, (int64_t)cj[j] * MGK + 2 * l);
#pragma unroll
            for (int j = 0; j < MG_UB; ++j)
                if (k + j * SL < k1) {
                    s.x = fma(fma(cc.x, w[j].x, w[j].y), v[j].x, s.x);
                    s.y = fma(fma(cc.y, w[j].x, w[j].y), v[j].y, s.y);
                }
        }
        if (SL >= 2) { s.x += __shfl_xor_sync(0xffffffffu, s.x, 8);  s.y += __shfl_xor_sync(0xffffffffu, s.y, 8); }
        if (SL >= 4) { s.x += __shfl_xor_sync(0xffffffffu, s.x, 16); s.y += __shfl_xor_sync(0xffffffffu, s.y, 16); }
        if (sl != 0 || !live) continue;
        const int64_t ri = row * MGK + 2 * l;
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
__global__ void __launch_bounds__(BLOCK) k_mg_jacobi0(MgMat g, MgCols cs, const double* __restrict__ r,
                                                      double* __restrict__ e) {
    constexpr int TPR = MGK / 2;
    constexpr int ROWS = BLOCK / TPR;
    const int l = threadIdx.x % TPR;
    const double2 cc = {cs.c[2 * l], cs.c[2 * l + 1]};
    for (int64_t row = (int64_t)blockIdx.x * ROWS + threadIdx.x / TPR; row < g.n; row += (int64_t)gridDim.x * ROWS) {
        const int64_t ri = row * MGK + 2 * l;
        const double2 d = g.diag[row];
        const double2 rv = ld2(r, ri);
        st2(e, ri, make_double2(g.omega * rv.x / fma(cc.x, d.x, d.y), g.omega * rv.y / fma(cc.y, d.x, d.y)));
    }
}

// y (+)= B x for a scalar CSR matrix (restriction R, prolongation P); thread mapping as above
template <int ACC, int SL>
__global__ void __launch_bounds__(BLOCK, IF_MG_MINB) k_mg_csr(const int64_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                                                  const double* __restrict__ val, int64_t n,
                                                  const double* __restrict__ x, double* __restrict__ y) {
    constexpr int WPB = BLOCK / (8 * SL);
    const int l = threadIdx.x % 8, sl = (threadIdx.x / 8) % SL;
    const int64_t per_block = ((n + gridDim.x - 1) / gridDim.x + WPB - 1) / WPB * WPB;   // contiguous rows per block
    const int64_t row_end = min((int64_t)(blockIdx.x + 1) * per_block, (n + 3) / 4 * 4);
    for (int64_t row = (int64_t)blockIdx.x * per_block + threadIdx.x / (8 * SL); row < row_end; row += WPB) {
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
            for (int j = 0; j < MG_UB; ++j) v[j] = ld2(x, (int64_t)cj[j] * MGK + 2 * l);
#pragma unroll
            for (int j = 0; j < MG_UB; ++j)
                if (k + j * SL < k1) {
                    s.x = fma(w[j], v[j].x, s.x);
                    s.y = fma(w[j], v[j].y, s.y);
                }
        }
        if (SL >= 2) { s.x += __shfl_xor_sync(0xffffffffu, s.x, 8);  s.y += __shfl_xor_sync(0xffffffffu, s.y, 8); }
        if (SL >= 4) { s.x += __shfl_xor_sync(0xffffffffu, s.x, 16); s.y += __shfl_xor_sync(0xffffffffu, s.y, 16); }
        if (sl != 0 || !live) continue;
        const int64_t ri = row * MGK + 2 * l;
        if (ACC) { const double2 o = ld2(y, ri); s.x += o.x; s.y += o.y; }
        st2(y, ri, s);
    }
}

// Prolongation onto the mesh fused with the first sweep:  e = omega r / d + P e_c  (8 threads per row as above; the
// prolongator has 2.6 entries per row).  k_spmm<16, MGR> then does not store its e = omega r'/d, and this kernel
// reads r' where k_mg_csr<1, 1> would read e back: one pass over a [V][16] vector less per iteration.
__global__ void __launch_bounds__(BLOCK, IF_MG_MINB) k_mg_prolong0(const int64_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                                                       const double* __restrict__ val, MgMat g, MgCols cs,
                                                       const double* __restrict__ x, const double* __restrict__ r,
                                                       double* __restrict__ y) {
    constexpr int WPB = BLOCK / 8;
    const int l = threadIdx.x % 8;
    const double2 cc = {cs.c[2 * l], cs.c[2 * l + 1]};
    const int64_t n = g.n;
    const int64_t per_block = ((n + gridDim.x - 1) / gridDim.x + WPB - 1) / WPB * WPB;   // contiguous rows per block
    const int64_t row_end = min((int64_t)(blockIdx.x + 1) * per_block, n);
    for (int64_t row = (int64_t)blockIdx.x * per_block + threadIdx.x / 8; row < row_end; row += WPB) {
        const int64_t ri = row * MGK + 2 * l;
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
            for (int j = 0; j < MG_UB; ++j) v[j] = ld2(x, (int64_t)cj[j] * MGK + 2 * l);
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

// coarsest level: dense Cholesky of A = M + c S per column (one block per column), then the two triangular solves
__global__ void __launch_bounds__(64) k_mg_coarse(MgMat g, MgCols cs, const double* __restrict__ r, double* __restrict__ e) {
    __shared__ double a[MG_COARSEST][MG_COARSEST + 1];
    __shared__ double v[MG_COARSEST];
    const int c = blockIdx.x, t = threadIdx.x, n = (int)g.n;
    const double cc = cs.c[c];
    for (int i = t; i < n; i += 64) {
        for (int j = 0; j < n; ++j) a[i][j] = 0.0;
        v[i] = r[(int64_t)i * MGK + c];
    }
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
    if (t == 0) {                                 // L y = v ; L^T x = y  (n <= 64: one thread is enough)
        for (int i = 0; i < n; ++i) {
            double s = v[i];
            for (int j = 0; j < i; ++j) s -= a[i][j] * v[j];
            v[i] = s / a[i][i];
        }
        for (int i = n - 1; i >= 0; --i) {
            double s = v[i];
            for (int j = i + 1; j < n; ++j) s -= a[j][i] * v[j];
            v[i] = s / a[i][i];
        }
    }
    __syncthreads();
    for (int i = t; i < n; i += 64) e[(int64_t)i * MGK + c] = v[i];
}

// ---- PCG vector kernels on [row][16]
// out = area * x
__global__ void __launch_bounds__(BLOCK) k_mg_mass(const double* __restrict__ area, int64_t n, const double* __restrict__ x,
                                                   double* __restrict__ out) {
    constexpr int TPR = MGK / 2;
    const int64_t i = (int64_t)blockIdx.x * BLOCK + threadIdx.x;
    if (i >= n * TPR) return;
    const double av = area[i / TPR];
    const double2 xv = ld2(x, 2 * i);
    st2(out, 2 * i, make_double2(av * xv.x, av * xv.y));
}
// per-block partial sums of a.b and a.c per column (fixed order); k_mg_dot_final adds the blocks in order
__global__ void __launch_bounds__(BLOCK) k_mg_dot(int64_t n, const double* __restrict__ a, const double* __restrict__ b,
                                                  const double* __restrict__ c, double* __restrict__ partials) {
    constexpr int TPR = MGK / 2;
    constexpr int ROWS = BLOCK / TPR;
    __shared__ double2 red[2][BLOCK];
    const int tid = threadIdx.x, l = tid % TPR;
    double2 s0 = {0.0, 0.0}, s1 = {0.0, 0.0};
    for (int64_t row = (int64_t)blockIdx.x * ROWS + tid / TPR; row < n; row += (int64_t)gridDim.x * ROWS) {
        const int64_t ri = row * MGK + 2 * l;
        const double2 av = ld2(a, ri), bv = ld2(b, ri), cv = ld2(c, ri);
        s0.x = fma(av.x, bv.x, s0.x); s0.y = fma(av.y, bv.y, s0.y);
        s1.x = fma(av.x, cv.x, s1.x); s1.y = fma(av.y, cv.y, s1.y);
    }
    red[0][tid] = s0;
    red[1][tid] = s1;
    __syncthreads();
    if (tid < 2 * TPR) {
        const int j = tid / TPR, ll = tid % TPR;
        double2 s = red[j][ll];
        for (int i = ll + TPR; i < BLOCK; i += TPR) { s.x += red[j][i].x; s.y += red[j][i].y; }
        partials[((size_t)blockIdx.x * 2 + j) * MGK + 2 * ll] = s.x;
        partials[((size_t)blockIdx.x * 2 + j) * MGK + 2 * ll + 1] = s.y;
    }
}
__global__ void k_mg_dot_final(const double* __restrict__ partials, int nblocks, double* __restrict__ out) {
    const int t = threadIdx.x;   // 2 * MGK threads
    if (t >= 2 * MGK) return;
    double s = 0.0;
    for (int b = 0; b < nblocks; ++b) s += partials[(size_t)b * 2 * MGK + t];
    out[t] = s;
}

// ------------------------------------------------------------------------------------------- host side
struct MgBuffers {
    double *x, *r[2], *p[2], *q, *za, *zb, *t;  // level 0, [n][16]; r is double-buffered (k_spmm<16, MGR>)
    double* lev[MG_MAX_LEVELS][4];              // levels >= 1: R, E, T, E2
    double* partials;                           // [grid][2][16]
    double* dots;                               // [32]
    int dot_grid;
    int ax_grid;                                // persistent grid of k_spmm<16, MODE_AX> (level-0 operator)
};

inline size_t mg_extra_bytes(const if_mesh_s* h) {
    if (h->mg_levels < 2) return 0;
    size_t b = 4 * align_up((size_t)h->n_vert * MGK * sizeof(double));        // za, zb, t, second r (level-0 vectors 6 to 9)
    for (int l = 1; l < h->mg_levels; ++l) b += 4 * align_up((size_t)h->mg[l].n * MGK * sizeof(double));
    b += align_up((size_t)h->n_sm * 4 * 2 * MGK * sizeof(double)) + align_up(2 * MGK * sizeof(double));
    return b;
}

inline MgBuffers mg_layout(const if_mesh_s* h, const Workspace& w, void* extra) {
    MgBuffers m{};
    m.x = w.x; m.r[0] = w.z; m.p[0] = w.p0; m.p[1] = w.p1; m.q = w.q;
    char* p = static_cast<char*>(extra);
    size_t off = 0;
    auto take = [&](size_t bytes) { void* r = p + off; off += align_up(bytes); return r; };
    m.za = (double*)take((size_t)h->n_vert * MGK * sizeof(double));
    m.zb = (double*)take((size_t)h->n_vert * MGK * sizeof(double));
    m.t = (double*)take((size_t)h->n_vert * MGK * sizeof(double));
    m.r[1] = (double*)take((size_t)h->n_vert * MGK * sizeof(double));
    for (int l = 1; l < h->mg_levels; ++l)
        for (int k = 0; k < 4; ++k) m.lev[l][k] = (double*)take((size_t)h->mg[l].n * MGK * sizeof(double));
    m.dot_grid = h->n_sm * 4;
    m.partials = (double*)take((size_t)m.dot_grid * 2 * MGK * sizeof(double));
    m.dots = (double*)take(2 * MGK * sizeof(double));
    return m;
}

// level 0: the prolongation kernel can form e = omega r'/d itself (short prolongator rows only)
inline bool mg_fused_prolongation(const MgLevel& g) { return g.p_nnz < IF_MG_WIDE * g.n; }
inline MgMat mg_mat(const MgLevel& g) { return MgMat{g.rowptr, g.col, g.sm, g.diag, g.n, g.omega}; }
inline int mg_grid(const if_mesh_s* h, int64_t n, int sl = 1) {
    const int64_t rows = BLOCK / (8 * sl);
    return (int)std::max<int64_t>(1, std::min<int64_t>((n + rows - 1) / rows, (int64_t)h->n_sm * IF_MG_BPS));
}

// One V cycle on level l: e = B_l r.  nu Jacobi sweeps (the first from a zero guess), coarse correction, nu sweeps;
// nu = 1 on level 0, MG_NU_L1 on level 1 and MG_NU_COARSE below.  R holds r and is not changed; E, T, E2 are work buffers of the
// level; *result is the one that holds e.
// On level 0 the caller may have done the first sweep and its residual already (first_done: E = omega r / d,
// T = r - A E, both by k_spmm<16, MGR>) and chooses the sub-mode of the last sweep (final_sub 3 / 4: with the CG
// bookkeeping, see kernels.cuh).
int mg_vcycle(const Run& r, const MgBuffers& b, const MgCols& cs, int l, double* R, double* E, double* T, double* E2,
              double** result, int final_sub = 2, bool first_done = false) {
    const if_mesh_s* h = r.h;
    const MgLevel& g = h->mg[l];
    const MgMat gm = mg_mat(g);
    const bool last = l == h->mg_levels - 1;
    if (last && g.n <= MG_COARSEST) {
        k_mg_coarse<<<MGK, 64, 0, r.st>>>(gm, cs, R, E);
        IF_LAUNCH_CHECK();
        *result = E;
        return IF_OK;
    }
    // rows with many entries (coarse levels, restriction) are split over four entry slices
    const bool wide = g.nnz >= IF_MG_WIDE * g.n;
    const int grid1 = mg_grid(h, g.n);
    const int grid = mg_grid(h, g.n, wide ? 4 : 1);
    // sub 1: out = rr - A v ;  sub 2: out = v + omega (rr - A v) / d      (level 0: the tiled TMA kernel)
    auto apply = [&](int sub, const double* v, double* out) -> int {
        if (l == 0) {
            SpmmArgs a{v, R, nullptr, out, nullptr, sub, 0, g.omega};
            return launch_spmm<MGK, MODE_AX>(r, b.ax_grid, a);
        }
        if (sub == 1) {
            if (wide) k_mg_apply<1, 4><<<grid, BLOCK, 0, r.st>>>(gm, cs, v, R, out);
            else k_mg_apply<1, 1><<<grid, BLOCK, 0, r.st>>>(gm, cs, v, R, out);
        } else {
            if (wide) k_mg_apply<2, 4><<<grid, BLOCK, 0, r.st>>>(gm, cs, v, R, out);
            else k_mg_apply<2, 1><<<grid, BLOCK, 0, r.st>>>(gm, cs, v, R, out);
        }
        IF_LAUNCH_CHECK();
        return IF_OK;
    };
    // a coarsest level too large for the dense solve (coarsening stalled): smoothing only
    const int nu = last ? 4 * MG_NU_COARSE : (l == 0 ? 1 : (l == 1 ? MG_NU_L1 : MG_NU_COARSE));
    int rc;
    double* cur = E;
    double* spare[2] = {E2, T};
    if (!(l == 0 && first_done)) {
        k_mg_jacobi0<<<grid1, BLOCK, 0, r.st>>>(gm, cs, R, cur);
        IF_LAUNCH_CHECK();
    }
    for (int k = 1; k < nu; ++k) {
        if ((rc = apply(2, cur, spare[0]))) return rc;
        std::swap(cur, spare[0]);
    }
    if (last) { *result = cur; return IF_OK; }
    if (!(l == 0 && first_done && nu == 1))
        if ((rc = apply(1, cur, spare[1]))) return rc;                // residual of the level
    double* const* nb = b.lev[l + 1];
    const bool wide_r = g.p_nnz >= IF_MG_WIDE * g.n_coarse, wide_p = g.p_nnz >= IF_MG_WIDE * g.n;
    if (wide_r) k_mg_csr<0, 4><<<mg_grid(h, g.n_coarse, 4), BLOCK, 0, r.st>>>(g.r_rowptr, g.r_col, g.r_val, g.n_coarse, spare[1], nb[0]);
    else k_mg_csr<0, 1><<<mg_grid(h, g.n_coarse), BLOCK, 0, r.st>>>(g.r_rowptr, g.r_col, g.r_val, g.n_coarse, spare[1], nb[0]);
    IF_LAUNCH_CHECK();
    double* ec = nullptr;
    if ((rc = mg_vcycle(r, b, cs, l + 1, nb[0], nb[1], nb[2], nb[3], &ec))) return rc;
    if (l == 0 && first_done && nu == 1 && mg_fused_prolongation(g))   // cur = omega R / d has not been stored
        k_mg_prolong0<<<grid1, BLOCK, 0, r.st>>>(g.p_rowptr, g.p_col, g.p_val, gm, cs, ec, R, cur);
    else if (wide_p) k_mg_csr<1, 4><<<mg_grid(h, g.n, 4), BLOCK, 0, r.st>>>(g.p_rowptr, g.p_col, g.p_val, g.n, ec, cur);
    else k_mg_csr<1, 1><<<grid1, BLOCK, 0, r.st>>>(g.p_rowptr, g.p_col, g.p_val, g.n, ec, cur);
    IF_LAUNCH_CHECK();
    for (int k = 0; k < nu; ++k) {
        if ((rc = apply((l == 0 && k == nu - 1) ? final_sub : 2, cur, spare[k & 1]))) return rc;
        std::swap(cur, spare[k & 1]);
    }
    *result = cur;
    return IF_OK;
}

// host copies of (a.b, a.c) per column
int mg_dots(const Run& r, const MgBuffers& b, const double* a, const double* bb, const double* cc, double* h_out /*[32] pinned*/) {
    k_mg_dot<<<b.dot_grid, BLOCK, 0, r.st>>>(r.h->n_vert, a, bb, cc, b.partials);
    IF_LAUNCH_CHECK();
    k_mg_dot_final<<<1, 2 * MGK, 0, r.st>>>(b.partials, b.dot_grid, b.dots);
    IF_LAUNCH_CHECK();
    IF_CUDA_TRY(cudaMemcpyAsync(h_out, b.dots, 2 * MGK * sizeof(double), cudaMemcpyDeviceToHost, r.st));
    IF_CUDA_TRY(cudaStreamSynchronize(r.st));
    return IF_OK;
}

// Up to 16 right-hand sides rhs[first .. first+count) by multigrid-preconditioned CG; results are finalised like in
// the Jacobi path (energy or scatter, per-RHS stats).
int mg_solve_batch(Run& r, Job job, const double* d_fields, const std::vector<Rhs>& rhs, size_t first, size_t count,
                   int n_ells, double* d_out, void* mg_extra, double* h_dots /*pinned [32]*/, int64_t* iters_total) {
    const if_mesh_s* h = r.h;
    const int64_t nv = h->n_vert;
    int rc;
    MgBuffers b = mg_layout(h, r.w, mg_extra);
    Ctrl hc = fresh_ctrl(r);
    StartParams sp;
    MgCols cs;
    memset(&sp, 0, sizeof(sp));
    memset(&cs, 0, sizeof(cs));
    for (int c = 0; c < KMAX; ++c) sp.field[c] = -1;
    for (size_t i = 0; i < count; ++i) {
        const Rhs& q = rhs[first + i];
        cs.c[i] = sp.c[i] = hc.c[i] = r.opt.gamma * q.ell * q.ell;
        sp.field[i] = hc.field[i] = q.f;
        sp.rhs[i] = hc.rhs[i] = q.f * n_ells + q.j;
    }
    const int64_t tiles = (nv + TILE_ROWS - 1) / TILE_ROWS;
    int cg_grid = 0;
    if ((rc = resident_grid(k_spmm<MGK, MODE_AX>, TileSmem<MGK, MODE_AX>::bytes, h->n_sm, tiles, &b.ax_grid,
                            SpmmCfg<MGK>::NT))) return rc;
    if ((rc = resident_grid(k_spmm<MGK, MODE_CG1>, TileSmem<MGK, MODE_CG1>::bytes, h->n_sm, tiles, &cg_grid,
                            SpmmCfg<MGK>::NT))) return rc;
    hc.all_done = 0;   // k_spmm reads c from the control block and returns at once when all_done is set
    IF_CUDA_TRY(cudaMemcpyAsync(r.w.ctrl, &hc, sizeof(Ctrl), cudaMemcpyHostToDevice, r.st));
    const unsigned eg = (unsigned)((nv * MGK + BLOCK - 1) / BLOCK);
    const unsigned vg = (unsigned)((nv * (MGK / 2) + BLOCK - 1) / BLOCK);
    const MgMat g0 = mg_mat(h->mg[0]);
    k_ingest<MGK><<<eg, BLOCK, 0, r.st>>>(r.m, sp, 0xffffu, d_fields, b.x);
    IF_LAUNCH_CHECK();
    k_mg_mass<<<vg, BLOCK, 0, r.st>>>(h->area, nv, b.x, b.za);               // b = M phi
    IF_LAUNCH_CHECK();
    int mgr_grid = 0;
    if ((rc = resident_grid(k_spmm<MGK, MODE_MGR>, TileSmem<MGK, MODE_MGR>::bytes, h->n_sm, tiles, &mgr_grid,
                            SpmmCfg<MGK>::NT))) return rc;
    {
        SpmmArgs a{b.x, b.za, nullptr, b.r[0], nullptr, 1, 0, 0.0};           // r = b - A x0
        if ((rc = launch_spmm<MGK, MODE_AX>(r, b.ax_grid, a))) return rc;
    }
    IF_CUDA_TRY(cudaMemsetAsync(b.p[0], 0, (size_t)nv * MGK * sizeof(double), r.st));
    IF_CUDA_TRY(cudaMemsetAsync(b.p[1], 0, (size_t)nv * MGK * sizeof(double), r.st));
    if ((rc = mg_dots(r, b, b.za, b.za, b.za, h_dots))) return rc;            // ||M phi||^2 (host sync)
    // the control block of the batch: unused columns stay done, the others start with rho, beta set by the first
    // preconditioner application (sub-mode 4)
    for (int c = 0; c < MGK; ++c) {
        hc.bb[c] = h_dots[c];
        hc.done[c] = (size_t)c < count ? 0 : 1;
    }
    IF_CUDA_TRY(cudaMemcpyAsync(r.w.ctrl, &hc, sizeof(Ctrl), cudaMemcpyHostToDevice, r.st));
    double* z = nullptr;
    if ((rc = mg_vcycle(r, b, cs, 0, b.r[0], b.za, b.t, b.zb, &z, 4, false))) return rc;
    int* h_flag = reinterpret_cast<int*>(h_dots);
    auto all_done = [&](bool* out) -> int {
        IF_CUDA_TRY(cudaMemcpyAsync(h_flag, &r.w.ctrl->all_done, sizeof(int), cudaMemcpyDeviceToHost, r.st));
        IF_CUDA_TRY(cudaStreamSynchronize(r.st));
        *out = *h_flag != 0;
        return IF_OK;
    };
    bool stop = false;
    if ((rc = all_done(&stop))) return rc;
    int64_t loops = 0;
    int cr = 0;
    while (!stop) {
        {
            SpmmArgs a{z, b.p[0], b.x, b.q, b.p[1], 0, 1, 0.0};  // kernel A of the Jacobi path
            if ((rc = launch_spmm<MGK, MODE_CG1>(r, cg_grid, a))) return rc;
        }
        {
            SpmmArgs a{b.r[cr], b.q, b.r[cr ^ 1], b.t, mg_fused_prolongation(h->mg[0]) ? nullptr : b.za, 0, 0, g0.omega};
            if ((rc = launch_spmm<MGK, MODE_MGR>(r, mgr_grid, a))) return rc;
        }
        cr ^= 1;
        if ((rc = mg_vcycle(r, b, cs, 0, b.r[cr], b.za, b.t, b.zb, &z, 3, true))) return rc;
        ++loops;
        if ((rc = all_done(&stop))) return rc;
    }
    *iters_total += loops;
    if (getenv("IF_VERBOSE"))
        fprintf(stderr, "[implicit_filter] multigrid batch: largest scale %.4g, %zu columns, %lld iterations\n",
                rhs[first].ell, count, (long long)loops);
    // the columns are finalised from the device control block (pending alpha p included, as in the Jacobi path)
    Run fr = r;
    fr.w.x = b.x;
    fr.g.stream = (int)std::max<int64_t>(1, std::min<int64_t>((nv + 31) / 32, (int64_t)h->n_sm * 4));
    if ((rc = finalize_columns<MGK>(fr, job, (count >= 16 ? 0xffffu : ((1u << count) - 1u)), d_out, d_fields))) return rc;
    IF_CUDA_TRY(cudaStreamSynchronize(r.st));   // hc lives on this stack frame
    return IF_OK;
}

}  // namespace
}  // namespace ifl
