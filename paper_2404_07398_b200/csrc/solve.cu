// Solving phase: batched multi-right-hand-side Jacobi-PCG on
//     A_c x_c = M phi_c,   A_c = M + c_c S (M^-1 S)^(n-1),   c_c = gamma l_c^(2n)
// for K = 4, 8 or 16 columns c at once, every column with its own scale l_c, field, alpha, beta and stop time.
//
// Layout: work vectors are [row][K] fp64 (K = 16: one 128-byte line per row), rows in the internal order.
// A row is handled by K/2 threads, each owning two adjacent columns (double2 = 16-byte loads/stores), so a warp
// covers 64/K rows and every gather of a neighbour row is one contiguous K*8-byte segment.
//
// CG is carried in the preconditioned residual z = r/d (d = diag(A_c), Jacobi):
//   kernel A (k_spmm, fused):  p' = z + beta p ;  x += alpha_prev p ;  q = A_c p' ;  partial p'.q
//                              the gather recomputes p'_j = z_j + beta p_j at the neighbours, p is double-buffered
//   kernel B (k_update):       z -= alpha q/d ;  partial rho' = sum d z^2 = r.z  and  ||r||^2 = sum (d z)^2
// Per-column scalars (alpha, beta, rho, done flags) live in a device control block and are produced by the
// last block to finish each kernel (single-pass, fixed-order, deterministic grid reduction); the host only polls
// one flag every `check_every` iterations, one CUDA graph launch behind.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <vector>

#include "common.cuh"

namespace ifl {
namespace {

constexpr int KMAX = 16;
constexpr int BLOCK = 256;
constexpr int MAX_RHS = 65536;

struct MeshView {
    const int64_t* __restrict__ chunk_ptr;
    const int32_t* __restrict__ col;
    const double* __restrict__ val;
    const double* __restrict__ area;
    const double* __restrict__ inv_area;
    const double* __restrict__ sdiag;
    const double* __restrict__ gdiag;
    const int32_t* __restrict__ perm;
    int64_t nv;
    int log2c;
};

struct Ctrl {
    double c[KMAX];       // gamma l^(2n)
    double alpha[KMAX];
    double beta[KMAX];
    double rho[KMAX];
    double bb[KMAX];      // ||M phi||^2
    double rr[KMAX];      // ||r||^2 (recursive)
    int field[KMAX];      // field of the column, -1 = unused column
    int rhs[KMAX];        // f * n_ells + j of the column
    int done[KMAX];
    int status[KMAX];
    int iters[KMAX];
    int all_done;
    int cur_p;            // which direction buffer the last kernel A wrote
    int max_iter;
    int pad_;
    double tol2;
    unsigned int ticket[4];
};

enum Mode { MODE_PLAIN = 0, MODE_CG1 = 1, MODE_CG2A = 2, MODE_CG2B = 3 };

__device__ __forceinline__ double2 ld2(const double* __restrict__ p, int64_t i) {
    return *reinterpret_cast<const double2*>(p + i);
}
__device__ __forceinline__ void st2(double* __restrict__ p, int64_t i, double2 v) {
    *reinterpret_cast<double2*>(p + i) = v;
}

// Fixed-order block reduction of NV double2 accumulators per thread over the threads owning the same column
// pair, then a ticket: the last block to arrive sums all blocks' partials in block order.
// Returns true in the last block, with the totals of value set j, column c in tot[j*KMAX + c] (shared memory).
template <int K, int NV>
__device__ __forceinline__ bool grid_reduce(const double2 (&acc)[NV], double* __restrict__ partials,
                                            unsigned int* ticket, double* tot /* shared [NV*KMAX] */) {
    constexpr int TPR = K / 2;
    __shared__ double2 red[BLOCK];
    __shared__ bool is_last;
    const int tid = threadIdx.x;
    for (int j = 0; j < NV; ++j) {
        red[tid] = acc[j];
        __syncthreads();
        if (tid < TPR) {
            double2 s = red[tid];
            for (int i = tid + TPR; i < BLOCK; i += TPR) { s.x += red[i].x; s.y += red[i].y; }
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
    double* redd = reinterpret_cast<double*>(red);   // [BLOCK] doubles (uses half of red)
    constexpr int LANES = BLOCK / K;                  // threads per column
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

struct SpmmArgs {
    const double* in0;   // PLAIN: x        CG1/CG2A: z        CG2B: t
    const double* in1;   //                 CG1/CG2A: p_old    CG2B: p (current)
    double* x;           //                 CG1/CG2A: x (in place)
    double* out0;        // PLAIN: y        CG1: q             CG2A: t            CG2B: q
    double* out1;        //                 CG1/CG2A: p_new
    int scale_inv_area;  // PLAIN: multiply the row result by 1/A_v
    int out_idx;         // CG1/CG2A: index of the direction buffer written (recorded in ctrl->cur_p)
};

template <int K, int MODE>
__global__ void __launch_bounds__(BLOCK) k_spmm(MeshView m, Ctrl* __restrict__ ctrl, double* __restrict__ partials,
                                                SpmmArgs a, int64_t rows_per_block) {
    constexpr int TPR = K / 2;
    constexpr int ROWS = BLOCK / TPR;
    if (MODE != MODE_PLAIN && ctrl->all_done) return;
    const int tid = threadIdx.x;
    const int l = tid % TPR;
    const int64_t r0 = (int64_t)blockIdx.x * rows_per_block;
    const int64_t r1 = min(r0 + rows_per_block, m.nv);
    double2 beta = {0.0, 0.0}, alpha = {0.0, 0.0}, cc = {0.0, 0.0};
    if (MODE != MODE_PLAIN) {
        beta = ld2(ctrl->beta, 2 * l);
        alpha = ld2(ctrl->alpha, 2 * l);
        cc = ld2(ctrl->c, 2 * l);
    }
    double2 acc[1] = {{0.0, 0.0}};
    const int C = 1 << m.log2c;
    for (int64_t row = r0 + tid / TPR; row < r1; row += ROWS) {
        const int64_t ch = row >> m.log2c;
        const int64_t cp0 = m.chunk_ptr[ch];
        const int w = (int)((m.chunk_ptr[ch + 1] - cp0) >> m.log2c);
        const int64_t o = cp0 + (row & (C - 1)) * w;
        const int64_t ri = row * K + 2 * l;
        // own row
        double2 own;   // the vector the operator is applied to, at this row
        if (MODE == MODE_CG1 || MODE == MODE_CG2A) {
            double2 zv = ld2(a.in0, ri), pv = ld2(a.in1, ri), xv = ld2(a.x, ri);
            own.x = fma(beta.x, pv.x, zv.x);
            own.y = fma(beta.y, pv.y, zv.y);
            xv.x = fma(alpha.x, pv.x, xv.x);
            xv.y = fma(alpha.y, pv.y, xv.y);
            st2(a.x, ri, xv);
            st2(a.out1, ri, own);
        } else {
            own = ld2(a.in0, ri);
        }
        // off-diagonal gather
        double2 s = {0.0, 0.0};
        for (int k = 0; k < w; k += 2) {
            const int2 cj = *reinterpret_cast<const int2*>(m.col + o + k);
            const double2 vj = ld2(m.val, o + k);
            const int64_t j0 = (int64_t)cj.x * K + 2 * l, j1 = (int64_t)cj.y * K + 2 * l;
            double2 g0, g1;
            if (MODE == MODE_CG1 || MODE == MODE_CG2A) {
                double2 z0 = ld2(a.in0, j0), p0 = ld2(a.in1, j0), z1 = ld2(a.in0, j1), p1 = ld2(a.in1, j1);
                g0.x = fma(beta.x, p0.x, z0.x); g0.y = fma(beta.y, p0.y, z0.y);
                g1.x = fma(beta.x, p1.x, z1.x); g1.y = fma(beta.y, p1.y, z1.y);
            } else {
                g0 = ld2(a.in0, j0);
                g1 = ld2(a.in0, j1);
            }
            s.x = fma(vj.x, g0.x, s.x); s.y = fma(vj.x, g0.y, s.y);
            s.x = fma(vj.y, g1.x, s.x); s.y = fma(vj.y, g1.y, s.y);
        }
        const double sd = m.sdiag[row];
        s.x = fma(sd, own.x, s.x);
        s.y = fma(sd, own.y, s.y);          // s = (S v)_row
        if (MODE == MODE_PLAIN) {
            if (a.scale_inv_area) { const double ia = m.inv_area[row]; s.x *= ia; s.y *= ia; }
            st2(a.out0, ri, s);
        } else if (MODE == MODE_CG2A) {
            const double ia = m.inv_area[row];
            s.x *= ia; s.y *= ia;            // t = M^-1 S p'
            st2(a.out0, ri, s);
        } else {
            // q = A_v p + c (S v)_row ; v = p (n = 1) or t (n = 2)
            const double av = m.area[row];
            double2 pv = (MODE == MODE_CG1) ? own : ld2(a.in1, ri);
            double2 q;
            q.x = fma(cc.x, s.x, av * pv.x);
            q.y = fma(cc.y, s.y, av * pv.y);
            st2(a.out0, ri, q);
            acc[0].x = fma(pv.x, q.x, acc[0].x);
            acc[0].y = fma(pv.y, q.y, acc[0].y);
        }
    }
    if (MODE == MODE_CG1 || MODE == MODE_CG2B) {
        __shared__ double tot[KMAX];
        if (grid_reduce<K, 1>(acc, partials, &ctrl->ticket[0], tot)) {
            if (tid < K) {
                const double pq = tot[tid];
                double al = 0.0;
                if (!ctrl->done[tid]) {
                    if (pq > 0.0 && isfinite(pq)) al = ctrl->rho[tid] / pq;
                    else { ctrl->done[tid] = 1; ctrl->status[tid] = 2; }
                }
                ctrl->alpha[tid] = al;
            }
        }
    }
    if ((MODE == MODE_CG1 || MODE == MODE_CG2A) && blockIdx.x == 0 && tid == 0) ctrl->cur_p = a.out_idx;
}

// x[row][c] = field_c[perm[row]]  (H0 ingest: gather through the permutation, replicate per scale, transpose)
template <int K>
__global__ void __launch_bounds__(BLOCK) k_ingest(MeshView m, const Ctrl* __restrict__ ctrl,
                                                  const double* __restrict__ fields, double* __restrict__ x) {
    const int64_t i = (int64_t)blockIdx.x * BLOCK + threadIdx.x;
    if (i >= m.nv * K) return;
    const int64_t row = i / K;
    const int c = (int)(i % K);
    const int f = ctrl->field[c];
    x[i] = f >= 0 ? fields[(int64_t)f * m.nv + m.perm[row]] : 0.0;
}

// Start of CG from x0 = phi: y = S (M^-1 S)^(n-1) phi is given;
// r0 = M phi - A_c phi = -c y ;  z0 = r0/d ;  p = 0 ;  rho0 = r0.z0 ;  ||r0||^2 ;  ||M phi||^2.
template <int K>
__global__ void __launch_bounds__(BLOCK) k_init(MeshView m, Ctrl* __restrict__ ctrl, double* __restrict__ partials,
                                                const double* __restrict__ x, const double* __restrict__ y,
                                                double* __restrict__ z, double* __restrict__ p0, int order_n,
                                                int64_t rows_per_block) {
    constexpr int TPR = K / 2;
    constexpr int ROWS = BLOCK / TPR;
    const int tid = threadIdx.x, l = tid % TPR;
    const int64_t r0 = (int64_t)blockIdx.x * rows_per_block;
    const int64_t r1 = min(r0 + rows_per_block, m.nv);
    const double2 cc = ld2(ctrl->c, 2 * l);
    const double* __restrict__ dg = order_n == 1 ? m.sdiag : m.gdiag;
    double2 acc[3] = {{0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}};
    for (int64_t row = r0 + tid / TPR; row < r1; row += ROWS) {
        const int64_t ri = row * K + 2 * l;
        const double av = m.area[row], dv = dg[row];
        const double2 d = {fma(cc.x, dv, av), fma(cc.y, dv, av)};
        const double2 xv = ld2(x, ri), yv = ld2(y, ri);
        const double2 r = {-cc.x * yv.x, -cc.y * yv.y};
        const double2 zv = {r.x / d.x, r.y / d.y};
        st2(z, ri, zv);
        st2(p0, ri, make_double2(0.0, 0.0));
        acc[0].x = fma(r.x, zv.x, acc[0].x); acc[0].y = fma(r.y, zv.y, acc[0].y);
        acc[1].x = fma(r.x, r.x, acc[1].x);  acc[1].y = fma(r.y, r.y, acc[1].y);
        const double2 b = {av * xv.x, av * xv.y};
        acc[2].x = fma(b.x, b.x, acc[2].x);  acc[2].y = fma(b.y, b.y, acc[2].y);
    }
    __shared__ double tot[3 * KMAX];
    if (grid_reduce<K, 3>(acc, partials, &ctrl->ticket[1], tot)) {
        __shared__ int any_active;
        if (tid == 0) any_active = 0;
        __syncthreads();
        if (tid < K) {
            const double rho = tot[tid], rr = tot[KMAX + tid], bb = tot[2 * KMAX + tid];
            ctrl->rho[tid] = rho; ctrl->rr[tid] = rr; ctrl->bb[tid] = bb;
            ctrl->alpha[tid] = 0.0; ctrl->beta[tid] = 0.0; ctrl->iters[tid] = 0;
            int st = 0;
            int dn = (ctrl->field[tid] < 0) || (rr <= ctrl->tol2 * bb);
            if (!isfinite(rr) || !isfinite(bb)) { dn = 1; st = 2; }
            ctrl->done[tid] = dn; ctrl->status[tid] = st;
            if (!dn) atomicOr(&any_active, 1);
        }
        __syncthreads();
        if (tid == 0) { ctrl->all_done = !any_active; ctrl->cur_p = 0; }
    }
}

// kernel B: z -= alpha q/d ; rho' = sum d z^2 ; ||r||^2 = sum (d z)^2 ; then (last block) beta, stop tests.
template <int K>
__global__ void __launch_bounds__(BLOCK) k_update(MeshView m, Ctrl* __restrict__ ctrl, double* __restrict__ partials,
                                                  double* __restrict__ z, const double* __restrict__ q, int order_n,
                                                  int64_t rows_per_block) {
    constexpr int TPR = K / 2;
    constexpr int ROWS = BLOCK / TPR;
    if (ctrl->all_done) return;
    const int tid = threadIdx.x, l = tid % TPR;
    const int64_t r0 = (int64_t)blockIdx.x * rows_per_block;
    const int64_t r1 = min(r0 + rows_per_block, m.nv);
    const double2 cc = ld2(ctrl->c, 2 * l);
    const double2 alpha = ld2(ctrl->alpha, 2 * l);
    const double* __restrict__ dg = order_n == 1 ? m.sdiag : m.gdiag;
    double2 acc[2] = {{0.0, 0.0}, {0.0, 0.0}};
#pragma unroll 2
    for (int64_t row = r0 + tid / TPR; row < r1; row += ROWS) {
        const int64_t ri = row * K + 2 * l;
        const double av = m.area[row], dv = dg[row];
        const double2 d = {fma(cc.x, dv, av), fma(cc.y, dv, av)};
        double2 zv = ld2(z, ri);
        const double2 qv = ld2(q, ri);
        zv.x -= alpha.x * qv.x / d.x;
        zv.y -= alpha.y * qv.y / d.y;
        st2(z, ri, zv);
        const double2 r = {d.x * zv.x, d.y * zv.y};
        acc[0].x = fma(r.x, zv.x, acc[0].x); acc[0].y = fma(r.y, zv.y, acc[0].y);
        acc[1].x = fma(r.x, r.x, acc[1].x);  acc[1].y = fma(r.y, r.y, acc[1].y);
    }
    __shared__ double tot[2 * KMAX];
    if (grid_reduce<K, 2>(acc, partials, &ctrl->ticket[2], tot)) {
        __shared__ int any_active;
        if (tid == 0) any_active = 0;
        __syncthreads();
        if (tid < K) {
            if (!ctrl->done[tid]) {
                const double rho_new = tot[tid], rr = tot[KMAX + tid];
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
        if (tid == 0) ctrl->all_done = !any_active;
    }
}

// H6b: x_final = x + alpha p (the update still pending), e_c = 1/2 sum_v A_v x_v^2 / sum_v A_v
template <int K>
__global__ void __launch_bounds__(BLOCK) k_energy(MeshView m, Ctrl* __restrict__ ctrl, double* __restrict__ partials,
                                                  const double* __restrict__ x, const double* __restrict__ pa,
                                                  const double* __restrict__ pb, double total_area,
                                                  double* __restrict__ energy, int64_t rows_per_block) {
    constexpr int TPR = K / 2;
    constexpr int ROWS = BLOCK / TPR;
    const int tid = threadIdx.x, l = tid % TPR;
    const int64_t r0 = (int64_t)blockIdx.x * rows_per_block;
    const int64_t r1 = min(r0 + rows_per_block, m.nv);
    const double* __restrict__ p = ctrl->cur_p ? pb : pa;
    const double2 alpha = ld2(ctrl->alpha, 2 * l);
    double2 acc[1] = {{0.0, 0.0}};
    for (int64_t row = r0 + tid / TPR; row < r1; row += ROWS) {
        const int64_t ri = row * K + 2 * l;
        const double av = m.area[row];
        const double2 xv = ld2(x, ri), pv = ld2(p, ri);
        const double2 xf = {fma(alpha.x, pv.x, xv.x), fma(alpha.y, pv.y, xv.y)};
        acc[0].x = fma(av * xf.x, xf.x, acc[0].x);
        acc[0].y = fma(av * xf.y, xf.y, acc[0].y);
    }
    __shared__ double tot[KMAX];
    if (grid_reduce<K, 1>(acc, partials, &ctrl->ticket[3], tot)) {
        if (tid < K && ctrl->field[tid] >= 0) energy[ctrl->rhs[tid]] = 0.5 * tot[tid] / total_area;
    }
}

// H6a: x_final scattered back to the caller's numbering: out[rhs][perm[row]]
template <int K>
__global__ void __launch_bounds__(BLOCK) k_scatter(MeshView m, const Ctrl* __restrict__ ctrl,
                                                   const double* __restrict__ x, const double* __restrict__ pa,
                                                   const double* __restrict__ pb, int use_p, double* __restrict__ out) {
    __shared__ double tile[K][33];
    __shared__ int32_t dst[32];
    const int tid = threadIdx.x;
    const double* __restrict__ p = ctrl->cur_p ? pb : pa;
    // BLOCK threads move 32 rows x K columns per step
    for (int64_t base = (int64_t)blockIdx.x * 32; base < m.nv; base += (int64_t)gridDim.x * 32) {
        for (int e = tid; e < 32 * K; e += BLOCK) {
            const int r = e / K, c = e % K;
            const int64_t row = base + r;
            double v = 0.0;
            if (row < m.nv) {
                v = x[row * K + c];
                if (use_p) v = fma(ctrl->alpha[c], p[row * K + c], v);
            }
            tile[c][r] = v;
        }
        if (tid < 32) dst[tid] = base + tid < m.nv ? m.perm[base + tid] : -1;
        __syncthreads();
        for (int e = tid; e < 32 * K; e += BLOCK) {
            const int c = e / 32, r = e % 32;
            if (ctrl->field[c] >= 0 && dst[r] >= 0) out[(int64_t)ctrl->rhs[c] * m.nv + dst[r]] = tile[c][r];
        }
        __syncthreads();
    }
}

__global__ void k_stats(const Ctrl* __restrict__ ctrl, int K, int32_t* __restrict__ iters, int32_t* __restrict__ status,
                        double* __restrict__ relres) {
    const int c = threadIdx.x;
    if (c < K && ctrl->field[c] >= 0) {
        const int r = ctrl->rhs[c];
        iters[r] = ctrl->iters[c];
        status[r] = ctrl->status[c];
        relres[r] = ctrl->bb[c] > 0.0 ? sqrt(ctrl->rr[c] / ctrl->bb[c]) : 0.0;
    }
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

// ------------------------------------------------------------------------------------------- host side
struct Workspace {
    Ctrl* ctrl;
    double* partials;
    double *x, *z, *p0, *p1, *q, *t;
    double *energy, *relres, *ells, *k_mid, *E;
    int32_t *iters, *status;
    size_t bytes;
};

inline size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }

Workspace layout_workspace(const if_mesh_s* h, int order_n, int batch, void* base) {
    Workspace w{};
    char* p = static_cast<char*>(base);
    size_t off = 0;
    auto take = [&](size_t bytes) { void* r = p ? p + off : nullptr; off += align_up(bytes); return r; };
    const size_t vec = (size_t)h->n_vert * batch * sizeof(double);
    const size_t gmax = (size_t)h->n_sm * 8;
    w.ctrl = (Ctrl*)take(sizeof(Ctrl));
    w.partials = (double*)take(3 * gmax * KMAX * sizeof(double));
    w.x = (double*)take(vec);
    w.z = (double*)take(vec);
    w.p0 = (double*)take(vec);
    w.p1 = (double*)take(vec);
    w.q = (double*)take(vec);
    w.t = order_n == 2 ? (double*)take(vec) : nullptr;
    w.energy = (double*)take(MAX_RHS * sizeof(double));
    w.relres = (double*)take(MAX_RHS * sizeof(double));
    w.ells = (double*)take(MAX_RHS * sizeof(double));
    w.k_mid = (double*)take(MAX_RHS * sizeof(double));
    w.E = (double*)take(MAX_RHS * sizeof(double));
    w.iters = (int32_t*)take(MAX_RHS * sizeof(int32_t));
    w.status = (int32_t*)take(MAX_RHS * sizeof(int32_t));
    w.bytes = off;
    return w;
}

struct Geo { int grid; int64_t rows_per_block; };

Geo geometry(int64_t nv, int K, int n_sm, int blocks_per_sm) {
    const int rows = BLOCK / (K / 2);
    const int64_t nblk = (nv + rows - 1) / rows;
    int64_t grid = std::min<int64_t>(nblk, (int64_t)n_sm * blocks_per_sm);
    const int64_t rpb = (nblk + grid - 1) / grid * rows;
    grid = (nv + rpb - 1) / rpb;
    return Geo{(int)grid, rpb};
}

enum Job { JOB_FILTER, JOB_SPECTRUM, JOB_APPLY };

struct Rhs { double ell; int f; int j; };

struct Run {
    const if_mesh_s* h;
    MeshView m;
    Workspace w;
    cudaStream_t st;
    int order_n;
    Options opt;
};

// Events recorded (as external event-record nodes) around one SpMM and one update launch of a captured graph,
// so that the per-launch duration of both kernels is measured live on the launching stream (if_stats).
struct TimingEvents {
    cudaEvent_t s0 = nullptr, s1 = nullptr, u1 = nullptr;   // before SpMM, after SpMM (= before update), after update
    int create() {
        IF_CUDA_TRY(cudaEventCreate(&s0));
        IF_CUDA_TRY(cudaEventCreate(&s1));
        IF_CUDA_TRY(cudaEventCreate(&u1));
        return IF_OK;
    }
    void destroy() {
        if (s0) cudaEventDestroy(s0);
        if (s1) cudaEventDestroy(s1);
        if (u1) cudaEventDestroy(u1);
        s0 = s1 = u1 = nullptr;
    }
};

template <int K>
int enqueue_two_iterations(const Run& r, const Geo& g, const TimingEvents* tev = nullptr) {
    // iteration with p0 -> p1, then p1 -> p0
    for (int half = 0; half < 2; ++half) {
        const bool timed = tev && half == 0;
        if (timed) IF_CUDA_TRY(cudaEventRecordWithFlags(tev->s0, r.st, cudaEventRecordExternal));
        const double* pold = half == 0 ? r.w.p0 : r.w.p1;
        double* pnew = half == 0 ? r.w.p1 : r.w.p0;
        if (r.order_n == 1) {
            SpmmArgs a{r.w.z, pold, r.w.x, r.w.q, pnew, 0, half == 0 ? 1 : 0};
            k_spmm<K, MODE_CG1><<<g.grid, BLOCK, 0, r.st>>>(r.m, r.w.ctrl, r.w.partials, a, g.rows_per_block);
            IF_LAUNCH_CHECK();
        } else {
            SpmmArgs a{r.w.z, pold, r.w.x, r.w.t, pnew, 0, half == 0 ? 1 : 0};
            k_spmm<K, MODE_CG2A><<<g.grid, BLOCK, 0, r.st>>>(r.m, r.w.ctrl, r.w.partials, a, g.rows_per_block);
            IF_LAUNCH_CHECK();
            SpmmArgs b{r.w.t, pnew, nullptr, r.w.q, nullptr, 0, 0};
            k_spmm<K, MODE_CG2B><<<g.grid, BLOCK, 0, r.st>>>(r.m, r.w.ctrl, r.w.partials, b, g.rows_per_block);
            IF_LAUNCH_CHECK();
        }
        if (timed) IF_CUDA_TRY(cudaEventRecordWithFlags(tev->s1, r.st, cudaEventRecordExternal));
        k_update<K><<<g.grid, BLOCK, 0, r.st>>>(r.m, r.w.ctrl, r.w.partials, r.w.z, r.w.q, r.order_n,
                                                g.rows_per_block);
        IF_LAUNCH_CHECK();
        if (timed) IF_CUDA_TRY(cudaEventRecordWithFlags(tev->u1, r.st, cudaEventRecordExternal));
    }
    return IF_OK;
}

// Two instantiations of the iteration graph, launched alternately: while one runs, the host reads the timing
// events of the other (an event must not be re-recorded while it is being read).
struct GraphSet {
    cudaGraphExec_t exec[2] = {nullptr, nullptr};
    TimingEvents tev[2];
    ~GraphSet() {
        for (int i = 0; i < 2; ++i) { if (exec[i]) cudaGraphExecDestroy(exec[i]); tev[i].destroy(); }
    }
};

struct KernelTimes { double spmm_ms = 0.0, update_ms = 0.0; int64_t samples = 0; };

struct PollState {
    int* flags = nullptr;          // pinned [4]
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
    bool own_pinned = false;
    if_mesh_s* h = nullptr;
    ~PollState() {
        for (auto& e : ev) if (e) cudaEventDestroy(e);
        if (own_pinned && flags) cudaFreeHost(flags);
        else if (h) h->pinned_busy.store(0);
    }
};

template <int K>
int solve_batch(Run& r, Job job, const double* d_fields, const std::vector<Rhs>& rhs, size_t first, size_t count,
                int n_ells, double* d_out, PollState& poll, int blocks_per_sm, GraphSet* graph_cache,
                int64_t* batch_iters, KernelTimes* times) {
    const if_mesh_s* h = r.h;
    const Geo g = geometry(h->n_vert, K, h->n_sm, blocks_per_sm);
    Ctrl hc;
    memset(&hc, 0, sizeof(hc));
    for (int c = 0; c < KMAX; ++c) { hc.field[c] = -1; hc.rhs[c] = 0; hc.done[c] = 1; }
    for (size_t i = 0; i < count; ++i) {
        const Rhs& q = rhs[first + i];
        hc.c[i] = r.opt.gamma * std::pow(q.ell, 2.0 * r.order_n);
        hc.field[i] = q.f;
        hc.rhs[i] = q.f * n_ells + q.j;
        hc.done[i] = 0;
    }
    hc.max_iter = r.opt.max_iter;
    hc.tol2 = r.opt.tol * r.opt.tol;
    IF_CUDA_TRY(cudaMemcpyAsync(r.w.ctrl, &hc, sizeof(Ctrl), cudaMemcpyHostToDevice, r.st));
    const unsigned eg = (unsigned)((h->n_vert * K + BLOCK - 1) / BLOCK);
    k_ingest<K><<<eg, BLOCK, 0, r.st>>>(r.m, r.w.ctrl, d_fields, r.w.x);
    IF_LAUNCH_CHECK();

    if (job == JOB_APPLY) {
        const double* v = r.w.x;
        if (r.order_n == 2) {
            SpmmArgs a{r.w.x, nullptr, nullptr, r.w.t, nullptr, 1, 0};
            k_spmm<K, MODE_PLAIN><<<g.grid, BLOCK, 0, r.st>>>(r.m, r.w.ctrl, r.w.partials, a, g.rows_per_block);
            IF_LAUNCH_CHECK();
            v = r.w.t;
        }
        SpmmArgs b{v, r.w.x, nullptr, r.w.q, nullptr, 0, 0};
        k_spmm<K, MODE_CG2B><<<g.grid, BLOCK, 0, r.st>>>(r.m, r.w.ctrl, r.w.partials, b, g.rows_per_block);
        IF_LAUNCH_CHECK();
        k_scatter<K><<<std::min<int64_t>((h->n_vert + 31) / 32, (int64_t)h->n_sm * 8), BLOCK, 0, r.st>>>(
            r.m, r.w.ctrl, r.w.q, r.w.p0, r.w.p1, 0, d_out);
        IF_LAUNCH_CHECK();
        return IF_OK;
    }

    // y = S (M^-1 S)^(n-1) phi  -> q
    if (r.order_n == 1) {
        SpmmArgs a{r.w.x, nullptr, nullptr, r.w.q, nullptr, 0, 0};
        k_spmm<K, MODE_PLAIN><<<g.grid, BLOCK, 0, r.st>>>(r.m, r.w.ctrl, r.w.partials, a, g.rows_per_block);
        IF_LAUNCH_CHECK();
    } else {
        SpmmArgs a{r.w.x, nullptr, nullptr, r.w.t, nullptr, 1, 0};
        k_spmm<K, MODE_PLAIN><<<g.grid, BLOCK, 0, r.st>>>(r.m, r.w.ctrl, r.w.partials, a, g.rows_per_block);
        IF_LAUNCH_CHECK();
        SpmmArgs b{r.w.t, nullptr, nullptr, r.w.q, nullptr, 0, 0};
        k_spmm<K, MODE_PLAIN><<<g.grid, BLOCK, 0, r.st>>>(r.m, r.w.ctrl, r.w.partials, b, g.rows_per_block);
        IF_LAUNCH_CHECK();
    }
    k_init<K><<<g.grid, BLOCK, 0, r.st>>>(r.m, r.w.ctrl, r.w.partials, r.w.x, r.w.q, r.w.z, r.w.p0, r.order_n,
                                          g.rows_per_block);
    IF_LAUNCH_CHECK();

    // the iteration loop: `check_every` iterations per CUDA graph launch, flag polled one launch behind
    const int pairs = r.opt.check_every / 2;
    const int launches_per_graph = pairs * 2 * (r.order_n == 1 ? 2 : 3);
    GraphSet& gs = *graph_cache;
    if (!gs.exec[0] && r.st != nullptr && r.st != cudaStreamLegacy) {
        for (int gi = 0; gi < 2; ++gi) {
            if (gs.tev[gi].create() != IF_OK) return IF_ECUDA;
            cudaGraph_t graph = nullptr;
            if (cudaStreamBeginCapture(r.st, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
                cudaGetLastError();   // stream cannot be captured: fall through to direct launches
                break;
            }
            int rc = IF_OK;
            const int timed_pair = pairs > 1 ? 1 : 0;
            for (int i = 0; i < pairs && rc == IF_OK; ++i)
                rc = enqueue_two_iterations<K>(r, g, i == timed_pair ? &gs.tev[gi] : nullptr);
            g_launches -= (long long)launches_per_graph;   // captured, not launched
            cudaError_t e = cudaStreamEndCapture(r.st, &graph);
            if (rc != IF_OK || e != cudaSuccess) { if (graph) cudaGraphDestroy(graph); cudaGetLastError(); return IF_ECUDA; }
            e = cudaGraphInstantiate(&gs.exec[gi], graph, 0);
            cudaGraphDestroy(graph);
            if (e != cudaSuccess) { gs.exec[gi] = nullptr; cudaGetLastError(); return IF_ECUDA; }
        }
    }
    const bool use_graph = gs.exec[0] && gs.exec[1];
    const int64_t max_loops = (r.opt.max_iter + r.opt.check_every - 1) / r.opt.check_every + 2;
    for (int64_t it = 0; it < max_loops; ++it) {
        if (use_graph) {
            IF_CUDA_TRY(cudaGraphLaunch(gs.exec[it & 1], r.st));
            g_launches += (long long)launches_per_graph;
        } else {
            for (int i = 0; i < pairs; ++i) {
                int rc = enqueue_two_iterations<K>(r, g);
                if (rc != IF_OK) return rc;
            }
        }
        *batch_iters += r.opt.check_every;
        const int slot = (int)(it & 3);
        IF_CUDA_TRY(cudaMemcpyAsync(&poll.flags[slot], &r.w.ctrl->all_done, sizeof(int), cudaMemcpyDeviceToHost, r.st));
        IF_CUDA_TRY(cudaEventRecord(poll.ev[slot], r.st));
        if (it >= 1) {
            const int prev = (int)((it - 1) & 3);
            IF_CUDA_TRY(cudaEventSynchronize(poll.ev[prev]));
            if (use_graph && !poll.flags[prev]) {
                // launch it-1 did full work in every kernel: take its timing sample (graph (it-1)&1 is idle now)
                const TimingEvents& te = gs.tev[(it - 1) & 1];
                float a = 0.f, b = 0.f;
                if (cudaEventElapsedTime(&a, te.s0, te.s1) == cudaSuccess &&
                    cudaEventElapsedTime(&b, te.s1, te.u1) == cudaSuccess) {
                    times->spmm_ms += a; times->update_ms += b; times->samples += 1;
                } else {
                    cudaGetLastError();
                }
            }
            if (poll.flags[prev]) break;
        }
    }
    const int sgrid = (int)std::min<int64_t>((h->n_vert + 31) / 32, (int64_t)h->n_sm * 8);
    if (job == JOB_SPECTRUM) {
        k_energy<K><<<g.grid, BLOCK, 0, r.st>>>(r.m, r.w.ctrl, r.w.partials, r.w.x, r.w.p0, r.w.p1, h->total_area,
                                                r.w.energy, g.rows_per_block);
        IF_LAUNCH_CHECK();
    } else {
        k_scatter<K><<<sgrid, BLOCK, 0, r.st>>>(r.m, r.w.ctrl, r.w.x, r.w.p0, r.w.p1, 1, d_out);
        IF_LAUNCH_CHECK();
    }
    k_stats<<<1, 32, 0, r.st>>>(r.w.ctrl, K, r.w.iters, r.w.status, r.w.relres);
    IF_LAUNCH_CHECK();
    return IF_OK;
}

int dispatch_batch(int K, Run& r, Job job, const double* d_fields, const std::vector<Rhs>& rhs, size_t first,
                   size_t count, int n_ells, double* d_out, PollState& poll, int bps, GraphSet* cache,
                   int64_t* bi, KernelTimes* kt) {
    switch (K) {
        case 4: return solve_batch<4>(r, job, d_fields, rhs, first, count, n_ells, d_out, poll, bps, &cache[0], bi, kt);
        case 8: return solve_batch<8>(r, job, d_fields, rhs, first, count, n_ells, d_out, poll, bps, &cache[1], bi, kt);
        default: return solve_batch<16>(r, job, d_fields, rhs, first, count, n_ells, d_out, poll, bps, &cache[2], bi, kt);
    }
}

int run_job(if_handle h, Job job, const double* d_fields, int n_fields, const double* ells, int n_ells, int order_n,
            double* d_out, double* energy, double* k_mid, double* E, void* d_ws, size_t ws_bytes, void* stream,
            const if_options* opt_in, if_stats* stats) {
    if (!h || !d_fields || !ells || n_fields < 1 || n_ells < 1 || (order_n != 1 && order_n != 2) || !d_ws)
        return IF_EINVAL;
    if (job != JOB_SPECTRUM && !d_out) return IF_EINVAL;
    if (job == JOB_SPECTRUM && n_ells < 2) return IF_EINVAL;
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
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return IF_ECUDA; }
    if (dev != h->device) IF_CUDA_TRY(cudaSetDevice(h->device));
    r.w = layout_workspace(h, order_n, r.opt.batch, d_ws);
    if (ws_bytes < r.w.bytes) return IF_EWORKSPACE;
    int log2c = 0;
    while ((1 << log2c) < h->sell_c) ++log2c;
    r.m = MeshView{h->chunk_ptr, h->sell_col, h->sell_val, h->area, h->inv_area, h->sdiag, h->gdiag, h->perm,
                   h->n_vert, log2c};

    PollState poll;
    int expected = 0;
    if (h->h_pinned && h->pinned_busy.compare_exchange_strong(expected, 1)) {
        poll.flags = static_cast<int*>(h->h_pinned);
        poll.h = h;
    } else {
        IF_CUDA_TRY(cudaHostAlloc((void**)&poll.flags, 4 * sizeof(int), cudaHostAllocDefault));
        poll.own_pinned = true;
    }
    for (auto& e : poll.ev) IF_CUDA_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    cudaEvent_t t0 = nullptr, t1 = nullptr;
    IF_CUDA_TRY(cudaEventCreate(&t0));
    IF_CUDA_TRY(cudaEventCreate(&t1));
    struct EvGuard { cudaEvent_t a, b; ~EvGuard() { cudaEventDestroy(a); cudaEventDestroy(b); } } evg{t0, t1};
    IF_CUDA_TRY(cudaEventRecord(t0, r.st));

    int bps = 4;
    {
        int occ = 0;
        cudaError_t e = order_n == 1
            ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_spmm<16, MODE_CG1>, BLOCK, 0)
            : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_spmm<16, MODE_CG2A>, BLOCK, 0);
        if (e == cudaSuccess && occ > 0) bps = occ > 8 ? 8 : occ; else cudaGetLastError();
    }

    // right-hand sides sorted by scale so the columns of a batch need similar iteration counts
    std::vector<Rhs> rhs;
    rhs.reserve((size_t)R);
    for (int f = 0; f < n_fields; ++f)
        for (int j = 0; j < n_ells; ++j) rhs.push_back(Rhs{ells[j], f, j});
    if (job != JOB_APPLY)
        std::stable_sort(rhs.begin(), rhs.end(), [](const Rhs& a, const Rhs& b) { return a.ell < b.ell; });

    GraphSet cache[3];
    KernelTimes ktimes;
    std::vector<std::pair<size_t, size_t>> batches;
    int64_t launched_iters = 0;
    size_t first = 0;
    while (first < (size_t)R) {
        const size_t remaining = (size_t)R - first;
        int K = r.opt.batch;
        while (K > 4 && remaining <= (size_t)K / 2) K /= 2;
        const size_t count = remaining < (size_t)K ? remaining : (size_t)K;
        rc = dispatch_batch(K, r, job, d_fields, rhs, first, count, n_ells, d_out, poll, bps, cache, &launched_iters, &ktimes);
        if (rc != IF_OK) { cudaStreamSynchronize(r.st); return rc; }
        batches.emplace_back(first, count);
        first += count;
    }
    if (job == JOB_SPECTRUM) {
        IF_CUDA_TRY(cudaMemcpyAsync(r.w.ells, ells, (size_t)n_ells * sizeof(double), cudaMemcpyHostToDevice, r.st));
        const int nb = n_fields * (n_ells - 1);
        k_spectrum<<<(nb + 127) / 128, 128, 0, r.st>>>(r.w.energy, r.w.ells, n_fields, n_ells, r.w.k_mid, r.w.E);
        IF_LAUNCH_CHECK();
    }
    IF_CUDA_TRY(cudaEventRecord(t1, r.st));

    // results back to the host (small), then one synchronisation
    std::vector<int32_t> h_status((size_t)R, 0), h_iters((size_t)R, 0);
    std::vector<double> h_relres((size_t)R, 0.0);
    if (job != JOB_APPLY) {
        IF_CUDA_TRY(cudaMemcpyAsync(h_status.data(), r.w.status, (size_t)R * 4, cudaMemcpyDeviceToHost, r.st));
        IF_CUDA_TRY(cudaMemcpyAsync(h_iters.data(), r.w.iters, (size_t)R * 4, cudaMemcpyDeviceToHost, r.st));
        IF_CUDA_TRY(cudaMemcpyAsync(h_relres.data(), r.w.relres, (size_t)R * 8, cudaMemcpyDeviceToHost, r.st));
    }
    if (job == JOB_SPECTRUM) {
        if (energy) IF_CUDA_TRY(cudaMemcpyAsync(energy, r.w.energy, (size_t)R * 8, cudaMemcpyDeviceToHost, r.st));
        if (k_mid) IF_CUDA_TRY(cudaMemcpyAsync(k_mid, r.w.k_mid, (size_t)(n_ells - 1) * 8, cudaMemcpyDeviceToHost, r.st));
        if (E) IF_CUDA_TRY(cudaMemcpyAsync(E, r.w.E, (size_t)n_fields * (n_ells - 1) * 8, cudaMemcpyDeviceToHost, r.st));
    }
    IF_CUDA_TRY(cudaStreamSynchronize(r.st));
    int result = IF_OK;
    for (int64_t i = 0; i < R; ++i) if (h_status[(size_t)i] != 0) result = IF_WNOTCONVERGED;
    if (stats) {
        float ms = 0.f;
        IF_CUDA_TRY(cudaEventElapsedTime(&ms, t0, t1));
        stats->seconds = ms * 1e-3;
        stats->batch_iters = 0;
        stats->rhs_iters = 0;
        stats->spmm_seconds = ktimes.samples ? 1e-3 * ktimes.spmm_ms / (double)ktimes.samples : 0.0;
        stats->update_seconds = ktimes.samples ? 1e-3 * ktimes.update_ms / (double)ktimes.samples : 0.0;
        stats->kernel_samples = ktimes.samples;
        for (auto& b : batches) {
            int mx = 0;
            for (size_t i = 0; i < b.second; ++i) {
                const Rhs& q = rhs[b.first + i];
                mx = std::max(mx, (int)h_iters[(size_t)q.f * n_ells + q.j]);
            }
            stats->batch_iters += mx;
        }
        for (int64_t i = 0; i < R; ++i) {
            stats->rhs_iters += h_iters[(size_t)i];
            if (stats->iters) stats->iters[i] = h_iters[(size_t)i];
            if (stats->status) stats->status[i] = h_status[(size_t)i];
            if (stats->rel_res) stats->rel_res[i] = h_relres[(size_t)i];
        }
    }
    return result;
}

}  // namespace
}  // namespace ifl

using namespace ifl;

extern "C" int if_workspace_bytes(if_handle h, int order_n, int batch, size_t* bytes) {
    if (!h || !bytes || (order_n != 1 && order_n != 2)) return IF_EINVAL;
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

extern "C" int if_apply(if_handle h, const double* d_fields, int n_fields, const double* ells, int n_ells, int order_n,
                        double* d_out, void* d_workspace, size_t ws_bytes, void* cuda_stream, const if_options* opt) {
    return run_job(h, JOB_APPLY, d_fields, n_fields, ells, n_ells, order_n, d_out, nullptr, nullptr, nullptr,
                   d_workspace, ws_bytes, cuda_stream, opt, nullptr);
}
