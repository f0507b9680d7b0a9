// Multigrid hierarchy for the n = 1 systems (M + c S) x = M phi at large scales (the cost and the
// loss of convergence of plain CG at large l are the paper's stated open problem).
//
// Smoothed aggregation on the internal (space-filling-curve) row order:
//   aggregates      greedy over the graph of the strong connections of S (|S_ij| >= MG_THETA sqrt(S_ii S_jj)), in
//                   row order: a row whose neighbours are all free becomes a root and takes them; leftovers join a
//                   neighbouring aggregate (tentative prolongator P_t: piecewise constant).  Graph aggregates never join two connected components of the masked mesh, which
//                   blocks of consecutive rows did; it is a serial sweep and runs on the host (once per mesh).
//   prolongator     P = (I - omega_p D_S^-1 S) P_t, omega_p = 4 / (3 rho(D_S^-1 S)), rho by power iteration
//                   (smoothed with the stiffness only, so P does not depend on the scale)
//   coarse pair     S_c = P^T S P ,  M_c = P^T M P               (Galerkin; A_c = M_c + c S_c for every column)
// All sparse products are built as "emit (key, value) triples -> radix sort -> reduce by key", the pattern the
// assembly of S already uses (prepare.cu).  Built once per mesh by if_prepare(IF_FLAG_MULTIGRID).
#include <cub/cub.cuh>

#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <new>
#include <vector>

#include "common.cuh"

namespace ifl {
namespace {

constexpr int MG_POWER_ITERS = 24;     // power iteration for rho(D_S^-1 S)
constexpr double MG_RHO_SAFETY = 1.05;  // the iteration approaches rho from below

// Scratch and result buffers of the build come from the device's stream-ordered pool (cudaMallocAsync on the build's
// stream): the build makes some forty allocations per level, and with cudaMalloc / cudaFree their fixed cost (a
// millisecond each, with a device synchronisation) was most of the build time on the small levels.  mg_build keeps
// the pool from returning memory to the driver while it runs and trims it at the end.
struct DBuf {
    void* p = nullptr;
    ~DBuf() { if (p) cudaFreeAsync(p, 0); }
    cudaError_t alloc(size_t bytes) {
        if (p) { cudaFreeAsync(p, 0); p = nullptr; }
        return cudaMallocAsync(&p, bytes + 16, 0);      // +16: the row-block kernels bulk-copy 16-byte multiples
    }
    template <class T> T* as() const { return static_cast<T*>(p); }
    void* release() { void* q = p; p = nullptr; return q; }
};

struct Add2 {
    __device__ __forceinline__ double2 operator()(const double2& a, const double2& b) const {
        return make_double2(a.x + b.x, a.y + b.y);
    }
};

typedef unsigned long long u64;
inline unsigned gridf(int64_t n, int block = 256) { return (unsigned)((n + block - 1) / block); }
inline int bitsf(uint64_t n) { int b = 1; while ((1ull << b) < n && b < 63) ++b; return b; }

// rowptr[r] = first sorted key whose row (high 32 bits) >= r
__global__ void k_mg_rowptr(const u64* __restrict__ keys, int64_t nnz, int64_t n, int64_t* __restrict__ rowptr) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i > nnz) return;
    int64_t row_i = i < nnz ? (int64_t)(keys[i] >> 32) : n;
    int64_t row_p = i > 0 ? (int64_t)(keys[i - 1] >> 32) : -1;
    for (int64_t r = row_p + 1; r <= row_i; ++r) rowptr[r] = i;
}
__global__ void k_mg_cols(const u64* __restrict__ keys, int64_t nnz, int32_t* __restrict__ col) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < nnz) col[i] = (int32_t)(keys[i] & 0xffffffffull);
}

// level 0 from the SELL matrix: row lengths (diagonal + off-diagonals that are not padding), then the entries
__global__ void k_mg_l0_len(const int64_t* __restrict__ chunk_ptr, const int32_t* __restrict__ scol, int log2c,
                            int64_t nv, int64_t* __restrict__ len) {
    int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r > nv) return;
    if (r == nv) { len[r] = 0; return; }
    const int C = 1 << log2c;
    const int64_t ch = r >> log2c, cp0 = chunk_ptr[ch];
    const int w = (int)((chunk_ptr[ch + 1] - cp0) >> log2c);
    const int64_t o = cp0 + (r & (C - 1)) * w;
    int n = 1;
    for (int k = 0; k < w; ++k) n += (scol[o + k] != (int32_t)r);
    len[r] = n;
}
__global__ void k_mg_l0_fill(const int64_t* __restrict__ chunk_ptr, const int32_t* __restrict__ scol,
                             const double* __restrict__ sval, const double* __restrict__ sdiag,
                             const double* __restrict__ area, int log2c, int64_t nv,
                             const int64_t* __restrict__ rowptr, int32_t* __restrict__ col, double2* __restrict__ sm,
                             double2* __restrict__ diag) {
    int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= nv) return;
    const int C = 1 << log2c;
    const int64_t ch = r >> log2c, cp0 = chunk_ptr[ch];
    const int w = (int)((chunk_ptr[ch + 1] - cp0) >> log2c);
    const int64_t o = cp0 + (r & (C - 1)) * w;
    int64_t e = rowptr[r];
    col[e] = (int32_t)r;
    sm[e] = make_double2(sdiag[r], area[r]);
    ++e;
    for (int k = 0; k < w; ++k) {
        const int32_t c = scol[o + k];
        if (c == (int32_t)r) continue;
        col[e] = c;
        sm[e] = make_double2(sval[o + k], 0.0);
        ++e;
    }
    diag[r] = make_double2(sdiag[r], area[r]);
}

// P = (I - omega D_S^-1 S) P_t : one triple per matrix entry, keyed (row, aggregate of the column)
__global__ void k_mg_emit_p(const int64_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                            const double2* __restrict__ sm, const double2* __restrict__ diag,
                            const int32_t* __restrict__ agg, double omega_p, int64_t n,
                            u64* __restrict__ keys, double* __restrict__ vals) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double sii = diag[i].x;
    const double f = sii > 0.0 ? -omega_p / sii : 0.0;
    const int64_t b = rowptr[i], e = rowptr[i + 1];
    const int64_t o = b + i;   // one extra triple per row (the tentative prolongator)
    keys[o] = ((u64)i << 32) | (u64)agg[i];
    vals[o] = 1.0;
    for (int64_t k = b; k < e; ++k) {
        keys[o + 1 + (k - b)] = ((u64)i << 32) | (u64)agg[col[k]];
        vals[o + 1 + (k - b)] = f * sm[k].x;
    }
}

// triples of P with swapped key (aggregate, row): sorted they are R = P^T by rows
__global__ void k_mg_swap_keys(const int64_t* __restrict__ p_rowptr, const int32_t* __restrict__ p_col, int64_t n,
                               u64* __restrict__ keys) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    for (int64_t k = p_rowptr[i]; k < p_rowptr[i + 1]; ++k) keys[k] = ((u64)p_col[k] << 32) | (u64)i;
}

// T = G P (G = the level's (S, M) pair): counts per row, then the triples keyed (row, aggregate)
__global__ void k_mg_count_t(const int64_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                             const int64_t* __restrict__ p_rowptr, int64_t n, int64_t* __restrict__ cnt) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i > n) return;
    int64_t c = 0;
    if (i < n)
        for (int64_t k = rowptr[i]; k < rowptr[i + 1]; ++k) c += p_rowptr[col[k] + 1] - p_rowptr[col[k]];
    cnt[i] = c;
}
__global__ void k_mg_emit_t(const int64_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                            const double2* __restrict__ sm, const int64_t* __restrict__ p_rowptr,
                            const int32_t* __restrict__ p_col, const double* __restrict__ p_val, int64_t n,
                            const int64_t* __restrict__ off, u64* __restrict__ keys, double2* __restrict__ vals) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int64_t o = off[i];
    for (int64_t k = rowptr[i]; k < rowptr[i + 1]; ++k) {
        const int64_t j = col[k];
        const double2 g = sm[k];
        for (int64_t q = p_rowptr[j]; q < p_rowptr[j + 1]; ++q) {
            keys[o] = ((u64)i << 32) | (u64)p_col[q];
            vals[o] = make_double2(g.x * p_val[q], g.y * p_val[q]);
            ++o;
        }
    }
}

// G_c = P^T T : counts per fine row, then the triples keyed (aggregate a, aggregate b)
__global__ void k_mg_count_c(const int64_t* __restrict__ p_rowptr, const int64_t* __restrict__ t_rowptr, int64_t n,
                             int64_t* __restrict__ cnt) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i > n) return;
    cnt[i] = i < n ? (p_rowptr[i + 1] - p_rowptr[i]) * (t_rowptr[i + 1] - t_rowptr[i]) : 0;
}
__global__ void k_mg_emit_c(const int64_t* __restrict__ p_rowptr, const int32_t* __restrict__ p_col,
                            const double* __restrict__ p_val, const int64_t* __restrict__ t_rowptr,
                            const int32_t* __restrict__ t_col, const double2* __restrict__ t_sm, int64_t n,
                            const int64_t* __restrict__ off, u64* __restrict__ keys, double2* __restrict__ vals) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int64_t o = off[i];
    for (int64_t q = p_rowptr[i]; q < p_rowptr[i + 1]; ++q) {
        const u64 a = (u64)p_col[q];
        const double pv = p_val[q];
        for (int64_t k = t_rowptr[i]; k < t_rowptr[i + 1]; ++k) {
            keys[o] = (a << 32) | (u64)t_col[k];
            vals[o] = make_double2(pv * t_sm[k].x, pv * t_sm[k].y);
            ++o;
        }
    }
}

__global__ void k_mg_diag(const int64_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                          const double2* __restrict__ sm, int64_t n, double2* __restrict__ diag) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double2 d = make_double2(0.0, 0.0);
    for (int64_t k = rowptr[i]; k < rowptr[i + 1]; ++k)
        if (col[k] == (int32_t)i) { d.x += sm[k].x; d.y += sm[k].y; }
    diag[i] = d;
}

// sort (key, value) pairs by key and add the values of equal keys; the inputs are released
template <class V, class Op>
int sort_reduce(DBuf& keys, DBuf& vals, int64_t n, int key_bits, Op op, DBuf& ukeys, DBuf& uvals, int64_t* n_unique,
                cudaStream_t st) {
    DBuf k1, v1, tmp, d_n;
    IF_CUDA_TRY(k1.alloc((size_t)n * sizeof(u64)));
    IF_CUDA_TRY(v1.alloc((size_t)n * sizeof(V)));
    size_t tb = 0;
    IF_CUDA_TRY(cub::DeviceRadixSort::SortPairs(nullptr, tb, keys.as<u64>(), k1.as<u64>(), vals.as<V>(), v1.as<V>(), n, 0,
                                                key_bits, st));
    IF_CUDA_TRY(tmp.alloc(tb));
    IF_CUDA_TRY(cub::DeviceRadixSort::SortPairs(tmp.p, tb, keys.as<u64>(), k1.as<u64>(), vals.as<V>(), v1.as<V>(), n, 0,
                                                key_bits, st));
    ++g_launches;
    IF_CUDA_TRY(cudaStreamSynchronize(st));
    keys.alloc(0);
    vals.alloc(0);
    IF_CUDA_TRY(ukeys.alloc((size_t)n * sizeof(u64)));
    IF_CUDA_TRY(uvals.alloc((size_t)n * sizeof(V)));
    IF_CUDA_TRY(d_n.alloc(sizeof(int64_t)));
    tb = 0;
    IF_CUDA_TRY(cub::DeviceReduce::ReduceByKey(nullptr, tb, k1.as<u64>(), ukeys.as<u64>(), v1.as<V>(), uvals.as<V>(),
                                               d_n.as<int64_t>(), op, n, st));
    IF_CUDA_TRY(tmp.alloc(tb));
    IF_CUDA_TRY(cub::DeviceReduce::ReduceByKey(tmp.p, tb, k1.as<u64>(), ukeys.as<u64>(), v1.as<V>(), uvals.as<V>(),
                                               d_n.as<int64_t>(), op, n, st));
    ++g_launches;
    IF_CUDA_TRY(cudaMemcpyAsync(n_unique, d_n.p, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
    IF_CUDA_TRY(cudaStreamSynchronize(st));
    return IF_OK;
}

// CSR (rowptr, col) from sorted unique keys (row << 32 | col)
int csr_from_keys(const u64* ukeys, int64_t nnz, int64_t n_rows, DBuf& rowptr, DBuf& col, cudaStream_t st) {
    IF_CUDA_TRY(rowptr.alloc((size_t)(n_rows + 1) * sizeof(int64_t)));
    IF_CUDA_TRY(col.alloc((size_t)nnz * sizeof(int32_t)));
    k_mg_rowptr<<<gridf(nnz + 1), 256, 0, st>>>(ukeys, nnz, n_rows, rowptr.as<int64_t>());
    IF_LAUNCH_CHECK();
    k_mg_cols<<<gridf(nnz), 256, 0, st>>>(ukeys, nnz, col.as<int32_t>());
    IF_LAUNCH_CHECK();
    return IF_OK;
}

int exclusive_scan(int64_t* d_in, int64_t* d_out, int64_t n, int64_t* total, cudaStream_t st) {
    DBuf tmp;
    size_t tb = 0;
    IF_CUDA_TRY(cub::DeviceScan::ExclusiveSum(nullptr, tb, d_in, d_out, n, st));
    IF_CUDA_TRY(tmp.alloc(tb));
    IF_CUDA_TRY(cub::DeviceScan::ExclusiveSum(tmp.p, tb, d_in, d_out, n, st));
    ++g_launches;
    IF_CUDA_TRY(cudaMemcpyAsync(total, d_out + (n - 1), sizeof(int64_t), cudaMemcpyDeviceToHost, st));
    IF_CUDA_TRY(cudaStreamSynchronize(st));
    return IF_OK;
}

// power iteration on D_S^-1 S (part 0) or D_M^-1 M (part 1): y = D^-1 B x, sq = y^2 ;  x = y / ||y||
__global__ void k_mg_power_start(int64_t n, double* __restrict__ x) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    u64 z = (u64)i * 0x9E3779B97F4A7C15ull + 0x632BE59BD9B4E019ull;   // splitmix64 finaliser: fixed pseudo-random signs
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    z ^= z >> 31;
    x[i] = (double)(z >> 11) * (2.0 / 9007199254740992.0) - 1.0;
}
__global__ void k_mg_power_apply(const int64_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                                 const double2* __restrict__ sm, const double2* __restrict__ diag, int part, int64_t n,
                                 const double* __restrict__ x, double* __restrict__ y, double* __restrict__ sq) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double s = 0.0;
    for (int64_t k = rowptr[i]; k < rowptr[i + 1]; ++k) s = fma(part ? sm[k].y : sm[k].x, x[col[k]], s);
    const double d = part ? diag[i].y : diag[i].x;
    s = d > 0.0 ? s / d : 0.0;
    y[i] = s;
    sq[i] = s * s;
}
__global__ void k_mg_power_scale(int64_t n, const double* __restrict__ y, const double* __restrict__ sumsq,
                                 double* __restrict__ x) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double nrm = sqrt(*sumsq);
    x[i] = nrm > 0.0 ? y[i] / nrm : 0.0;
}

// rho(D_S^-1 S) (part 0) or rho(D_M^-1 M) (part 1) of a level; >= 1 is returned.  The mass part is diagonal on the
// mesh (rho = 1) but not below it: M_l = P^T M P has positive off-diagonal entries and its Jacobi-scaled spectrum
// reaches 2-3, with the smooth vectors on top -- the damping of the smoother must cover both parts, since the
// Rayleigh quotients of D^-1 (M_l + c S_l) lie between those of the two parts for every c.
int spectral_radius(const MgLevel& f, int part, double* rho, cudaStream_t st) {
    const int64_t n = f.n;
    DBuf x, y, sq, sum, tmp;
    IF_CUDA_TRY(x.alloc((size_t)n * sizeof(double)));
    IF_CUDA_TRY(y.alloc((size_t)n * sizeof(double)));
    IF_CUDA_TRY(sq.alloc((size_t)n * sizeof(double)));
    IF_CUDA_TRY(sum.alloc(sizeof(double)));
    size_t tb = 0;
    IF_CUDA_TRY(cub::DeviceReduce::Sum(nullptr, tb, sq.as<double>(), sum.as<double>(), n, st));
    IF_CUDA_TRY(tmp.alloc(tb));
    k_mg_power_start<<<gridf(n), 256, 0, st>>>(n, y.as<double>());
    IF_LAUNCH_CHECK();
    double h_sum = (double)n;   // rough norm^2 of the start vector; from the second step on x has norm 1 exactly
    IF_CUDA_TRY(cudaMemcpyAsync(sum.p, &h_sum, sizeof(double), cudaMemcpyHostToDevice, st));
    IF_CUDA_TRY(cudaStreamSynchronize(st));
    for (int it = 0; it < MG_POWER_ITERS; ++it) {
        k_mg_power_scale<<<gridf(n), 256, 0, st>>>(n, y.as<double>(), sum.as<double>(), x.as<double>());
        IF_LAUNCH_CHECK();
        k_mg_power_apply<<<gridf(n), 256, 0, st>>>(f.rowptr, f.col, f.sm, f.diag, part, n, x.as<double>(), y.as<double>(),
                                                  sq.as<double>());
        IF_LAUNCH_CHECK();
        IF_CUDA_TRY(cub::DeviceReduce::Sum(tmp.p, tb, sq.as<double>(), sum.as<double>(), n, st));
        ++g_launches;
    }
    IF_CUDA_TRY(cudaMemcpyAsync(&h_sum, sum.p, sizeof(double), cudaMemcpyDeviceToHost, st));
    IF_CUDA_TRY(cudaStreamSynchronize(st));
    const double r = std::sqrt(h_sum) * MG_RHO_SAFETY;
    *rho = (std::isfinite(r) && r > 1.0) ? r : 1.0;
    return IF_OK;
}

// strength of connection: keep[k] = 1 for the diagonal and for the entries with S_ij^2 >= theta^2 S_ii S_jj
__global__ void k_mg_strong(const int64_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                            const double2* __restrict__ sm, const double2* __restrict__ diag, double theta2, int64_t n,
                            uint8_t* __restrict__ keep) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double sii = diag[i].x;
    for (int64_t k = rowptr[i]; k < rowptr[i + 1]; ++k) {
        const int32_t j = col[k];
        const double sij = sm[k].x;
        keep[k] = (j == i || sij * sij >= theta2 * sii * diag[j].x) ? 1 : 0;
    }
}

// Aggregation over the graph of the level's matrix, on the device.  Roots = a maximal set of rows that are pairwise
// more than two strong connections apart (a distance-2 maximal independent set): every root takes its strong
// neighbours, and what is left -- rows two connections away from the nearest root -- joins the aggregate of its first
// aggregated neighbour.  That is what a serial greedy sweep builds too (a row whose neighbours are all free becomes
// a root and takes them; round 1 ran that sweep on the host, 0.2-0.4 s per level for 7.3 M rows); here the roots are
// found in parallel rounds with hashed priorities (Luby's scheme over two-ring maxima: an undecided row whose key is
// the largest within distance two becomes a root, a row that sees a root within distance two is out), a dozen
// rounds of two passes over the graph.  Aggregates are numbered in the order of their roots, so the coarse
// numbering follows the fine one along the curve.
// The graph is that of the strong connections (MG_THETA): weak ones -- across a sliver, or the small entries the
// Galerkin products accumulate on the coarse levels -- do not pull a row into an aggregate.  Should the filtered
// graph coarsen by less than MG_MIN_COARSENING (the prolongator is smoothed with the whole matrix, so small
// aggregates mean fill-in on the next level), the level falls back to the whole graph.
// key of a row: state (2 = root, 1 = undecided, 0 = out) << 61 | 30 hashed bits << 31 | row id
__device__ __forceinline__ u64 agg_key(int state, int64_t i) {
    if (state == 0) return 0ull;
    u64 z = (u64)i * 0x9E3779B97F4A7C15ull + 0x7F4A7C159E3779B9ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    z ^= z >> 31;
    return ((u64)state << 61) | ((z & 0x3fffffffull) << 31) | (u64)i;
}
__global__ void k_agg_init(int64_t n, u64* __restrict__ key) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) key[i] = agg_key(1, i);
}
// out[i] = max of in over the row itself and its strong neighbours
__global__ void k_agg_max(const int64_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                          const uint8_t* __restrict__ keep, int64_t n, const u64* __restrict__ in, u64* __restrict__ out) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    u64 m = in[i];
    for (int64_t k = rowptr[i]; k < rowptr[i + 1]; ++k)
        if (keep[k]) { const u64 v = in[col[k]]; m = v > m ? v : m; }
    out[i] = m;
}
// t2 = two-ring maximum of the keys: decide the undecided rows
__global__ void k_agg_decide(int64_t n, const u64* __restrict__ t2, u64* __restrict__ key, int* __restrict__ undecided) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const u64 k = key[i];
    if ((k >> 61) != 1ull) return;
    const u64 m = t2[i];
    if (m == k) key[i] = agg_key(2, i);
    else if ((m >> 61) == 2ull) key[i] = 0ull;
    else atomicAdd(undecided, 1);
}
__global__ void k_agg_root_flag(int64_t n, const u64* __restrict__ key, int64_t* __restrict__ flag) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i <= n) flag[i] = (i < n && (key[i] >> 61) == 2ull) ? 1 : 0;
}
// pass 1: a root and its strong neighbours (a row has at most one root among them)
__global__ void k_agg_assign1(const int64_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                              const uint8_t* __restrict__ keep, int64_t n, const u64* __restrict__ key,
                              const int64_t* __restrict__ root_id, int32_t* __restrict__ agg) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int32_t a = -1;
    if ((key[i] >> 61) == 2ull) a = (int32_t)root_id[i];
    else
        for (int64_t k = rowptr[i]; k < rowptr[i + 1]; ++k)
            if (keep[k] && (key[col[k]] >> 61) == 2ull) { a = (int32_t)root_id[col[k]]; break; }
    agg[i] = a;
}
// pass 2: a leftover joins the aggregate (as of pass 1) of its first aggregated neighbour; leftover[i] = 1 if none
__global__ void k_agg_assign2(const int64_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                              const uint8_t* __restrict__ keep, int64_t n, const int32_t* __restrict__ agg1,
                              int32_t* __restrict__ agg, int64_t* __restrict__ leftover) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i > n) return;
    if (i == n) { leftover[i] = 0; return; }
    int32_t a = agg1[i];
    if (a < 0)
        for (int64_t k = rowptr[i]; k < rowptr[i + 1]; ++k)
            if (keep[k] && agg1[col[k]] >= 0) { a = agg1[col[k]]; break; }
    agg[i] = a;
    leftover[i] = a < 0 ? 1 : 0;
}
// pass 3: what is still free becomes its own aggregate, numbered after the others
__global__ void k_agg_assign3(int64_t n, const int64_t* __restrict__ left_id, int64_t n_roots, int32_t* __restrict__ agg) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n && agg[i] < 0) agg[i] = (int32_t)(n_roots + left_id[i]);
}
__global__ void k_fill_u8(int64_t n, uint8_t v, uint8_t* __restrict__ p) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = v;
}

int exclusive_scan(int64_t* d_in, int64_t* d_out, int64_t n, int64_t* total, cudaStream_t st);

int aggregate_graph(const MgLevel& f, const uint8_t* keep, DBuf& d_agg, int64_t* n_agg, cudaStream_t st) {
    const int64_t n = f.n;
    DBuf key, t1, t2, cnt, flag, ids, agg1, left, left_id;
    IF_CUDA_TRY(key.alloc((size_t)n * 8));
    IF_CUDA_TRY(t1.alloc((size_t)n * 8));
    IF_CUDA_TRY(t2.alloc((size_t)n * 8));
    IF_CUDA_TRY(cnt.alloc(sizeof(int)));
    k_agg_init<<<gridf(n), 256, 0, st>>>(n, key.as<u64>());
    IF_LAUNCH_CHECK();
    for (int round = 0; round < 200; ++round) {
        IF_CUDA_TRY(cudaMemsetAsync(cnt.p, 0, sizeof(int), st));
        k_agg_max<<<gridf(n), 256, 0, st>>>(f.rowptr, f.col, keep, n, key.as<u64>(), t1.as<u64>());
        IF_LAUNCH_CHECK();
        k_agg_max<<<gridf(n), 256, 0, st>>>(f.rowptr, f.col, keep, n, t1.as<u64>(), t2.as<u64>());
        IF_LAUNCH_CHECK();
        k_agg_decide<<<gridf(n), 256, 0, st>>>(n, t2.as<u64>(), key.as<u64>(), cnt.as<int>());
        IF_LAUNCH_CHECK();
        int undecided = 0;
        IF_CUDA_TRY(cudaMemcpyAsync(&undecided, cnt.p, sizeof(int), cudaMemcpyDeviceToHost, st));
        IF_CUDA_TRY(cudaStreamSynchronize(st));
        if (undecided == 0) break;
    }
    IF_CUDA_TRY(flag.alloc((size_t)(n + 1) * 8));
    IF_CUDA_TRY(ids.alloc((size_t)(n + 1) * 8));
    k_agg_root_flag<<<gridf(n + 1), 256, 0, st>>>(n, key.as<u64>(), flag.as<int64_t>());
    IF_LAUNCH_CHECK();
    int64_t n_roots = 0;
    int rc = exclusive_scan(flag.as<int64_t>(), ids.as<int64_t>(), n + 1, &n_roots, st);
    if (rc) return rc;
    IF_CUDA_TRY(agg1.alloc((size_t)n * 4));
    IF_CUDA_TRY(d_agg.alloc((size_t)n * 4));
    IF_CUDA_TRY(left.alloc((size_t)(n + 1) * 8));
    IF_CUDA_TRY(left_id.alloc((size_t)(n + 1) * 8));
    k_agg_assign1<<<gridf(n), 256, 0, st>>>(f.rowptr, f.col, keep, n, key.as<u64>(), ids.as<int64_t>(), agg1.as<int32_t>());
    IF_LAUNCH_CHECK();
    k_agg_assign2<<<gridf(n + 1), 256, 0, st>>>(f.rowptr, f.col, keep, n, agg1.as<int32_t>(), d_agg.as<int32_t>(),
                                                left.as<int64_t>());
    IF_LAUNCH_CHECK();
    int64_t n_left = 0;
    if ((rc = exclusive_scan(left.as<int64_t>(), left_id.as<int64_t>(), n + 1, &n_left, st))) return rc;
    if (n_left > 0) {
        k_agg_assign3<<<gridf(n), 256, 0, st>>>(n, left_id.as<int64_t>(), n_roots, d_agg.as<int32_t>());
        IF_LAUNCH_CHECK();
    }
    *n_agg = n_roots + n_left;
    return IF_OK;
}

int aggregate_rows(const MgLevel& f, DBuf& d_agg, int64_t* n_agg, cudaStream_t st) {
    const int64_t n = f.n;
    DBuf d_keep;
    IF_CUDA_TRY(d_keep.alloc((size_t)f.nnz));
    int rc;
    if (MG_THETA > 0.0) {
        k_mg_strong<<<gridf(n), 256, 0, st>>>(f.rowptr, f.col, f.sm, f.diag, MG_THETA * MG_THETA, n, d_keep.as<uint8_t>());
        IF_LAUNCH_CHECK();
        if ((rc = aggregate_graph(f, d_keep.as<uint8_t>(), d_agg, n_agg, st))) return rc;
        if ((double)*n_agg * MG_MIN_COARSENING <= (double)n) return IF_OK;
    }
    k_fill_u8<<<gridf(f.nnz), 256, 0, st>>>(f.nnz, 1, d_keep.as<uint8_t>());
    IF_LAUNCH_CHECK();
    return aggregate_graph(f, d_keep.as<uint8_t>(), d_agg, n_agg, st);
}

// transfer operators and the Galerkin pair of level `f` -> fills f.p_*, f.r_* and the matrix of level c
int build_next_level(MgLevel& f, MgLevel& c, cudaStream_t st) {
    const int64_t n = f.n;
    int rc;
    DBuf agg;
    int64_t nc = 0;
    const bool verbose = getenv("IF_VERBOSE") != nullptr;
    auto t_prev = std::chrono::steady_clock::now();
    auto lap = [&](const char* what) {
        if (!verbose) return;
        cudaStreamSynchronize(st);
        const auto t = std::chrono::steady_clock::now();
        fprintf(stderr, "[implicit_filter]   %lld rows: %s %.1f ms\n", (long long)n, what,
                1e3 * std::chrono::duration<double>(t - t_prev).count());
        t_prev = t;
    };
    if ((rc = aggregate_rows(f, agg, &nc, st))) return rc;
    lap("aggregates");
    const double omega_p = 4.0 / (3.0 * f.rho);
    // ---- P
    {
        const int64_t ne = f.nnz + n;
        DBuf keys, vals, uk, uv;
        IF_CUDA_TRY(keys.alloc((size_t)ne * sizeof(u64)));
        IF_CUDA_TRY(vals.alloc((size_t)ne * sizeof(double)));
        k_mg_emit_p<<<gridf(n), 256, 0, st>>>(f.rowptr, f.col, f.sm, f.diag, agg.as<int32_t>(), omega_p, n,
                                             keys.as<u64>(), vals.as<double>());
        IF_LAUNCH_CHECK();
        int64_t pn = 0;
        if ((rc = sort_reduce<double>(keys, vals, ne, 32 + bitsf((uint64_t)n), cub::Sum(), uk, uv, &pn, st))) return rc;
        DBuf prow, pcol, pval;
        if ((rc = csr_from_keys(uk.as<u64>(), pn, n, prow, pcol, st))) return rc;
        IF_CUDA_TRY(pval.alloc((size_t)pn * sizeof(double)));
        IF_CUDA_TRY(cudaMemcpyAsync(pval.p, uv.p, (size_t)pn * sizeof(double), cudaMemcpyDeviceToDevice, st));
        IF_CUDA_TRY(cudaStreamSynchronize(st));
        f.n_coarse = nc; f.p_nnz = pn;
        f.p_rowptr = (int64_t*)prow.release(); f.p_col = (int32_t*)pcol.release(); f.p_val = (double*)pval.release();
    }
    lap("P");
    // ---- R = P^T
    {
        DBuf keys, vals, k1, v1, tmp;
        IF_CUDA_TRY(keys.alloc((size_t)f.p_nnz * sizeof(u64)));
        IF_CUDA_TRY(k1.alloc((size_t)f.p_nnz * sizeof(u64)));
        IF_CUDA_TRY(v1.alloc((size_t)f.p_nnz * sizeof(double)));
        k_mg_swap_keys<<<gridf(n), 256, 0, st>>>(f.p_rowptr, f.p_col, n, keys.as<u64>());
        IF_LAUNCH_CHECK();
        size_t tb = 0;
        IF_CUDA_TRY(cub::DeviceRadixSort::SortPairs(nullptr, tb, keys.as<u64>(), k1.as<u64>(), f.p_val, v1.as<double>(),
                                                    f.p_nnz, 0, 32 + bitsf((uint64_t)nc), st));
        IF_CUDA_TRY(tmp.alloc(tb));
        IF_CUDA_TRY(cub::DeviceRadixSort::SortPairs(tmp.p, tb, keys.as<u64>(), k1.as<u64>(), f.p_val, v1.as<double>(),
                                                    f.p_nnz, 0, 32 + bitsf((uint64_t)nc), st));
        ++g_launches;
        DBuf rrow, rcol;
        if ((rc = csr_from_keys(k1.as<u64>(), f.p_nnz, nc, rrow, rcol, st))) return rc;
        IF_CUDA_TRY(cudaStreamSynchronize(st));
        f.r_rowptr = (int64_t*)rrow.release(); f.r_col = (int32_t*)rcol.release(); f.r_val = (double*)v1.release();
    }
    lap("R");
    // ---- T = G P
    DBuf trow, tcol, tsm;
    int64_t tn = 0;
    {
        DBuf cnt, off;
        IF_CUDA_TRY(cnt.alloc((size_t)(n + 1) * sizeof(int64_t)));
        IF_CUDA_TRY(off.alloc((size_t)(n + 1) * sizeof(int64_t)));
        k_mg_count_t<<<gridf(n + 1), 256, 0, st>>>(f.rowptr, f.col, f.p_rowptr, n, cnt.as<int64_t>());
        IF_LAUNCH_CHECK();
        int64_t ne = 0;
        if ((rc = exclusive_scan(cnt.as<int64_t>(), off.as<int64_t>(), n + 1, &ne, st))) return rc;
        DBuf keys, vals, uk, uv;
        IF_CUDA_TRY(keys.alloc((size_t)ne * sizeof(u64)));
        IF_CUDA_TRY(vals.alloc((size_t)ne * sizeof(double2)));
        k_mg_emit_t<<<gridf(n), 256, 0, st>>>(f.rowptr, f.col, f.sm, f.p_rowptr, f.p_col, f.p_val, n, off.as<int64_t>(),
                                             keys.as<u64>(), vals.as<double2>());
        IF_LAUNCH_CHECK();
        if ((rc = sort_reduce<double2>(keys, vals, ne, 32 + bitsf((uint64_t)n), Add2(), uk, uv, &tn, st))) return rc;
        if ((rc = csr_from_keys(uk.as<u64>(), tn, n, trow, tcol, st))) return rc;
        IF_CUDA_TRY(tsm.alloc((size_t)tn * sizeof(double2)));
        IF_CUDA_TRY(cudaMemcpyAsync(tsm.p, uv.p, (size_t)tn * sizeof(double2), cudaMemcpyDeviceToDevice, st));
        IF_CUDA_TRY(cudaStreamSynchronize(st));
    }
    lap("T = G P");
    // ---- G_c = P^T T
    {
        DBuf cnt, off;
        IF_CUDA_TRY(cnt.alloc((size_t)(n + 1) * sizeof(int64_t)));
        IF_CUDA_TRY(off.alloc((size_t)(n + 1) * sizeof(int64_t)));
        k_mg_count_c<<<gridf(n + 1), 256, 0, st>>>(f.p_rowptr, trow.as<int64_t>(), n, cnt.as<int64_t>());
        IF_LAUNCH_CHECK();
        int64_t ne = 0;
        if ((rc = exclusive_scan(cnt.as<int64_t>(), off.as<int64_t>(), n + 1, &ne, st))) return rc;
        DBuf keys, vals, uk, uv;
        IF_CUDA_TRY(keys.alloc((size_t)ne * sizeof(u64)));
        IF_CUDA_TRY(vals.alloc((size_t)ne * sizeof(double2)));
        k_mg_emit_c<<<gridf(n), 256, 0, st>>>(f.p_rowptr, f.p_col, f.p_val, trow.as<int64_t>(), tcol.as<int32_t>(),
                                             tsm.as<double2>(), n, off.as<int64_t>(), keys.as<u64>(), vals.as<double2>());
        IF_LAUNCH_CHECK();
        int64_t cn = 0;
        if ((rc = sort_reduce<double2>(keys, vals, ne, 32 + bitsf((uint64_t)nc), Add2(), uk, uv, &cn, st))) return rc;
        DBuf crow, ccol, csm, cdiag;
        if ((rc = csr_from_keys(uk.as<u64>(), cn, nc, crow, ccol, st))) return rc;
        IF_CUDA_TRY(csm.alloc((size_t)cn * sizeof(double2)));
        IF_CUDA_TRY(cudaMemcpyAsync(csm.p, uv.p, (size_t)cn * sizeof(double2), cudaMemcpyDeviceToDevice, st));
        IF_CUDA_TRY(cdiag.alloc((size_t)nc * sizeof(double2)));
        k_mg_diag<<<gridf(nc), 256, 0, st>>>(crow.as<int64_t>(), ccol.as<int32_t>(), csm.as<double2>(), nc,
                                            cdiag.as<double2>());
        IF_LAUNCH_CHECK();
        IF_CUDA_TRY(cudaStreamSynchronize(st));
        c.n = nc; c.nnz = cn;
        c.rowptr = (int64_t*)crow.release(); c.col = (int32_t*)ccol.release();
        c.sm = (double2*)csm.release(); c.diag = (double2*)cdiag.release();
    }
    lap("P^T T");
    return IF_OK;
}

}  // namespace

namespace {
__global__ void k_mg_tile_cap(const int64_t* __restrict__ rowptr, int64_t n, int* __restrict__ cap) {
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t r0 = t * MG_TILE;
    if (r0 >= n) return;
    const int64_t r1 = r0 + MG_TILE < n ? r0 + MG_TILE : n;
    atomicMax(cap, (int)(rowptr[r1] - rowptr[r0]));
}
}  // namespace

int mg_tile_caps(if_mesh_s* h) {
    if (h->mg_levels < 1) return IF_OK;
    int* d = nullptr;
    IF_CUDA_TRY(cudaMalloc((void**)&d, 3 * MG_MAX_LEVELS * sizeof(int)));
    IF_CUDA_TRY(cudaMemset(d, 0, 3 * MG_MAX_LEVELS * sizeof(int)));
    for (int l = 0; l < h->mg_levels; ++l) {
        const MgLevel& g = h->mg[l];
        const unsigned ga = (unsigned)(((g.n + MG_TILE - 1) / MG_TILE + 255) / 256);
        k_mg_tile_cap<<<ga, 256>>>(g.rowptr, g.n, d + 3 * l);
        if (l + 1 < h->mg_levels && g.p_rowptr) {
            k_mg_tile_cap<<<ga, 256>>>(g.p_rowptr, g.n, d + 3 * l + 1);
            const unsigned gr = (unsigned)(((g.n_coarse + MG_TILE - 1) / MG_TILE + 255) / 256);
            k_mg_tile_cap<<<gr, 256>>>(g.r_rowptr, g.n_coarse, d + 3 * l + 2);
        }
    }
    int host[3 * MG_MAX_LEVELS];
    cudaError_t e = cudaMemcpy(host, d, sizeof(host), cudaMemcpyDeviceToHost);
    cudaFree(d);
    IF_CUDA_TRY(e);
    for (int l = 0; l < h->mg_levels; ++l) { h->mg[l].cap_a = host[3 * l]; h->mg[l].cap_p = host[3 * l + 1]; h->mg[l].cap_r = host[3 * l + 2]; }
    return IF_OK;
}

void mg_free(if_mesh_s* h) {
    for (int l = 0; l < MG_MAX_LEVELS; ++l) {
        MgLevel& g = h->mg[l];
        cudaFree(g.rowptr); cudaFree(g.col); cudaFree(g.sm); cudaFree(g.diag);
        cudaFree(g.p_rowptr); cudaFree(g.p_col); cudaFree(g.p_val);
        cudaFree(g.r_rowptr); cudaFree(g.r_col); cudaFree(g.r_val);
        g = MgLevel();
    }
    h->mg_levels = 0;
}

struct PoolHold {     // keep freed blocks in the pool for the duration of the build
    cudaMemPool_t pool = nullptr;
    PoolHold(int device) {
        if (cudaDeviceGetDefaultMemPool(&pool, device) != cudaSuccess) { pool = nullptr; cudaGetLastError(); return; }
        uint64_t keep = ~0ull;
        cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
    }
    ~PoolHold() {
        if (!pool) return;
        uint64_t keep = 0;
        cudaStreamSynchronize(0);
        cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
        cudaMemPoolTrimTo(pool, 0);
    }
};

int mg_build(if_mesh_s* h) {
    const auto t_start = std::chrono::steady_clock::now();
    cudaStream_t st = 0;
    PoolHold hold(h->device);
    const int64_t nv = h->n_vert;
    int log2c = 0;
    while ((1 << log2c) < h->sell_c) ++log2c;
    // level 0: the (S, M) pair in CSR, internal order, diagonal first in every row
    {
        DBuf len, rowptr, col, sm, diag;
        IF_CUDA_TRY(len.alloc((size_t)(nv + 1) * sizeof(int64_t)));
        IF_CUDA_TRY(rowptr.alloc((size_t)(nv + 1) * sizeof(int64_t)));
        k_mg_l0_len<<<gridf(nv + 1), 256, 0, st>>>(h->chunk_ptr, h->sell_col, log2c, nv, len.as<int64_t>());
        IF_LAUNCH_CHECK();
        int64_t nnz = 0;
        int rc = exclusive_scan(len.as<int64_t>(), rowptr.as<int64_t>(), nv + 1, &nnz, st);
        if (rc) return rc;
        IF_CUDA_TRY(col.alloc((size_t)nnz * sizeof(int32_t)));
        IF_CUDA_TRY(sm.alloc((size_t)nnz * sizeof(double2)));
        IF_CUDA_TRY(diag.alloc((size_t)nv * sizeof(double2)));
        k_mg_l0_fill<<<gridf(nv), 256, 0, st>>>(h->chunk_ptr, h->sell_col, h->sell_val, h->sdiag, h->area, log2c, nv,
                                               rowptr.as<int64_t>(), col.as<int32_t>(), sm.as<double2>(),
                                               diag.as<double2>());
        IF_LAUNCH_CHECK();
        IF_CUDA_TRY(cudaStreamSynchronize(st));
        MgLevel& g = h->mg[0];
        g.n = nv; g.nnz = nnz;
        g.rowptr = (int64_t*)rowptr.release(); g.col = (int32_t*)col.release();
        g.sm = (double2*)sm.release(); g.diag = (double2*)diag.release();
    }
    int L = 1;
    for (;;) {
        MgLevel& g = h->mg[L - 1];
        int rc = spectral_radius(g, 0, &g.rho, st);
        if (rc == IF_OK && L > 1) rc = spectral_radius(g, 1, &g.rho_m, st);
        if (rc != IF_OK) { mg_free(h); return rc; }
        g.omega = std::min(MG_OMEGA_MAX, 1.6 / std::max(g.rho, g.rho_m));
        if (g.n <= MG_COARSEST || L >= MG_MAX_LEVELS) break;
        rc = build_next_level(g, h->mg[L], st);
        if (rc != IF_OK) { mg_free(h); return rc; }
        if (h->mg[L].n >= g.n) break;            // no coarsening (a graph without edges): stop here
        ++L;
    }
    h->mg_levels = L;
    IF_CUDA_TRY(cudaStreamSynchronize(st));
    { int rc = mg_tile_caps(h); if (rc != IF_OK) { mg_free(h); return rc; } }
    h->mg_build_seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count();
    if (getenv("IF_VERBOSE"))
        for (int l = 0; l < L; ++l)
            fprintf(stderr, "[implicit_filter] multigrid level %d: %lld rows, %.1f entries per row, rho(S) %.3f, rho(M) %.3f, "
                            "omega %.3f, P %.1f entries per row\n", l, (long long)h->mg[l].n,
                    (double)h->mg[l].nnz / (double)h->mg[l].n, h->mg[l].rho, h->mg[l].rho_m, h->mg[l].omega,
                    h->mg[l].n ? (double)h->mg[l].p_nnz / (double)h->mg[l].n : 0.0);
    return IF_OK;
}

}  // namespace ifl
