// Preparation phase: mesh -> device-resident S (SELL-C-sigma), A_v and diagonals.
//
//   P1  triangle geometry: edge vectors (minimum image on periodic axes), |e1 x e2|, cotangents
//       S_ab += -1/2 cot(angle opposite ab)   = integral grad N_a . grad N_b dS
//   P2  half-edge assembly: 6 directed off-diagonal contributions + 3 area contributions per triangle,
//       radix-sorted by (row, col) and summed by key; edges seen by one triangle only (boundary) keep the
//       single contribution = natural no-normal-flux condition; S_vv = -sum_j S_vj
//   P3  A_v = sum over triangles of area/3 (median-dual = lumped P1 mass, PAPER.md:41 Fig. 1a, :61)
//   P4  Morton order of the quantised coordinates (space-filling curve) -> perm
//   P5  SELL-C-sigma: rows sorted by length inside windows of sigma rows, slices of C rows padded to the
//       slice maximum (rounded up to even so int2/double2 loads stay aligned), row-major inside a slice
//   P6  Jacobi ingredients S_vv and g_v = sum_j S_vj^2/A_j = diag(S M^-1 S)
#include <cub/cub.cuh>

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "common.cuh"

namespace ifl {

std::atomic<long long> g_launches{0};

namespace {

struct DevBuf {
    void* p = nullptr;
    ~DevBuf() { if (p) cudaFree(p); }
    cudaError_t alloc(size_t bytes) {
        if (p) { cudaFree(p); p = nullptr; }
        return cudaMalloc(&p, bytes ? bytes : 1);
    }
    template <class T> T* as() const { return static_cast<T*>(p); }
    void* release() { void* q = p; p = nullptr; return q; }
};

enum { FLAG_INDEX = 1, FLAG_DEGENERATE = 2, FLAG_ORPHAN = 4 };

struct Period { double p[3]; };

__device__ inline void edge_vec(const double* __restrict__ coords, int dim, const Period& per, int64_t from,
                                int64_t to, double e[3]) {
    e[0] = e[1] = e[2] = 0.0;
    for (int d = 0; d < dim; ++d) {
        double v = coords[to * dim + d] - coords[from * dim + d];
        if (per.p[d] > 0.0) v -= per.p[d] * rint(v / per.p[d]);
        e[d] = v;
    }
}

// P1 + P2 (emit): 9 keyed contributions per triangle.
__global__ void k_tri_emit(const double* __restrict__ coords, int dim, int64_t nv, const int32_t* __restrict__ tri,
                           int64_t nt, Period per, unsigned long long* __restrict__ keys, double* __restrict__ vals,
                           int* __restrict__ flags) {
    int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nt) return;
    int64_t v[3] = {tri[3 * t], tri[3 * t + 1], tri[3 * t + 2]};
    int64_t base = 9 * t;
    bool bad = false;
    for (int c = 0; c < 3; ++c) bad |= (v[c] < 0 || v[c] >= nv);
    bad |= (v[0] == v[1] || v[0] == v[2] || v[1] == v[2]);
    if (bad) {
        atomicOr(flags, FLAG_INDEX);
        for (int i = 0; i < 9; ++i) { keys[base + i] = 0ull; vals[base + i] = 0.0; }
        return;
    }
    double tarea = 0.0;
    for (int c = 0; c < 3; ++c) {
        int64_t vc = v[c], va = v[(c + 1) % 3], vb = v[(c + 2) % 3];
        double e1[3], e2[3];
        edge_vec(coords, dim, per, vc, va, e1);
        edge_vec(coords, dim, per, vc, vb, e2);
        double cx = e1[1] * e2[2] - e1[2] * e2[1];
        double cy = e1[2] * e2[0] - e1[0] * e2[2];
        double cz = e1[0] * e2[1] - e1[1] * e2[0];
        double cr = sqrt(cx * cx + cy * cy + cz * cz);
        double dt = e1[0] * e2[0] + e1[1] * e2[1] + e1[2] * e2[2];
        double n1 = e1[0] * e1[0] + e1[1] * e1[1] + e1[2] * e1[2];
        double n2 = e2[0] * e2[0] + e2[1] * e2[1] + e2[2] * e2[2];
        if (!(cr > 1e-14 * (n1 + n2))) { atomicOr(flags, FLAG_DEGENERATE); cr = 1.0; }
        double w = -0.5 * dt / cr;
        keys[base + 2 * c] = ((unsigned long long)va << 32) | (unsigned long long)vb;
        vals[base + 2 * c] = w;
        keys[base + 2 * c + 1] = ((unsigned long long)vb << 32) | (unsigned long long)va;
        vals[base + 2 * c + 1] = w;
        if (c == 0) tarea = 0.5 * cr;
    }
    for (int c = 0; c < 3; ++c) {
        keys[base + 6 + c] = ((unsigned long long)v[c] << 32) | (unsigned long long)v[c];
        vals[base + 6 + c] = tarea / 3.0;
    }
}

// Vector filter: per triangle the 9 contributions to D~ = int (grad N_v . grad N_v' + (R_e^-2 + m^2) N_v N_v')
// and to T = int m (-N_v' dx N_v + N_v dx N_v'), with the same 9 keys (row, col) as the stiffness assembly, so that after
// sort + sum by key the entries line up one to one with the CSR of S.  The triangle is the flat 3-D triangle; latitude
// and zonal direction are those of its centroid, m = tan(latitude) / R_e constant on it; P1 gradients
// grad N_a = n x (x_c - x_b) / (2 area); int N_a N_b = area (1 + delta_ab) / 12, int N_a = area / 3.
struct Add2v {
    __device__ __forceinline__ double2 operator()(const double2& a, const double2& b) const {
        return make_double2(a.x + b.x, a.y + b.y);
    }
};
__global__ void k_tri_emit_vec(const double* __restrict__ coords, int dim, const int32_t* __restrict__ tri, int64_t nt,
                               Period per, double inv_r, unsigned long long* __restrict__ keys, double2* __restrict__ vals) {
    int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nt) return;
    const int64_t v[3] = {tri[3 * t], tri[3 * t + 1], tri[3 * t + 2]};
    double x[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
    for (int d = 0; d < dim; ++d) x[0][d] = coords[v[0] * dim + d];
    for (int c = 1; c < 3; ++c) {
        double e[3];
        edge_vec(coords, dim, per, v[0], v[c], e);
        for (int d = 0; d < 3; ++d) x[c][d] = x[0][d] + e[d];
    }
    double e1[3], e2[3], nrm[3];
    for (int d = 0; d < 3; ++d) { e1[d] = x[1][d] - x[0][d]; e2[d] = x[2][d] - x[0][d]; }
    nrm[0] = e1[1] * e2[2] - e1[2] * e2[1];
    nrm[1] = e1[2] * e2[0] - e1[0] * e2[2];
    nrm[2] = e1[0] * e2[1] - e1[1] * e2[0];
    const double cr = sqrt(nrm[0] * nrm[0] + nrm[1] * nrm[1] + nrm[2] * nrm[2]);
    const double area = 0.5 * cr;
    for (int d = 0; d < 3; ++d) nrm[d] /= cr;
    double g[3][3];
    for (int a = 0; a < 3; ++a) {
        const int b = (a + 1) % 3, c = (a + 2) % 3;
        const double ed[3] = {x[c][0] - x[b][0], x[c][1] - x[b][1], x[c][2] - x[b][2]};
        g[a][0] = (nrm[1] * ed[2] - nrm[2] * ed[1]) / cr;
        g[a][1] = (nrm[2] * ed[0] - nrm[0] * ed[2]) / cr;
        g[a][2] = (nrm[0] * ed[1] - nrm[1] * ed[0]) / cr;
    }
    double mt = 0.0, east[3] = {1.0, 0.0, 0.0};
    if (dim == 3 && inv_r > 0.0) {
        const double cx = (x[0][0] + x[1][0] + x[2][0]) / 3.0, cy = (x[0][1] + x[1][1] + x[2][1]) / 3.0;
        const double cz = (x[0][2] + x[1][2] + x[2][2]) / 3.0;
        const double rho = sqrt(cx * cx + cy * cy);
        mt = (cz / rho) * inv_r;
        east[0] = -cy / rho; east[1] = cx / rho; east[2] = 0.0;
    }
    double gx[3];
    for (int a = 0; a < 3; ++a) gx[a] = g[a][0] * east[0] + g[a][1] * east[1] + g[a][2] * east[2];
    const double mass_c = inv_r * inv_r + mt * mt;
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) {
            const double gg = g[a][0] * g[b][0] + g[a][1] * g[b][1] + g[a][2] * g[b][2];
            keys[9 * t + 3 * a + b] = ((unsigned long long)v[a] << 32) | (unsigned long long)v[b];
            vals[9 * t + 3 * a + b] = make_double2(area * gg + mass_c * area * (a == b ? 2.0 : 1.0) / 12.0,
                                                   mt * (area / 3.0) * (gx[b] - gx[a]));
        }
}

// the (D~, T) pairs of the CSR (caller numbering) into the SELL slots of the internal order, exactly as k_sell_fill
// placed the entries of S; per row D~_vv and diag(D_2 M_2^-1 D_2)_v = sum_j (D~_vj^2 + T_vj^2) / A_j
__global__ void k_sell_fill_vec(const int32_t* __restrict__ perm, const int64_t* __restrict__ rowptr,
                                const int32_t* __restrict__ col, const double2* __restrict__ dt,
                                const double* __restrict__ area_u, int64_t nv, int64_t n_chunks, int C,
                                const int64_t* __restrict__ chunk_ptr, double* __restrict__ sell_dval,
                                double* __restrict__ sell_tval, double* __restrict__ ddiag, double* __restrict__ gdiag_vec) {
    int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_chunks * C) return;
    const int64_t c = r / C;
    const int64_t w = (chunk_ptr[c + 1] - chunk_ptr[c]) / C;
    const int64_t o = chunk_ptr[c] + (r - c * C) * w;
    int64_t k = 0;
    if (r < nv) {
        const int64_t u = perm[r];
        double gv = 0.0;
        for (int64_t i = rowptr[u]; i < rowptr[u + 1]; ++i) {
            const double2 e = dt[i];
            gv += (e.x * e.x + e.y * e.y) / area_u[col[i]];
            if (col[i] == u) { ddiag[r] = e.x; continue; }
            sell_dval[o + k] = e.x;
            sell_tval[o + k] = e.y;
            ++k;
        }
        gdiag_vec[r] = gv;
    }
    for (; k < w; ++k) { sell_dval[o + k] = 0.0; sell_tval[o + k] = 0.0; }
}

// rowptr[r] = first unique entry whose row >= r.
__global__ void k_rowptr(const unsigned long long* __restrict__ ukeys, int64_t nnz, int64_t nv,
                         int64_t* __restrict__ rowptr) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i > nnz) return;
    int64_t row_i = i < nnz ? (int64_t)(ukeys[i] >> 32) : nv;
    int64_t row_p = i > 0 ? (int64_t)(ukeys[i - 1] >> 32) : -1;
    for (int64_t r = row_p + 1; r <= row_i; ++r) rowptr[r] = i;
}

// Per caller row: the keyed sum at (v,v) is A_v; replace it by S_vv = -sum of off-diagonals.
__global__ void k_row_finish(const unsigned long long* __restrict__ ukeys, const int64_t* __restrict__ rowptr,
                             int64_t nv, double* __restrict__ val, int32_t* __restrict__ col,
                             double* __restrict__ area, double* __restrict__ sdiag, int32_t* __restrict__ len,
                             int* __restrict__ flags) {
    int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= nv) return;
    int64_t b = rowptr[v], e = rowptr[v + 1];
    double off = 0.0, a = 0.0;
    int64_t dpos = -1;
    for (int64_t i = b; i < e; ++i) {
        int32_t c = (int32_t)(ukeys[i] & 0xffffffffull);
        col[i] = c;
        if (c == v) { dpos = i; a = val[i]; } else off += val[i];
    }
    if (dpos < 0 || !(a > 0.0)) { atomicOr(flags, FLAG_ORPHAN); area[v] = 1.0; sdiag[v] = 0.0; len[v] = 0; return; }
    val[dpos] = -off;
    area[v] = a;
    sdiag[v] = -off;
    len[v] = (int32_t)(e - b - 1);
}

__global__ void k_gdiag(const int64_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                        const double* __restrict__ val, const double* __restrict__ area, int64_t nv,
                        double* __restrict__ gdiag) {
    int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= nv) return;
    double g = 0.0;
    for (int64_t i = rowptr[v]; i < rowptr[v + 1]; ++i) g += val[i] * val[i] / area[col[i]];
    gdiag[v] = g;
}

// Jacobi diagonals of the higher orders ("can be generalized to higher-order filters"), exactly.
// With y = column v of M^-1 S (the one-ring of v: y_j = S_vj / A_j, S symmetric):
//   n = 3:  diag(S M^-1 S M^-1 S)_v = y^T S y = sum_j y_j sum_{k in row(j), k in row(v)} S_jk y_k
//   n = 4:  diag(S (M^-1 S)^3)_v = z^T M^-1 z,  z = S y (the two-ring of v) = sum_k z_k^2 / A_k
// Columns are ascending inside a CSR row, so membership in row(v) is a binary search; z is accumulated in a small
// per-thread table (a two-ring beyond its capacity -- valences of several dozen -- falls back to the k = v term alone,
// a positive lower bound: the preconditioner stays symmetric positive definite, only weaker for that row).
constexpr int RING2_CAP = 192;
__global__ void k_gdiag_higher(const int64_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                               const double* __restrict__ val, const double* __restrict__ area, int64_t nv,
                               double* __restrict__ gdiag3, double* __restrict__ gdiag4) {
    int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= nv) return;
    const int64_t b = rowptr[v], e = rowptr[v + 1];
    int32_t kk[RING2_CAP];
    double zz[RING2_CAP];
    int nz = 0;
    bool overflow = false;
    double d3 = 0.0, zv = 0.0;
    for (int64_t a = b; a < e; ++a) {
        const int64_t j = col[a];
        const double yj = val[a] / area[j];
        double sy = 0.0;                                   // (S y)_j restricted to row(v) -- y vanishes elsewhere
        for (int64_t i = rowptr[j]; i < rowptr[j + 1]; ++i) {
            const int32_t k = col[i];
            const double sjk = val[i];
            int64_t lo = b, hi = e - 1;                    // k in row(v)?
            while (lo < hi) { const int64_t mid = (lo + hi) >> 1; if (col[mid] < k) lo = mid + 1; else hi = mid; }
            if (col[lo] == k) sy += sjk * (val[lo] / area[k]);
            // z_k += S_kj y_j
            if (k == v) zv += sjk * yj;
            int t = 0;
            while (t < nz && kk[t] != k) ++t;
            if (t == nz) {
                if (nz < RING2_CAP) { kk[nz] = k; zz[nz] = 0.0; ++nz; } else { overflow = true; continue; }
            }
            zz[t] += sjk * yj;
        }
        d3 += yj * sy;
    }
    double d4 = 0.0;
    if (overflow) d4 = zv * zv / area[v];
    else for (int t = 0; t < nz; ++t) d4 += zz[t] * zz[t] / area[kk[t]];
    gdiag3[v] = d3;
    gdiag4[v] = d4;
}

// length of each edge once (row < col), 0 elsewhere
__global__ void k_edge_len(const double* __restrict__ coords, int dim, Period per, const int64_t* __restrict__ rowptr,
                           const int32_t* __restrict__ col, int64_t nv, double* __restrict__ out) {
    int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= nv) return;
    for (int64_t i = rowptr[v]; i < rowptr[v + 1]; ++i) {
        double l = 0.0;
        if (col[i] > v) {
            double e[3];
            edge_vec(coords, dim, per, v, col[i], e);
            l = sqrt(e[0] * e[0] + e[1] * e[1] + e[2] * e[2]);
        }
        out[i] = l;
    }
}

__device__ inline unsigned long long spread3(unsigned long long x) {   // 21 bits -> every third bit
    x &= 0x1fffffull;
    x = (x | x << 32) & 0x1f00000000ffffull;
    x = (x | x << 16) & 0x1f0000ff0000ffull;
    x = (x | x << 8) & 0x100f00f00f00f00full;
    x = (x | x << 4) & 0x10c30c30c30c30c3ull;
    x = (x | x << 2) & 0x1249249249249249ull;
    return x;
}
__device__ inline unsigned long long spread2(unsigned long long x) {   // 31 bits -> every second bit
    x &= 0x7fffffffull;
    x = (x | x << 16) & 0x0000ffff0000ffffull;
    x = (x | x << 8) & 0x00ff00ff00ff00ffull;
    x = (x | x << 4) & 0x0f0f0f0f0f0f0f0full;
    x = (x | x << 2) & 0x3333333333333333ull;
    x = (x | x << 1) & 0x5555555555555555ull;
    return x;
}

struct Box { double lo[3]; double scale[3]; };

__global__ void k_morton(const double* __restrict__ coords, int dim, int64_t nv, Box box,
                         unsigned long long* __restrict__ keys, int32_t* __restrict__ ids, int identity) {
    int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= nv) return;
    ids[v] = (int32_t)v;
    if (identity) { keys[v] = (unsigned long long)v; return; }
    unsigned long long q[3] = {0, 0, 0};
    const double top = dim == 3 ? 2097151.0 : 2147483647.0;
    for (int d = 0; d < dim; ++d) {
        double s = (coords[v * dim + d] - box.lo[d]) * box.scale[d] * top;
        s = fmin(fmax(s, 0.0), top);
        q[d] = (unsigned long long)s;
    }
    keys[v] = dim == 3 ? (spread3(q[0]) | spread3(q[1]) << 1 | spread3(q[2]) << 2)
                       : (spread2(q[0]) | spread2(q[1]) << 1);
}

// sigma-window key: rows of one window sorted by descending length (stable)
__global__ void k_sigma_key(const int32_t* __restrict__ order0, const int32_t* __restrict__ len, int64_t nv,
                            int sigma, unsigned long long* __restrict__ keys) {
    int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= nv) return;
    int l = len[order0[r]];
    l = l > 255 ? 255 : l;
    keys[r] = ((unsigned long long)(r / sigma) << 8) | (unsigned long long)(255 - l);
}

__global__ void k_invert_perm(const int32_t* __restrict__ perm, int64_t nv, int32_t* __restrict__ iperm) {
    int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r < nv) iperm[perm[r]] = (int32_t)r;
}

// slots of slice c = C * even(max row length in the slice)
__global__ void k_chunk_slots(const int32_t* __restrict__ perm, const int32_t* __restrict__ len, int64_t nv,
                              int64_t n_chunks, int C, int64_t* __restrict__ slots) {
    int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c > n_chunks) return;
    if (c == n_chunks) { slots[c] = 0; return; }
    int w = 0;
    for (int i = 0; i < C; ++i) {
        int64_t r = c * C + i;
        if (r < nv) w = max(w, len[perm[r]]);
    }
    w = (w + 1) & ~1;
    slots[c] = (int64_t)w * C;
}

__global__ void k_sell_fill(const int32_t* __restrict__ perm, const int32_t* __restrict__ iperm,
                            const int64_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                            const double* __restrict__ val, const double* __restrict__ area_u,
                            const double* __restrict__ sdiag_u, const double* __restrict__ gdiag_u,
                            const double* __restrict__ g3_u, const double* __restrict__ g4_u, int64_t nv,
                            int64_t n_chunks, int C, const int64_t* __restrict__ chunk_ptr,
                            int32_t* __restrict__ sell_col, double* __restrict__ sell_val, double* __restrict__ area,
                            double* __restrict__ inv_area, double* __restrict__ sdiag, double* __restrict__ gdiag,
                            double* __restrict__ gdiag3, double* __restrict__ gdiag4) {
    int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_chunks * C) return;
    int64_t c = r / C;
    int64_t w = (chunk_ptr[c + 1] - chunk_ptr[c]) / C;
    int64_t o = chunk_ptr[c] + (r - c * C) * w;
    int64_t k = 0;
    int32_t self = (int32_t)(r < nv ? r : nv - 1);
    if (r < nv) {
        int64_t u = perm[r];
        for (int64_t i = rowptr[u]; i < rowptr[u + 1]; ++i) {
            if (col[i] == u) continue;
            sell_col[o + k] = iperm[col[i]];
            sell_val[o + k] = val[i];
            ++k;
        }
        area[r] = area_u[u];
        inv_area[r] = 1.0 / area_u[u];
        sdiag[r] = sdiag_u[u];
        gdiag[r] = gdiag_u[u];
        gdiag3[r] = g3_u[u];
        gdiag4[r] = g4_u[u];
    }
    for (; k < w; ++k) { sell_col[o + k] = self; sell_val[o + k] = 0.0; }
}


// Per row tile of TILE_ROWS rows (one block each): the sorted, unique out-of-tile columns ("halo", stored with a
// fixed stride of HALO_CAP per tile, unused entries = the tile's first row), the SELL columns rewritten as
// tile-local ids, and a 64-byte descriptor the SpMM kernel prefetches one tile ahead:
//   desc[0..1] first SELL slot of the tile (int64), [2] slots, [3] halo rows or -1 (tile not staged),
//   desc[4..12] slot offset of each SELL slice of the tile relative to the first (TILE_ROWS/C + 1 entries)
constexpr int ECAP = 1024;   // out-of-tile references a tile may have before it is left unstaged
__global__ void __launch_bounds__(128) k_tile_halo(const int64_t* __restrict__ chunk_ptr, const int32_t* __restrict__ col,
                                                   int64_t nv, int log2c, int32_t* __restrict__ halo_n,
                                                   int32_t* __restrict__ halo_rows, int32_t* __restrict__ lcol,
                                                   int32_t* __restrict__ desc) {
    __shared__ int ext[ECAP];
    __shared__ int n_ext, n_uniq;
    const int tid = threadIdx.x;
    const int64_t tile = blockIdx.x;
    const int64_t row0 = tile * TILE_ROWS;
    const int nrows = (int)min((int64_t)TILE_ROWS, nv - row0);
    const int C = 1 << log2c;
    const int64_t ch0 = row0 >> log2c;
    const int nch = (nrows + C - 1) >> log2c;
    const int64_t cp_first = chunk_ptr[ch0];
    const int64_t slots = chunk_ptr[ch0 + nch] - cp_first;
    if (tid == 0) { n_ext = 0; n_uniq = 0; }
    __syncthreads();
    for (int64_t s = tid; s < slots; s += 128) {
        const int64_t c = col[cp_first + s];
        if (c < row0 || c >= row0 + nrows) {
            const int i = atomicAdd(&n_ext, 1);
            if (i < ECAP) ext[i] = (int)c;
        }
    }
    __syncthreads();
    const int ne = n_ext;
    bool over = ne > ECAP;
    if (!over) {
        int np2 = 1;
        while (np2 < ne) np2 <<= 1;
        for (int i = ne + tid; i < np2; i += 128) ext[i] = 0x7fffffff;
        __syncthreads();
        for (int k = 2; k <= np2; k <<= 1)
            for (int j = k >> 1; j > 0; j >>= 1) {
                for (int i = tid; i < np2; i += 128) {
                    const int ixj = i ^ j;
                    if (ixj > i) {
                        const bool up = (i & k) == 0;
                        const int a = ext[i], b = ext[ixj];
                        if ((a > b) == up) { ext[i] = b; ext[ixj] = a; }
                    }
                }
                __syncthreads();
            }
        if (tid == 0) {
            int nu = 0;
            for (int i = 0; i < ne; ++i)
                if (i == 0 || ext[i] != ext[i - 1]) ext[nu++] = ext[i];
            n_uniq = nu;
        }
        __syncthreads();
        over = n_uniq > HALO_CAP;
    }
    const int nu = over ? -1 : n_uniq;
    if (tid == 0) halo_n[tile] = nu;
    if (tid < 16) {
        int v = 0;
        if (tid == 0) v = (int)(cp_first & 0xffffffffll);
        else if (tid == 1) v = (int)(cp_first >> 32);
        else if (tid == 2) v = (int)slots;
        else if (tid == 3) v = nu;
        else if (tid - 4 <= nch) v = (int)(chunk_ptr[ch0 + tid - 4] - cp_first);
        desc[tile * 16 + tid] = v;
    }
    for (int i = tid; i < HALO_CAP; i += 128) halo_rows[tile * HALO_CAP + i] = (nu > 0 && i < nu) ? ext[i] : (int)row0;
    for (int64_t s = tid; s < slots; s += 128) {
        int lc = 0;
        if (nu >= 0) {
            const int64_t c = col[cp_first + s];
            if (c >= row0 && c < row0 + nrows) {
                lc = (int)(c - row0);
            } else {
                int lo = 0, hi = nu - 1;
                while (lo < hi) {
                    const int mid = (lo + hi) >> 1;
                    if (ext[mid] < (int)c) lo = mid + 1; else hi = mid;
                }
                lc = TILE_ROWS + lo;
            }
        }
        lcol[cp_first + s] = lc;
    }
}

inline unsigned grid_for(int64_t n, int block = 256) { return (unsigned)((n + block - 1) / block); }
inline int bits_for(uint64_t n) { int b = 1; while ((1ull << b) < n && b < 63) ++b; return b; }

}  // namespace

int resolve_options(const if_options* in, const Options* base, Options* out) {
    Options o = base ? *base : Options();
    if (in) {
        if (in->gamma != 0.0) o.gamma = in->gamma;
        if (in->tol != 0.0) o.tol = in->tol;
        if (in->max_iter != 0) o.max_iter = in->max_iter;
        if (in->check_every != 0) o.check_every = in->check_every;
        if (in->batch != 0) o.batch = in->batch;
        if (in->solver != 0) o.solver = in->solver;
        if (in->mg_min_ell != 0.0) o.mg_min_ell = in->mg_min_ell;
        if (!base && in->radius != 0.0) o.radius = in->radius;
        if (!base) {   // mesh-layout options are fixed at if_prepare
            if (in->sell_c != 0) o.sell_c = in->sell_c;
            if (in->sell_sigma != 0) o.sell_sigma = in->sell_sigma;
            o.sfc_kind = in->sfc_kind;
            o.flags = in->flags;
        } else {   // per-call flags
            // per-call flags; IF_FLAG_VECTOR per call = "these fields are (u, v) pairs", valid on a handle that has the
            // metric terms (checked in run_job)
            const int per_call = IF_FLAG_HIGHPASS | IF_FLAG_PAIRS | IF_FLAG_VECTOR | IF_FLAG_TRUE_RESIDUAL;
            const bool has_metric = (o.flags & IF_FLAG_VECTOR) != 0;
            o.flags = (o.flags & ~per_call) | (in->flags & per_call);
            if ((o.flags & IF_FLAG_VECTOR) && !has_metric) return IF_EINVAL;
        }
    }
    if (!(o.gamma > 0.0) || !std::isfinite(o.gamma) || !(o.tol > 0.0) || !std::isfinite(o.tol)) return IF_EINVAL;
    if (!(o.radius >= 0.0) || !std::isfinite(o.radius)) return IF_EINVAL;
    if (o.max_iter < 1 || o.check_every < 1) return IF_EINVAL;
    if (o.batch != 4 && o.batch != 8 && o.batch != 16) return IF_EINVAL;
    if ((o.sell_c != 32 && o.sell_c != 64 && o.sell_c != 128) || TILE_ROWS % o.sell_c != 0) return IF_EINVAL;   // must divide the SpMM row tile
    if (o.sell_sigma < o.sell_c || o.sell_sigma % o.sell_c != 0) return IF_EINVAL;
    if (o.sfc_kind != 0 && o.sfc_kind != 1) return IF_EINVAL;
    if (o.solver == 2) o.solver = 0;   // 2 = Jacobi-PCG explicitly (a per-call 0 inherits the handle's choice)
    if ((o.solver != 0 && o.solver != 1) || !(o.mg_min_ell >= 0.0) || !std::isfinite(o.mg_min_ell)) return IF_EINVAL;
    *out = o;
    return IF_OK;
}

}  // namespace ifl

using namespace ifl;

extern "C" void if_destroy(if_handle h) {
    if (!h) return;
    int prev = 0;
    cudaGetDevice(&prev);
    cudaSetDevice(h->device);
    cudaFree(h->chunk_ptr); cudaFree(h->sell_col); cudaFree(h->sell_val); cudaFree(h->area);
    cudaFree(h->inv_area); cudaFree(h->sdiag); cudaFree(h->gdiag); cudaFree(h->gdiag3); cudaFree(h->gdiag4);
    cudaFree(h->sell_dval); cudaFree(h->sell_tval); cudaFree(h->ddiag); cudaFree(h->gdiag_vec); cudaFree(h->perm); cudaFree(h->iperm);
    cudaFree(h->sell_lcol); cudaFree(h->halo_n); cudaFree(h->tile_desc); cudaFree(h->halo_rows);
    ifl::mg_free(h);
    cudaFree(h->csr_rowptr); cudaFree(h->csr_col); cudaFree(h->csr_val); cudaFree(h->csr_area);
    if (h->h_pinned) cudaFreeHost(h->h_pinned);
    cudaSetDevice(prev);
    delete h;
}

static int prepare_impl(const double* coords, int dim, int64_t nv, const int32_t* tri, int64_t nt,
                        const double* period, const Options& opt, if_mesh_s* h) {
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return IF_ECUDA;
    IF_CUDA_TRY(cudaGetDevice(&h->device));
    IF_CUDA_TRY(cudaDeviceGetAttribute(&h->n_sm, cudaDevAttrMultiProcessorCount, h->device));
    h->n_vert = nv;
    h->opt = opt;
    h->sell_c = opt.sell_c;
    cudaStream_t st = 0;

    Period per{{0.0, 0.0, 0.0}};
    if (period)
        for (int d = 0; d < dim; ++d) {
            if (!(period[d] >= 0.0) || !std::isfinite(period[d])) return IF_EINVAL;
            per.p[d] = period[d];
        }
    // bounding box for the space-filling curve (host pass over the caller's coordinates)
    Box box;
    for (int d = 0; d < 3; ++d) { box.lo[d] = 0.0; box.scale[d] = 0.0; }
    {
        double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
        for (int64_t v = 0; v < nv; ++v)
            for (int d = 0; d < dim; ++d) {
                double x = coords[v * dim + d];
                if (!std::isfinite(x)) return IF_EINVAL;
                lo[d] = x < lo[d] ? x : lo[d];
                hi[d] = x > hi[d] ? x : hi[d];
            }
        double ext = 0.0;
        for (int d = 0; d < dim; ++d) ext = hi[d] - lo[d] > ext ? hi[d] - lo[d] : ext;
        for (int d = 0; d < dim; ++d) { box.lo[d] = lo[d]; box.scale[d] = ext > 0.0 ? 1.0 / ext : 0.0; }
    }

    DevBuf d_coords, d_tri, d_flags;
    IF_CUDA_TRY(d_coords.alloc((size_t)nv * dim * sizeof(double)));
    IF_CUDA_TRY(d_tri.alloc((size_t)nt * 3 * sizeof(int32_t)));
    IF_CUDA_TRY(d_flags.alloc(sizeof(int)));
    IF_CUDA_TRY(cudaMemcpyAsync(d_coords.p, coords, (size_t)nv * dim * sizeof(double), cudaMemcpyHostToDevice, st));
    IF_CUDA_TRY(cudaMemcpyAsync(d_tri.p, tri, (size_t)nt * 3 * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    IF_CUDA_TRY(cudaMemsetAsync(d_flags.p, 0, sizeof(int), st));

    // ---- P1/P2: emit, sort by (row, col), sum by key
    const int64_t n_emit = 9 * nt;
    DevBuf k0, k1, v0, v1, tmp, d_nruns;
    IF_CUDA_TRY(k0.alloc((size_t)n_emit * 8));
    IF_CUDA_TRY(k1.alloc((size_t)n_emit * 8));
    IF_CUDA_TRY(v0.alloc((size_t)n_emit * 8));
    IF_CUDA_TRY(v1.alloc((size_t)n_emit * 8));
    IF_CUDA_TRY(d_nruns.alloc(sizeof(int64_t)));
    k_tri_emit<<<grid_for(nt), 256, 0, st>>>(d_coords.as<double>(), dim, nv, d_tri.as<int32_t>(), nt, per,
                                            k0.as<unsigned long long>(), v0.as<double>(), d_flags.as<int>());
    IF_LAUNCH_CHECK();
    int flags = 0;
    IF_CUDA_TRY(cudaMemcpyAsync(&flags, d_flags.p, sizeof(int), cudaMemcpyDeviceToHost, st));
    IF_CUDA_TRY(cudaStreamSynchronize(st));
    if (flags & FLAG_INDEX) return IF_EINDEX;
    if (flags & FLAG_DEGENERATE) return IF_EDEGENERATE;

    const int key_bits = 32 + bits_for((uint64_t)nv);
    size_t tb = 0;
    IF_CUDA_TRY(cub::DeviceRadixSort::SortPairs(nullptr, tb, k0.as<unsigned long long>(), k1.as<unsigned long long>(),
                                                v0.as<double>(), v1.as<double>(), n_emit, 0, key_bits, st));
    IF_CUDA_TRY(tmp.alloc(tb));
    IF_CUDA_TRY(cub::DeviceRadixSort::SortPairs(tmp.p, tb, k0.as<unsigned long long>(), k1.as<unsigned long long>(),
                                                v0.as<double>(), v1.as<double>(), n_emit, 0, key_bits, st));
    ++g_launches;
    tb = 0;
    IF_CUDA_TRY(cub::DeviceReduce::ReduceByKey(nullptr, tb, k1.as<unsigned long long>(), k0.as<unsigned long long>(),
                                               v1.as<double>(), v0.as<double>(), d_nruns.as<int64_t>(), cub::Sum(),
                                               n_emit, st));
    IF_CUDA_TRY(tmp.alloc(tb));
    IF_CUDA_TRY(cub::DeviceReduce::ReduceByKey(tmp.p, tb, k1.as<unsigned long long>(), k0.as<unsigned long long>(),
                                               v1.as<double>(), v0.as<double>(), d_nruns.as<int64_t>(), cub::Sum(),
                                               n_emit, st));
    ++g_launches;
    int64_t nnz = 0;
    IF_CUDA_TRY(cudaMemcpyAsync(&nnz, d_nruns.p, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
    IF_CUDA_TRY(cudaStreamSynchronize(st));
    h->nnz = nnz;
    k1.alloc(0); v1.alloc(0);   // sorted copies no longer needed
    // now: k0 = unique keys [nnz], v0 = summed values [nnz]

    // ---- CSR in the caller's numbering, A_v, S_vv, g_v
    DevBuf rowptr, ccol, area_u, sdiag_u, gdiag_u, g3_u, g4_u, len;
    IF_CUDA_TRY(rowptr.alloc((size_t)(nv + 1) * sizeof(int64_t)));
    IF_CUDA_TRY(ccol.alloc((size_t)nnz * sizeof(int32_t)));
    IF_CUDA_TRY(area_u.alloc((size_t)nv * 8));
    IF_CUDA_TRY(sdiag_u.alloc((size_t)nv * 8));
    IF_CUDA_TRY(gdiag_u.alloc((size_t)nv * 8));
    IF_CUDA_TRY(g3_u.alloc((size_t)nv * 8));
    IF_CUDA_TRY(g4_u.alloc((size_t)nv * 8));
    IF_CUDA_TRY(len.alloc((size_t)nv * 4));
    k_rowptr<<<grid_for(nnz + 1), 256, 0, st>>>(k0.as<unsigned long long>(), nnz, nv, rowptr.as<int64_t>());
    IF_LAUNCH_CHECK();
    k_row_finish<<<grid_for(nv), 256, 0, st>>>(k0.as<unsigned long long>(), rowptr.as<int64_t>(), nv, v0.as<double>(),
                                              ccol.as<int32_t>(), area_u.as<double>(), sdiag_u.as<double>(),
                                              len.as<int32_t>(), d_flags.as<int>());
    IF_LAUNCH_CHECK();
    IF_CUDA_TRY(cudaMemcpyAsync(&flags, d_flags.p, sizeof(int), cudaMemcpyDeviceToHost, st));
    IF_CUDA_TRY(cudaStreamSynchronize(st));
    if (flags & FLAG_ORPHAN) return IF_EORPHAN;
    k_gdiag<<<grid_for(nv), 256, 0, st>>>(rowptr.as<int64_t>(), ccol.as<int32_t>(), v0.as<double>(),
                                         area_u.as<double>(), nv, gdiag_u.as<double>());
    IF_LAUNCH_CHECK();
    k_gdiag_higher<<<grid_for(nv, 128), 128, 0, st>>>(rowptr.as<int64_t>(), ccol.as<int32_t>(), v0.as<double>(),
                                                      area_u.as<double>(), nv, g3_u.as<double>(), g4_u.as<double>());
    IF_LAUNCH_CHECK();

    // total area and mean edge length (deterministic device reductions)
    {
        DevBuf d_sum, elen;
        IF_CUDA_TRY(d_sum.alloc(2 * sizeof(double)));
        IF_CUDA_TRY(elen.alloc((size_t)nnz * 8));
        k_edge_len<<<grid_for(nv), 256, 0, st>>>(d_coords.as<double>(), dim, per, rowptr.as<int64_t>(),
                                                ccol.as<int32_t>(), nv, elen.as<double>());
        IF_LAUNCH_CHECK();
        tb = 0;
        IF_CUDA_TRY(cub::DeviceReduce::Sum(nullptr, tb, elen.as<double>(), d_sum.as<double>(), nnz, st));
        IF_CUDA_TRY(tmp.alloc(tb));
        IF_CUDA_TRY(cub::DeviceReduce::Sum(tmp.p, tb, area_u.as<double>(), d_sum.as<double>(), nv, st));
        IF_CUDA_TRY(cub::DeviceReduce::Sum(tmp.p, tb, elen.as<double>(), d_sum.as<double>() + 1, nnz, st));
        g_launches += 2;
        double s[2] = {0.0, 0.0};
        IF_CUDA_TRY(cudaMemcpyAsync(s, d_sum.p, sizeof(s), cudaMemcpyDeviceToHost, st));
        IF_CUDA_TRY(cudaStreamSynchronize(st));
        h->total_area = s[0];
        int64_t n_edges = (nnz - nv) / 2;
        h->mean_edge = n_edges > 0 ? s[1] / (double)n_edges : 0.0;
    }

    // ---- P4: space-filling-curve order; P5: sigma-window sort by row length
    DevBuf mk0, mk1, id0, id1, perm, iperm;
    IF_CUDA_TRY(mk0.alloc((size_t)nv * 8));
    IF_CUDA_TRY(mk1.alloc((size_t)nv * 8));
    IF_CUDA_TRY(id0.alloc((size_t)nv * 4));
    IF_CUDA_TRY(id1.alloc((size_t)nv * 4));
    IF_CUDA_TRY(perm.alloc((size_t)nv * 4));
    IF_CUDA_TRY(iperm.alloc((size_t)nv * 4));
    k_morton<<<grid_for(nv), 256, 0, st>>>(d_coords.as<double>(), dim, nv, box, mk0.as<unsigned long long>(),
                                          id0.as<int32_t>(), opt.sfc_kind == 1);
    IF_LAUNCH_CHECK();
    tb = 0;
    IF_CUDA_TRY(cub::DeviceRadixSort::SortPairs(nullptr, tb, mk0.as<unsigned long long>(), mk1.as<unsigned long long>(),
                                                id0.as<int32_t>(), id1.as<int32_t>(), nv, 0, 64, st));
    IF_CUDA_TRY(tmp.alloc(tb));
    IF_CUDA_TRY(cub::DeviceRadixSort::SortPairs(tmp.p, tb, mk0.as<unsigned long long>(), mk1.as<unsigned long long>(),
                                                id0.as<int32_t>(), id1.as<int32_t>(), nv, 0, 64, st));
    ++g_launches;
    // id1 = SFC order (rank -> caller id)
    if (opt.sell_sigma > opt.sell_c) {
        k_sigma_key<<<grid_for(nv), 256, 0, st>>>(id1.as<int32_t>(), len.as<int32_t>(), nv, opt.sell_sigma,
                                                 mk0.as<unsigned long long>());
        IF_LAUNCH_CHECK();
        const int sb = 8 + bits_for((uint64_t)(nv / opt.sell_sigma + 1));
        IF_CUDA_TRY(cub::DeviceRadixSort::SortPairs(tmp.p, tb, mk0.as<unsigned long long>(),
                                                    mk1.as<unsigned long long>(), id1.as<int32_t>(),
                                                    perm.as<int32_t>(), nv, 0, sb, st));
        ++g_launches;
    } else {
        IF_CUDA_TRY(cudaMemcpyAsync(perm.p, id1.p, (size_t)nv * 4, cudaMemcpyDeviceToDevice, st));
    }
    k_invert_perm<<<grid_for(nv), 256, 0, st>>>(perm.as<int32_t>(), nv, iperm.as<int32_t>());
    IF_LAUNCH_CHECK();

    const int C = opt.sell_c;
    const int64_t n_chunks = (nv + C - 1) / C;
    h->n_chunks = n_chunks;
    DevBuf slots, chunk_ptr;
    IF_CUDA_TRY(slots.alloc((size_t)(n_chunks + 1) * 8));
    IF_CUDA_TRY(chunk_ptr.alloc((size_t)(n_chunks + 1) * 8));
    k_chunk_slots<<<grid_for(n_chunks + 1), 256, 0, st>>>(perm.as<int32_t>(), len.as<int32_t>(), nv, n_chunks, C,
                                                         slots.as<int64_t>());
    IF_LAUNCH_CHECK();
    tb = 0;
    IF_CUDA_TRY(cub::DeviceScan::ExclusiveSum(nullptr, tb, slots.as<int64_t>(), chunk_ptr.as<int64_t>(),
                                              n_chunks + 1, st));
    IF_CUDA_TRY(tmp.alloc(tb));
    IF_CUDA_TRY(cub::DeviceScan::ExclusiveSum(tmp.p, tb, slots.as<int64_t>(), chunk_ptr.as<int64_t>(), n_chunks + 1,
                                              st));
    ++g_launches;
    int64_t sell_slots = 0;
    IF_CUDA_TRY(cudaMemcpyAsync(&sell_slots, chunk_ptr.as<int64_t>() + n_chunks, 8, cudaMemcpyDeviceToHost, st));
    IF_CUDA_TRY(cudaStreamSynchronize(st));
    h->sell_slots = sell_slots;

    DevBuf scol, sval, area, inv_area, sdiag, gdiag, gdiag3, gdiag4;
    IF_CUDA_TRY(scol.alloc((size_t)sell_slots * 4 + 16));
    IF_CUDA_TRY(sval.alloc((size_t)sell_slots * 8 + 16));
    IF_CUDA_TRY(area.alloc((size_t)nv * 8 + 16));   // +16: the SpMM kernel bulk-copies 16-byte multiples
    IF_CUDA_TRY(cudaMemsetAsync(area.p, 0, (size_t)nv * 8 + 16, st));
    IF_CUDA_TRY(inv_area.alloc((size_t)nv * 8 + 16));   // +16: the SpMM kernel bulk-copies 16-byte multiples
    IF_CUDA_TRY(cudaMemsetAsync(inv_area.p, 0, (size_t)nv * 8 + 16, st));
    IF_CUDA_TRY(sdiag.alloc((size_t)nv * 8 + 16));   // +16: the SpMM kernel bulk-copies 16-byte multiples
    IF_CUDA_TRY(cudaMemsetAsync(sdiag.p, 0, (size_t)nv * 8 + 16, st));
    IF_CUDA_TRY(gdiag.alloc((size_t)nv * 8 + 16));   // +16: the SpMM kernel bulk-copies 16-byte multiples
    IF_CUDA_TRY(cudaMemsetAsync(gdiag.p, 0, (size_t)nv * 8 + 16, st));
    IF_CUDA_TRY(gdiag3.alloc((size_t)nv * 8 + 16));
    IF_CUDA_TRY(cudaMemsetAsync(gdiag3.p, 0, (size_t)nv * 8 + 16, st));
    IF_CUDA_TRY(gdiag4.alloc((size_t)nv * 8 + 16));
    IF_CUDA_TRY(cudaMemsetAsync(gdiag4.p, 0, (size_t)nv * 8 + 16, st));
    k_sell_fill<<<grid_for(n_chunks * C), 256, 0, st>>>(
        perm.as<int32_t>(), iperm.as<int32_t>(), rowptr.as<int64_t>(), ccol.as<int32_t>(), v0.as<double>(),
        area_u.as<double>(), sdiag_u.as<double>(), gdiag_u.as<double>(), g3_u.as<double>(), g4_u.as<double>(), nv,
        n_chunks, C, chunk_ptr.as<int64_t>(), scol.as<int32_t>(), sval.as<double>(), area.as<double>(),
        inv_area.as<double>(), sdiag.as<double>(), gdiag.as<double>(), gdiag3.as<double>(), gdiag4.as<double>());
    IF_LAUNCH_CHECK();
    IF_CUDA_TRY(cudaStreamSynchronize(st));

    // ---- vector filter: metric terms (D~, T) on the slots of S
    if (opt.flags & IF_FLAG_VECTOR) {
        double radius = 0.0;
        if (dim == 3) {
            radius = opt.radius;
            if (radius == 0.0) {           // mean |x_v| (host pass, like the bounding box)
                double sum = 0.0;
                for (int64_t v = 0; v < nv; ++v)
                    sum += std::sqrt(coords[3 * v] * coords[3 * v] + coords[3 * v + 1] * coords[3 * v + 1] +
                                     coords[3 * v + 2] * coords[3 * v + 2]);
                radius = sum / (double)nv;
            }
            if (!(radius > 0.0)) return IF_EINVAL;
        }
        h->radius = radius;
        DevBuf ek, ev, ek1, ev1, uk, uv, d_n;
        IF_CUDA_TRY(ek.alloc((size_t)n_emit * 8));
        IF_CUDA_TRY(ev.alloc((size_t)n_emit * 16));
        IF_CUDA_TRY(ek1.alloc((size_t)n_emit * 8));
        IF_CUDA_TRY(ev1.alloc((size_t)n_emit * 16));
        k_tri_emit_vec<<<grid_for(nt), 256, 0, st>>>(d_coords.as<double>(), dim, d_tri.as<int32_t>(), nt, per,
                                                    radius > 0.0 ? 1.0 / radius : 0.0, ek.as<unsigned long long>(),
                                                    ev.as<double2>());
        IF_LAUNCH_CHECK();
        tb = 0;
        IF_CUDA_TRY(cub::DeviceRadixSort::SortPairs(nullptr, tb, ek.as<unsigned long long>(), ek1.as<unsigned long long>(),
                                                    ev.as<double2>(), ev1.as<double2>(), n_emit, 0, key_bits, st));
        IF_CUDA_TRY(tmp.alloc(tb));
        IF_CUDA_TRY(cub::DeviceRadixSort::SortPairs(tmp.p, tb, ek.as<unsigned long long>(), ek1.as<unsigned long long>(),
                                                    ev.as<double2>(), ev1.as<double2>(), n_emit, 0, key_bits, st));
        ++g_launches;
        ek.alloc(0); ev.alloc(0);
        IF_CUDA_TRY(uk.alloc((size_t)n_emit * 8));
        IF_CUDA_TRY(uv.alloc((size_t)n_emit * 16));
        IF_CUDA_TRY(d_n.alloc(sizeof(int64_t)));
        tb = 0;
        IF_CUDA_TRY(cub::DeviceReduce::ReduceByKey(nullptr, tb, ek1.as<unsigned long long>(), uk.as<unsigned long long>(),
                                                   ev1.as<double2>(), uv.as<double2>(), d_n.as<int64_t>(), Add2v(), n_emit, st));
        IF_CUDA_TRY(tmp.alloc(tb));
        IF_CUDA_TRY(cub::DeviceReduce::ReduceByKey(tmp.p, tb, ek1.as<unsigned long long>(), uk.as<unsigned long long>(),
                                                   ev1.as<double2>(), uv.as<double2>(), d_n.as<int64_t>(), Add2v(), n_emit, st));
        ++g_launches;
        int64_t n_u = 0;
        IF_CUDA_TRY(cudaMemcpyAsync(&n_u, d_n.p, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
        IF_CUDA_TRY(cudaStreamSynchronize(st));
        if (n_u != nnz) return IF_ECUDA;      // cannot happen: the keys are those of the stiffness assembly
        DevBuf dval, tval, ddiag, gvec;
        IF_CUDA_TRY(dval.alloc((size_t)sell_slots * 8 + 16));
        IF_CUDA_TRY(tval.alloc((size_t)sell_slots * 8 + 16));
        IF_CUDA_TRY(ddiag.alloc((size_t)nv * 8 + 16));
        IF_CUDA_TRY(cudaMemsetAsync(ddiag.p, 0, (size_t)nv * 8 + 16, st));
        IF_CUDA_TRY(gvec.alloc((size_t)nv * 8 + 16));
        IF_CUDA_TRY(cudaMemsetAsync(gvec.p, 0, (size_t)nv * 8 + 16, st));
        k_sell_fill_vec<<<grid_for(n_chunks * C), 256, 0, st>>>(perm.as<int32_t>(), rowptr.as<int64_t>(), ccol.as<int32_t>(),
                                                               uv.as<double2>(), area_u.as<double>(), nv, n_chunks, C,
                                                               chunk_ptr.as<int64_t>(), dval.as<double>(), tval.as<double>(),
                                                               ddiag.as<double>(), gvec.as<double>());
        IF_LAUNCH_CHECK();
        IF_CUDA_TRY(cudaStreamSynchronize(st));
        h->sell_dval = (double*)dval.release();
        h->sell_tval = (double*)tval.release();
        h->ddiag = (double*)ddiag.release();
        h->gdiag_vec = (double*)gvec.release();
    }

    // ---- row tiles of the SpMM kernel: halo lists and tile-local column ids
    const int64_t n_tiles = (nv + TILE_ROWS - 1) / TILE_ROWS;
    h->n_tiles = n_tiles;
    int log2c = 0;
    while ((1 << log2c) < C) ++log2c;
    DevBuf halo_n, halo_rows, lcol, tile_desc;
    IF_CUDA_TRY(halo_n.alloc((size_t)n_tiles * 4));
    IF_CUDA_TRY(halo_rows.alloc((size_t)n_tiles * HALO_CAP * 4));
    IF_CUDA_TRY(tile_desc.alloc((size_t)(n_tiles + 1) * 64));
    IF_CUDA_TRY(cudaMemsetAsync(tile_desc.p, 0, (size_t)(n_tiles + 1) * 64, st));
    IF_CUDA_TRY(lcol.alloc((size_t)sell_slots * 4 + 16));
    k_tile_halo<<<(unsigned)n_tiles, 128, 0, st>>>(chunk_ptr.as<int64_t>(), scol.as<int32_t>(), nv, log2c,
                                                   halo_n.as<int32_t>(), halo_rows.as<int32_t>(), lcol.as<int32_t>(),
                                                   tile_desc.as<int32_t>());
    IF_LAUNCH_CHECK();
    IF_CUDA_TRY(cudaStreamSynchronize(st));
    {
        std::vector<int32_t> hn((size_t)n_tiles);
        IF_CUDA_TRY(cudaMemcpy(hn.data(), halo_n.p, (size_t)n_tiles * 4, cudaMemcpyDeviceToHost));
        h->unstaged_tiles = 0;
        h->halo_max = 0;
        h->halo_total = 0;
        for (int32_t v : hn) {
            if (v < 0) { ++h->unstaged_tiles; continue; }
            h->halo_total += v;
            if (v > h->halo_max) h->halo_max = v;
        }
    }
    h->sell_lcol = (int32_t*)lcol.release();
    h->halo_n = (int32_t*)halo_n.release();
    h->tile_desc = (int32_t*)tile_desc.release();
    h->halo_rows = (int32_t*)halo_rows.release();

    if (opt.flags & IF_FLAG_KEEP_CSR) {
        // v0 holds [9 n_tri] doubles; keep a right-sized copy instead
        DevBuf cval;
        IF_CUDA_TRY(cval.alloc((size_t)nnz * 8));
        IF_CUDA_TRY(cudaMemcpy(cval.p, v0.p, (size_t)nnz * 8, cudaMemcpyDeviceToDevice));
        h->csr_rowptr = (int64_t*)rowptr.release();
        h->csr_col = (int32_t*)ccol.release();
        h->csr_val = (double*)cval.release();
        h->csr_area = (double*)area_u.release();
    }
    h->chunk_ptr = (int64_t*)chunk_ptr.release();
    h->sell_col = (int32_t*)scol.release();
    h->sell_val = (double*)sval.release();
    h->area = (double*)area.release();
    h->inv_area = (double*)inv_area.release();
    h->sdiag = (double*)sdiag.release();
    h->gdiag = (double*)gdiag.release();
    h->gdiag3 = (double*)gdiag3.release();
    h->gdiag4 = (double*)gdiag4.release();
    h->perm = (int32_t*)perm.release();
    h->iperm = (int32_t*)iperm.release();

    h->h_pinned_bytes = 1 << 20;
    IF_CUDA_TRY(cudaHostAlloc(&h->h_pinned, h->h_pinned_bytes, cudaHostAllocDefault));
    if (opt.flags & IF_FLAG_MULTIGRID) {
        int rc = mg_build(h);
        if (rc != IF_OK) return rc;
    }
    return IF_OK;
}

extern "C" int if_prepare(const double* coords, int dim, int64_t n_vert, const int32_t* tri, int64_t n_tri,
                          const double* period, const if_options* opt, if_handle* out) {
    if (!coords || !tri || !out || (dim != 2 && dim != 3) || n_vert < 3 || n_tri < 1) return IF_EINVAL;
    if (n_vert > 0x7fffffffLL || n_tri > 0x7fffffffLL / 9) return IF_EINVAL;
    Options o;
    int rc = resolve_options(opt, nullptr, &o);
    if (rc != IF_OK) return rc;
    if_mesh_s* h = new (std::nothrow) if_mesh_s();
    if (!h) return IF_ENOMEM;
    rc = prepare_impl(coords, dim, n_vert, tri, n_tri, period, o, h);
    if (rc == IF_OK) rc = ifl::na_setup(h);
    if (rc != IF_OK) {
        if_destroy(h);
        return rc;
    }
    *out = h;
    return IF_OK;
}

extern "C" int if_mesh_info(if_handle h, int64_t* n_vert, int64_t* nnz, double* total_area, double* mean_edge,
                            int64_t* sell_slots) {
    if (!h) return IF_EINVAL;
    if (n_vert) *n_vert = h->n_vert;
    if (nnz) *nnz = h->nnz;
    if (total_area) *total_area = h->total_area;
    if (mean_edge) *mean_edge = h->mean_edge;
    if (sell_slots) *sell_slots = h->sell_slots;
    return IF_OK;
}

extern "C" int if_mesh_tile_info(if_handle h, int64_t* n_tiles, int64_t* halo_rows, int64_t* halo_max,
                                 int64_t* unstaged_tiles) {
    if (!h) return IF_EINVAL;
    if (n_tiles) *n_tiles = h->n_tiles;
    if (halo_rows) *halo_rows = h->halo_total;
    if (halo_max) *halo_max = h->halo_max;
    if (unstaged_tiles) *unstaged_tiles = h->unstaged_tiles;
    return IF_OK;
}

extern "C" int if_mesh_export_csr(if_handle h, int64_t* rowptr, int32_t* col, double* val, double* area) {
    if (!h || !h->csr_rowptr) return IF_EINVAL;
    IF_CUDA_TRY(cudaSetDevice(h->device));
    if (rowptr) IF_CUDA_TRY(cudaMemcpy(rowptr, h->csr_rowptr, (size_t)(h->n_vert + 1) * 8, cudaMemcpyDeviceToHost));
    if (col) IF_CUDA_TRY(cudaMemcpy(col, h->csr_col, (size_t)h->nnz * 4, cudaMemcpyDeviceToHost));
    if (val) IF_CUDA_TRY(cudaMemcpy(val, h->csr_val, (size_t)h->nnz * 8, cudaMemcpyDeviceToHost));
    if (area) IF_CUDA_TRY(cudaMemcpy(area, h->csr_area, (size_t)h->n_vert * 8, cudaMemcpyDeviceToHost));
    return IF_OK;
}

extern "C" int if_mesh_export_perm(if_handle h, int32_t* perm) {
    if (!h) return IF_EINVAL;
    IF_CUDA_TRY(cudaSetDevice(h->device));
    if (perm) IF_CUDA_TRY(cudaMemcpy(perm, h->perm, (size_t)h->n_vert * 4, cudaMemcpyDeviceToHost));
    return IF_OK;
}

// ------------------------------------------------------------------------------------------- save / load
namespace {
struct FileHeader {
    char magic[8];            // "IFMESH02"
    int32_t tile_rows, halo_cap, sell_c, pad_;
    int64_t n_vert, nnz, n_chunks, sell_slots, n_tiles, halo_total, halo_max, unstaged_tiles;
    double total_area, mean_edge;
    ifl::Options opt;
};

struct LevelHeader {          // one multigrid level in the file
    int64_t n, nnz, n_coarse, p_nnz;
    double rho, rho_m, omega;
};

int write_dev(FILE* f, const void* d, size_t bytes, std::vector<char>& buf) {
    buf.resize(bytes);
    if (bytes) IF_CUDA_TRY(cudaMemcpy(buf.data(), d, bytes, cudaMemcpyDeviceToHost));
    return fwrite(buf.data(), 1, bytes, f) == bytes ? IF_OK : IF_EIO;
}
int read_dev(FILE* f, void** d, size_t bytes, size_t alloc_bytes, std::vector<char>& buf) {
    buf.resize(bytes);
    if (fread(buf.data(), 1, bytes, f) != bytes) return IF_EIO;
    IF_CUDA_TRY(cudaMalloc(d, alloc_bytes ? alloc_bytes : 1));
    IF_CUDA_TRY(cudaMemset(*d, 0, alloc_bytes ? alloc_bytes : 1));
    if (bytes) IF_CUDA_TRY(cudaMemcpy(*d, buf.data(), bytes, cudaMemcpyHostToDevice));
    return IF_OK;
}
}  // namespace

extern "C" int if_save(if_handle h, const char* path) {
    if (!h || !path) return IF_EINVAL;
    IF_CUDA_TRY(cudaSetDevice(h->device));
    FILE* f = fopen(path, "wb");
    if (!f) return IF_EIO;
    FileHeader hd;
    memset(&hd, 0, sizeof(hd));
    memcpy(hd.magic, "IFMESH02", 8);
    hd.tile_rows = TILE_ROWS; hd.halo_cap = HALO_CAP; hd.sell_c = h->sell_c;
    hd.pad_ = (int32_t)sizeof(ifl::Options);   // the options are stored raw: their layout is part of the format
    hd.n_vert = h->n_vert; hd.nnz = h->nnz; hd.n_chunks = h->n_chunks; hd.sell_slots = h->sell_slots;
    hd.n_tiles = h->n_tiles; hd.halo_total = h->halo_total; hd.halo_max = h->halo_max;
    hd.unstaged_tiles = h->unstaged_tiles; hd.total_area = h->total_area; hd.mean_edge = h->mean_edge;
    hd.opt = h->opt;
    hd.opt.radius = h->radius;     // the radius actually used
    hd.opt.flags &= ~(IF_FLAG_KEEP_CSR | IF_FLAG_HIGHPASS | IF_FLAG_PAIRS | IF_FLAG_TRUE_RESIDUAL);
    std::vector<char> buf;
    const size_t nv = (size_t)h->n_vert, ns = (size_t)h->sell_slots, nt = (size_t)h->n_tiles;
    int rc = fwrite(&hd, sizeof(hd), 1, f) == 1 ? IF_OK : IF_EIO;
    if (rc == IF_OK) rc = write_dev(f, h->chunk_ptr, (size_t)(h->n_chunks + 1) * 8, buf);
    if (rc == IF_OK) rc = write_dev(f, h->sell_col, ns * 4, buf);
    if (rc == IF_OK) rc = write_dev(f, h->sell_val, ns * 8, buf);
    if (rc == IF_OK) rc = write_dev(f, h->sell_lcol, ns * 4, buf);
    if (rc == IF_OK) rc = write_dev(f, h->area, nv * 8, buf);
    if (rc == IF_OK) rc = write_dev(f, h->inv_area, nv * 8, buf);
    if (rc == IF_OK) rc = write_dev(f, h->sdiag, nv * 8, buf);
    if (rc == IF_OK) rc = write_dev(f, h->gdiag, nv * 8, buf);
    if (rc == IF_OK) rc = write_dev(f, h->gdiag3, nv * 8, buf);
    if (rc == IF_OK) rc = write_dev(f, h->gdiag4, nv * 8, buf);
    if (h->opt.flags & IF_FLAG_VECTOR) {      // metric terms of the vector filter
        if (rc == IF_OK) rc = write_dev(f, h->sell_dval, ns * 8, buf);
        if (rc == IF_OK) rc = write_dev(f, h->sell_tval, ns * 8, buf);
        if (rc == IF_OK) rc = write_dev(f, h->ddiag, nv * 8, buf);
        if (rc == IF_OK) rc = write_dev(f, h->gdiag_vec, nv * 8, buf);
    }
    if (rc == IF_OK) rc = write_dev(f, h->perm, nv * 4, buf);
    if (rc == IF_OK) rc = write_dev(f, h->iperm, nv * 4, buf);
    if (rc == IF_OK) rc = write_dev(f, h->halo_n, nt * 4, buf);
    if (rc == IF_OK) rc = write_dev(f, h->halo_rows, nt * HALO_CAP * 4, buf);
    if (rc == IF_OK) rc = write_dev(f, h->tile_desc, (nt + 1) * 64, buf);
    // the multigrid hierarchy (IF_FLAG_MULTIGRID): level count, then per level its header, the (S, M) pair and the
    // transfer operators to the next level
    if (rc == IF_OK && (h->opt.flags & IF_FLAG_MULTIGRID)) {
        const int64_t L = h->mg_levels;
        rc = fwrite(&L, sizeof(L), 1, f) == 1 ? IF_OK : IF_EIO;
        for (int l = 0; l < h->mg_levels && rc == IF_OK; ++l) {
            const ifl::MgLevel& g = h->mg[l];
            LevelHeader lh{g.n, g.nnz, g.n_coarse, g.p_nnz, g.rho, g.rho_m, g.omega};
            rc = fwrite(&lh, sizeof(lh), 1, f) == 1 ? IF_OK : IF_EIO;
            if (rc == IF_OK) rc = write_dev(f, g.rowptr, (size_t)(g.n + 1) * 8, buf);
            if (rc == IF_OK) rc = write_dev(f, g.col, (size_t)g.nnz * 4, buf);
            if (rc == IF_OK) rc = write_dev(f, g.sm, (size_t)g.nnz * 16, buf);
            if (rc == IF_OK) rc = write_dev(f, g.diag, (size_t)g.n * 16, buf);
            if (l + 1 < h->mg_levels) {
                if (rc == IF_OK) rc = write_dev(f, g.p_rowptr, (size_t)(g.n + 1) * 8, buf);
                if (rc == IF_OK) rc = write_dev(f, g.p_col, (size_t)g.p_nnz * 4, buf);
                if (rc == IF_OK) rc = write_dev(f, g.p_val, (size_t)g.p_nnz * 8, buf);
                if (rc == IF_OK) rc = write_dev(f, g.r_rowptr, (size_t)(g.n_coarse + 1) * 8, buf);
                if (rc == IF_OK) rc = write_dev(f, g.r_col, (size_t)g.p_nnz * 4, buf);
                if (rc == IF_OK) rc = write_dev(f, g.r_val, (size_t)g.p_nnz * 8, buf);
            }
        }
    }
    if (fclose(f) != 0 && rc == IF_OK) rc = IF_EIO;
    return rc;
}

extern "C" int if_load(const char* path, if_handle* out) {
    if (!path || !out) return IF_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return IF_ECUDA; }
    FILE* f = fopen(path, "rb");
    if (!f) return IF_EIO;
    FileHeader hd;
    if (fread(&hd, sizeof(hd), 1, f) != 1 || memcmp(hd.magic, "IFMESH02", 8) != 0 || hd.tile_rows != TILE_ROWS ||
        hd.halo_cap != HALO_CAP || hd.n_vert < 3 || hd.sell_slots < 0 || hd.n_tiles != (hd.n_vert + TILE_ROWS - 1) / TILE_ROWS) {
        fclose(f);
        return IF_EIO;
    }
    {
        // the header is not trusted: sizes must fit each other, the library's allowed values and the file's length
        ifl::Options chk;
        bool ok = hd.pad_ == (int32_t)sizeof(ifl::Options) && (hd.sell_c == 32 || hd.sell_c == 64 || hd.sell_c == 128) &&
                  TILE_ROWS % hd.sell_c == 0 && hd.n_vert <= 0x7fffffffLL &&
                  hd.n_chunks == (hd.n_vert + hd.sell_c - 1) / hd.sell_c && hd.nnz >= hd.n_vert &&
                  hd.sell_slots >= hd.nnz - hd.n_vert && hd.sell_slots % 2 == 0 && hd.opt.sell_c == hd.sell_c;
        if (ok) {
            if_options raw{};
            raw.gamma = hd.opt.gamma; raw.tol = hd.opt.tol; raw.max_iter = hd.opt.max_iter;
            raw.check_every = hd.opt.check_every; raw.batch = hd.opt.batch; raw.sell_c = hd.opt.sell_c;
            raw.sell_sigma = hd.opt.sell_sigma; raw.sfc_kind = hd.opt.sfc_kind; raw.flags = hd.opt.flags;
            raw.solver = hd.opt.solver; raw.mg_min_ell = hd.opt.mg_min_ell; raw.radius = hd.opt.radius;
            ok = ifl::resolve_options(&raw, nullptr, &chk) == IF_OK;
        }
        if (ok) {
            const int64_t nv = hd.n_vert, ns = hd.sell_slots, nt = hd.n_tiles;
            const int64_t expect = (int64_t)sizeof(hd) + (hd.n_chunks + 1) * 8 + ns * 16 + nv * (6 * 8 + 2 * 4) + nt * 4 +
                                   nt * HALO_CAP * 4 + (nt + 1) * 64 +
                                   ((hd.opt.flags & IF_FLAG_VECTOR) ? ns * 16 + nv * 16 : 0);
            const bool with_mg = (hd.opt.flags & IF_FLAG_MULTIGRID) != 0;      // the hierarchy follows the mesh arrays
            ok = fseek(f, 0, SEEK_END) == 0 && (with_mg ? (int64_t)ftell(f) > expect : (int64_t)ftell(f) == expect) &&
                 fseek(f, (long)sizeof(hd), SEEK_SET) == 0;
        }
        if (!ok) { fclose(f); return IF_EIO; }
    }
    if_mesh_s* h = new (std::nothrow) if_mesh_s();
    if (!h) { fclose(f); return IF_ENOMEM; }
    auto fail = [&](int rc) { fclose(f); if_destroy(h); return rc; };
    if (cudaGetDevice(&h->device) != cudaSuccess ||
        cudaDeviceGetAttribute(&h->n_sm, cudaDevAttrMultiProcessorCount, h->device) != cudaSuccess)
        return fail(IF_ECUDA);
    h->n_vert = hd.n_vert; h->nnz = hd.nnz; h->n_chunks = hd.n_chunks; h->sell_slots = hd.sell_slots;
    h->n_tiles = hd.n_tiles; h->halo_total = hd.halo_total; h->halo_max = hd.halo_max;
    h->unstaged_tiles = hd.unstaged_tiles; h->total_area = hd.total_area; h->mean_edge = hd.mean_edge;
    h->opt = hd.opt; h->sell_c = hd.sell_c;
    std::vector<char> buf;
    const size_t nv = (size_t)h->n_vert, ns = (size_t)h->sell_slots, nt = (size_t)h->n_tiles;
    int rc;
    if ((rc = read_dev(f, (void**)&h->chunk_ptr, (size_t)(h->n_chunks + 1) * 8, (size_t)(h->n_chunks + 1) * 8, buf))) return fail(rc);
    {
        int64_t last = -1;
        memcpy(&last, buf.data() + (size_t)h->n_chunks * 8, 8);
        if (last != h->sell_slots) return fail(IF_EIO);
    }
    if ((rc = read_dev(f, (void**)&h->sell_col, ns * 4, ns * 4 + 16, buf))) return fail(rc);
    if ((rc = read_dev(f, (void**)&h->sell_val, ns * 8, ns * 8 + 16, buf))) return fail(rc);
    if ((rc = read_dev(f, (void**)&h->sell_lcol, ns * 4, ns * 4 + 16, buf))) return fail(rc);
    if ((rc = read_dev(f, (void**)&h->area, nv * 8, nv * 8 + 16, buf))) return fail(rc);
    if ((rc = read_dev(f, (void**)&h->inv_area, nv * 8, nv * 8 + 16, buf))) return fail(rc);
    if ((rc = read_dev(f, (void**)&h->sdiag, nv * 8, nv * 8 + 16, buf))) return fail(rc);
    if ((rc = read_dev(f, (void**)&h->gdiag, nv * 8, nv * 8 + 16, buf))) return fail(rc);
    if ((rc = read_dev(f, (void**)&h->gdiag3, nv * 8, nv * 8 + 16, buf))) return fail(rc);
    if ((rc = read_dev(f, (void**)&h->gdiag4, nv * 8, nv * 8 + 16, buf))) return fail(rc);
    if (h->opt.flags & IF_FLAG_VECTOR) {
        if ((rc = read_dev(f, (void**)&h->sell_dval, ns * 8, ns * 8 + 16, buf))) return fail(rc);
        if ((rc = read_dev(f, (void**)&h->sell_tval, ns * 8, ns * 8 + 16, buf))) return fail(rc);
        if ((rc = read_dev(f, (void**)&h->ddiag, nv * 8, nv * 8 + 16, buf))) return fail(rc);
        if ((rc = read_dev(f, (void**)&h->gdiag_vec, nv * 8, nv * 8 + 16, buf))) return fail(rc);
        h->radius = hd.opt.radius;
    }
    if ((rc = read_dev(f, (void**)&h->perm, nv * 4, nv * 4, buf))) return fail(rc);
    if ((rc = read_dev(f, (void**)&h->iperm, nv * 4, nv * 4, buf))) return fail(rc);
    if ((rc = read_dev(f, (void**)&h->halo_n, nt * 4, nt * 4, buf))) return fail(rc);
    if ((rc = read_dev(f, (void**)&h->halo_rows, nt * HALO_CAP * 4, nt * HALO_CAP * 4, buf))) return fail(rc);
    if ((rc = read_dev(f, (void**)&h->tile_desc, (nt + 1) * 64, (nt + 1) * 64, buf))) return fail(rc);
    if (h->opt.flags & IF_FLAG_MULTIGRID) {
        int64_t L = 0;
        if (fread(&L, sizeof(L), 1, f) != 1 || L < 0 || L > ifl::MG_MAX_LEVELS) return fail(IF_EIO);
        for (int l = 0; l < (int)L; ++l) {
            ifl::MgLevel& g = h->mg[l];
            LevelHeader lh;
            if (fread(&lh, sizeof(lh), 1, f) != 1 || lh.n < 1 || lh.nnz < lh.n || lh.p_nnz < 0 || lh.n_coarse < 0 ||
                (l == 0 && lh.n != h->n_vert) || (l > 0 && lh.n != h->mg[l - 1].n_coarse) || !(lh.omega > 0.0))
                return fail(IF_EIO);
            g.n = lh.n; g.nnz = lh.nnz; g.n_coarse = lh.n_coarse; g.p_nnz = lh.p_nnz;
            g.rho = lh.rho; g.rho_m = lh.rho_m; g.omega = lh.omega;
            h->mg_levels = l + 1;      // (if_destroy frees what has been read so far)
            // (+16: the row-block kernels of the cycle bulk-copy 16-byte multiples)
            if ((rc = read_dev(f, (void**)&g.rowptr, (size_t)(g.n + 1) * 8, (size_t)(g.n + 1) * 8 + 16, buf))) return fail(rc);
            if ((rc = read_dev(f, (void**)&g.col, (size_t)g.nnz * 4, (size_t)g.nnz * 4 + 16, buf))) return fail(rc);
            if ((rc = read_dev(f, (void**)&g.sm, (size_t)g.nnz * 16, (size_t)g.nnz * 16 + 16, buf))) return fail(rc);
            if ((rc = read_dev(f, (void**)&g.diag, (size_t)g.n * 16, (size_t)g.n * 16 + 16, buf))) return fail(rc);
            if (l + 1 < (int)L) {
                if ((rc = read_dev(f, (void**)&g.p_rowptr, (size_t)(g.n + 1) * 8, (size_t)(g.n + 1) * 8 + 16, buf))) return fail(rc);
                if ((rc = read_dev(f, (void**)&g.p_col, (size_t)g.p_nnz * 4, (size_t)g.p_nnz * 4 + 16, buf))) return fail(rc);
                if ((rc = read_dev(f, (void**)&g.p_val, (size_t)g.p_nnz * 8, (size_t)g.p_nnz * 8 + 16, buf))) return fail(rc);
                if ((rc = read_dev(f, (void**)&g.r_rowptr, (size_t)(g.n_coarse + 1) * 8, (size_t)(g.n_coarse + 1) * 8 + 16, buf))) return fail(rc);
                if ((rc = read_dev(f, (void**)&g.r_col, (size_t)g.p_nnz * 4, (size_t)g.p_nnz * 4 + 16, buf))) return fail(rc);
                if ((rc = read_dev(f, (void**)&g.r_val, (size_t)g.p_nnz * 8, (size_t)g.p_nnz * 8 + 16, buf))) return fail(rc);
            }
        }
    }
    char extra;
    if (fread(&extra, 1, 1, f) != 0) return fail(IF_EIO);   // trailing bytes: not a file of ours
    fclose(f);
    h->h_pinned_bytes = 1 << 20;
    if (cudaHostAlloc(&h->h_pinned, h->h_pinned_bytes, cudaHostAllocDefault) != cudaSuccess) {
        cudaGetLastError();
        if_destroy(h);
        return IF_ENOMEM;
    }
    if (ifl::na_setup(h) != IF_OK || ifl::mg_tile_caps(h) != IF_OK) { if_destroy(h); return IF_ECUDA; }
    *out = h;
    return IF_OK;
}

extern "C" const char* if_strerror(int code) {
    switch (code) {
        case IF_OK: return "ok";
        case IF_WNOTCONVERGED: return "some right-hand sides did not converge (max_iter or breakdown)";
        case IF_EINVAL: return "invalid argument";
        case IF_EINDEX: return "triangle vertex id out of range or repeated";
        case IF_EDEGENERATE: return "degenerate triangle";
        case IF_EORPHAN: return "vertex in no triangle";
        case IF_ENOMEM: return "out of memory";
        case IF_ECUDA: return "CUDA error or no device";
        case IF_EWORKSPACE: return "workspace too small";
        case IF_ELIMIT: return "more fields than the static scratch array of if_energy_noalloc serves per call (32)";
        case IF_EIO: return "file cannot be written or read, or is not a prepared mesh of this library build";
        default: return "unknown error";
    }
}

extern "C" int64_t if_launch_count(void) { return (int64_t)ifl::g_launches.load(); }
