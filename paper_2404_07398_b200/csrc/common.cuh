// Shared declarations of the implicit-filter CUDA library (sm_100a).  See include/implicit_filter.h
// for the C ABI and DESIGN.md for the data layout.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include <atomic>

#include "implicit_filter.h"

namespace ifl {

// Row tile of the fused SpMM kernel and the most out-of-tile rows ("halo") a tile may stage in shared memory.
// if_prepare builds tile-local column ids and halo lists for exactly this tile height.
#ifndef IF_TILE_ROWS
#define IF_TILE_ROWS 128
#endif
#ifndef IF_HALO_CAP
#define IF_HALO_CAP 128
#endif
constexpr int TILE_ROWS = IF_TILE_ROWS;   // 64 or 128
constexpr int HALO_CAP = IF_HALO_CAP;     // multiple of 32

extern std::atomic<long long> g_launches;   // kernels launched by this library (if_launch_count)

#define IF_CUDA_TRY(expr)                                                                          \
    do {                                                                                           \
        cudaError_t e__ = (expr);                                                                  \
        if (e__ != cudaSuccess) {                                                                  \
            fprintf(stderr, "[implicit_filter] CUDA error %s at %s:%d: %s\n", cudaGetErrorName(e__), \
                    __FILE__, __LINE__, cudaGetErrorString(e__));                                  \
            return e__ == cudaErrorMemoryAllocation ? IF_ENOMEM : IF_ECUDA;                        \
        }                                                                                          \
    } while (0)

#define IF_LAUNCH_CHECK()                        \
    do {                                         \
        ++::ifl::g_launches;                     \
        IF_CUDA_TRY(cudaGetLastError());         \
    } while (0)

// Resolved options (defaults filled in).
struct Options {
    double gamma = 0.5;
    double tol = 1e-12;
    int max_iter = 200000;
    int check_every = 16;
    int batch = 16;
    int sell_c = 32;
    int sell_sigma = TILE_ROWS;   // sorting inside a row tile keeps the tile spatially compact
    int sfc_kind = 0;
    int flags = 0;
    int solver = 0;
    double radius = 0.0;        // R_e of the vector filter's metric terms; 0: mean |x_v| (dim = 3)
    double mg_min_ell = 0.0;    // 0: the default of the order (mg_solve.cuh: 0.5 mean edges)
};

int resolve_options(const if_options* in, const Options* base, Options* out);
}  // namespace ifl
struct if_mesh_s;
namespace ifl {
int mg_build(if_mesh_s* h);    // mg.cu: builds h->mg from the SELL matrix and the areas
int mg_tile_caps(if_mesh_s* h);   // mg.cu: fills MgLevel::cap_* (after mg_build or if_load)
int na_setup(if_mesh_s* h);    // noalloc.cu: looks up the device address of its static scratch array (once per handle)
void mg_free(if_mesh_s* h);

// ---- multigrid hierarchy (optional, IF_FLAG_MULTIGRID): smoothed aggregation on the internal row order.
// Level 0 is the mesh itself; level l+1 has one unknown per graph aggregate of level l (mg.cu).  Every level stores
// the pair (S_l, M_l) on one sparsity pattern, so that A_l = M_l + c S_l is applied matrix-free for any scale.
constexpr int MG_MAX_LEVELS = 12;
constexpr int MG_TILE = 64;        // rows per tile of the row-block kernels (k_mg_rows, mg_solve.cuh)
constexpr int MG_COARSEST = 64;    // the hierarchy stops at a level with at most this many unknowns (dense solve)
// Cycle and aggregation parameters (macros: the tuning runs of DESIGN.md section 9b rebuild with -DIF_MG_...).
#ifndef IF_MG_THETA
#define IF_MG_THETA 0.08
#endif
#ifndef IF_MG_NU_L1
#define IF_MG_NU_L1 1
#endif
#ifndef IF_MG_NU_COARSE
#define IF_MG_NU_COARSE 2
#endif
// strength of connection for the aggregates: |S_ij| >= theta sqrt(S_ii S_jj); 0 = the whole graph
constexpr double MG_THETA = IF_MG_THETA;
// a level whose strong graph coarsens by less than this uses the whole graph (small aggregates + a prolongator
// smoothed with the whole matrix = fill-in on the next level)
constexpr double MG_MIN_COARSENING = 6.0;
constexpr double MG_OMEGA_MAX = 0.9;   // Jacobi damping of the smoother, lowered where rho(D^-1 S) is large
// smoothing sweeps before and after the coarse correction: one on level 0 (a sweep there is a pass over the mesh),
// MG_NU_L1 on level 1 (an eighth of the mesh: its sweeps are a fifth of the cycle), MG_NU_COARSE below (cheap).
// Config 4, whole spectrum: with theta = 0.08 (1, 1) 0.925 s, (1, 2) 0.932 s, (2, 2) 0.981 s, (2, 4) 1.031 s;
// with theta = 0 (2, 4) 1.072 s, (3, 3) 1.18 s, (1, 3) 1.15 s.
constexpr int MG_NU_L1 = IF_MG_NU_L1;
constexpr int MG_NU_COARSE = IF_MG_NU_COARSE;
struct MgLevel {
    int64_t n = 0, nnz = 0;
    double rho = 2.0;            // estimate of rho(D_S^-1 S) (power iteration, with a safety factor)
    double rho_m = 1.0;          // the same for D_M^-1 M (1 on the mesh, where M is diagonal)
    double omega = 0.7;          // Jacobi damping of the smoother on this level: min(MG_OMEGA_MAX, 1.6 / max(rho, rho_m))
    int64_t* rowptr = nullptr;   // [n+1]
    int32_t* col = nullptr;      // [nnz]
    double2* sm = nullptr;       // [nnz]  (S_ij, M_ij)
    double2* diag = nullptr;     // [n]    (S_ii, M_ii)
    // transfer to level l+1 (absent on the coarsest level): P [n x n_coarse] by rows, R = P^T by rows
    int64_t n_coarse = 0, p_nnz = 0;
    // most entries in a block of MG_TILE consecutive rows of the level's matrix, of P and of R (mg_tile_caps): what a
    // stage of the row-block kernels of the cycle must hold
    int cap_a = 0, cap_p = 0, cap_r = 0;
    int64_t* p_rowptr = nullptr;
    int32_t* p_col = nullptr;
    double* p_val = nullptr;
    int64_t* r_rowptr = nullptr;
    int32_t* r_col = nullptr;
    double* r_val = nullptr;
};

}  // namespace ifl

// Device-resident prepared mesh.  Rows are in the internal order (SFC + SELL window sort):
// internal row r is caller vertex perm[r]; iperm[perm[r]] = r.
struct if_mesh_s {
    int device = 0;
    int64_t n_vert = 0;
    int64_t nnz = 0;          // entries of S incl. diagonal
    int64_t n_chunks = 0;     // ceil(n_vert / sell_c)
    int64_t sell_slots = 0;   // padded off-diagonal slots
    int sell_c = 32;
    double total_area = 0.0;
    double mean_edge = 0.0;
    int n_sm = 148;
    ifl::Options opt;
    // SELL-C-sigma, off-diagonal entries only; slice c holds rows [c*C, (c+1)*C), row-major [row][width_c],
    // width_c even, padding = (col = own row, val = 0).
    int64_t* chunk_ptr = nullptr;   // [n_chunks+1] slot offsets (even)
    int32_t* sell_col = nullptr;    // [sell_slots] internal column ids
    double* sell_val = nullptr;     // [sell_slots]
    // per row tile of TILE_ROWS rows: the out-of-tile rows it gathers from (sorted, unique) and the same matrix
    // with tile-local column ids (tile row r -> r, halo slot s -> TILE_ROWS + s); halo_n = -1: tile not staged
    int32_t* sell_lcol = nullptr;   // [sell_slots]
    int32_t* halo_n = nullptr;      // [n_tiles]
    int32_t* halo_rows = nullptr;   // [n_tiles][HALO_CAP], unused entries = the tile's first row
    int32_t* tile_desc = nullptr;   // [n_tiles+1][16] per-tile descriptor (see k_tile_halo)
    int64_t n_tiles = 0;
    int64_t halo_total = 0;
    int64_t halo_max = 0;         // largest staged halo
    int64_t unstaged_tiles = 0;   // tiles whose halo or row width exceeds the shared-memory caps
    double* area = nullptr;         // [n_vert] A_v            (internal order)
    double* inv_area = nullptr;     // [n_vert] 1/A_v
    double* sdiag = nullptr;        // [n_vert] S_vv
    double* gdiag = nullptr;        // [n_vert] sum_j S_vj^2/A_j = diag(S M^-1 S)
    double* gdiag3 = nullptr;       // [n_vert] diag(S (M^-1 S)^2)   (filter order 3)
    double* gdiag4 = nullptr;       // [n_vert] diag(S (M^-1 S)^3)   (filter order 4)
    // vector filter with metric terms (IF_FLAG_VECTOR), same SELL slots as sell_val:
    double* sell_dval = nullptr;    // [sell_slots] D~_vv' / l^2 (off-diagonal)
    double* sell_tval = nullptr;    // [sell_slots] T_vv' / l^2
    double* ddiag = nullptr;        // [n_vert] D~_vv / l^2
    double* gdiag_vec = nullptr;    // [n_vert] diag(D_2 M_2^-1 D_2) = sum_j (D~_vj^2 + T_vj^2) / A_j
    double radius = 0.0;            // R_e used for the metric terms (0: planar mesh, none)
    int32_t* perm = nullptr;        // [n_vert] internal -> caller
    int32_t* iperm = nullptr;       // [n_vert] caller -> internal
    // optional unpermuted CSR (IF_FLAG_KEEP_CSR), caller numbering
    int64_t* csr_rowptr = nullptr;
    int32_t* csr_col = nullptr;
    double* csr_val = nullptr;
    double* csr_area = nullptr;
    // multigrid hierarchy (IF_FLAG_MULTIGRID), see MgLevel
    ifl::MgLevel mg[ifl::MG_MAX_LEVELS];
    int mg_levels = 0;              // 0: no hierarchy
    double mg_build_seconds = 0.0;  // wall clock of mg_build
    void* na_scratch = nullptr;     // device address of the static scratch array of if_energy_noalloc (noalloc.cu)
    // pinned host staging for per-call control data and read-back
    void* h_pinned = nullptr;
    size_t h_pinned_bytes = 0;
    std::atomic<int> pinned_busy{0};   // 1 while a solve call uses h_pinned (others allocate their own)
};
