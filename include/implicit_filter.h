/*
 * implicit_filter.h -- C ABI of the B200-native implicit-filter hot path (arXiv 2404.07398).
 *
 * Citations: "PAPER.md:NN" = line NN of the paper text this library was written from.
 *
 * The paper splits the computation into a mesh-only preparation phase and a solving phase
 * (PAPER.md:105).  This boundary follows that split:
 *
 *   if_prepare   once per mesh: P1 stiffness S (cotangent weights) and median-dual areas A_v
 *                (PAPER.md:57-61), space-filling-curve reordering, SELL-C-sigma packing.
 *   if_filter    coarse-grained fields  phibar_l  for many fields and scales l:
 *                    (M + gamma l^(2n) S (M^-1 S)^(n-1)) phibar_l = M phi        (eq.(1), :61, :63)
 *                M = diag(A_v), gamma = 1/2, n = 1 harmonic / n = 2 biharmonic / n = 3, 4 ("can be
 *                generalized to higher-order filters"; the four-Laplacian filter of PAPER.md:201-205),
 *                solved by Jacobi-preconditioned conjugate gradients started from phi.
 *   if_spectrum  the same solves followed by e_l = 1/2 sum_v A_v phibar_l,v^2 / sum_v A_v  ("second moment
 *                of the field over scales") and its differences over k_l = 1/l.
 *   if_apply     the operator alone: out = (M + gamma l^(2n) S (M^-1 S)^(n-1)) phi  (residual checks).
 *
 * Conventions
 *   - fp64 everywhere; vertex ids int32; all multi-dimensional arrays are C-contiguous.
 *   - Every argument says whether it is a HOST or a DEVICE pointer.  The caller owns every buffer it
 *     passes (inputs, outputs, workspace); the handle owns the device arrays it built and if_destroy frees
 *     them.  The library keeps no caller pointer past return and never frees or resizes caller memory.
 *   - Inputs and outputs use the CALLER's vertex numbering; the internal reordering is invisible.
 *   - Work is enqueued on `cuda_stream` (a cudaStream_t passed as void*; NULL = default stream).  The solving calls
 *     (if_filter, if_spectrum, if_spectrum_host, if_apply) are synchronous: they poll the convergence flags while the
 *     iteration runs and wait for the stream before returning, on success and on every error path; outputs are
 *     complete on return.  if_energy_noalloc only enqueues.  The handle's device is made current for the duration of
 *     a solving call and the caller's current device is restored before it returns.
 *   - Return value: 0 on success; negative IF_E* on error (outputs untouched, nothing thrown);
 *     positive IF_WNOTCONVERGED when some right-hand side hit max_iter or broke down -- an expected outcome
 *     for n = 2 at large l; outputs then hold the last iterate and if_stats says which.
 *   - A handle is read-only after if_prepare: concurrent calls on one handle are safe if their workspaces
 *     and streams differ.  There is no CPU fallback: without a CUDA device every call fails with IF_ECUDA.
 */
#ifndef IMPLICIT_FILTER_H
#define IMPLICIT_FILTER_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct if_mesh_s* if_handle; /* opaque; owns all device-resident mesh arrays */

enum {
    IF_OK = 0,
    IF_WNOTCONVERGED = 1, /* some right-hand side stopped on max_iter or breakdown                         */
    IF_EINVAL = -1,       /* null pointer, dim not 2|3, order_n not 1..4, l <= 0 or non-finite, too few scales */
    IF_EINDEX = -2,       /* triangle vertex id out of range, or a vertex repeated inside a triangle       */
    IF_EDEGENERATE = -3,  /* triangle with |e1 x e2| <= 1e-14 (|e1|^2 + |e2|^2)                             */
    IF_EORPHAN = -4,      /* vertex in no triangle: A_v = 0, M singular                                    */
    IF_ENOMEM = -5,       /* host or device allocation failed                                              */
    IF_ECUDA = -6,        /* CUDA runtime error, or no device                                              */
    IF_EWORKSPACE = -7,   /* workspace smaller than if_workspace_bytes says                                */
    IF_EIO = -8,          /* if_save / if_load: file cannot be written / read, or is not a prepared mesh   */
    IF_ELIMIT = -9        /* if_energy_noalloc: more fields than its static scratch array serves per call  */
};

enum {
    IF_FLAG_KEEP_CSR = 1, /* if_prepare keeps the unpermuted CSR of S so if_mesh_export_csr works */
    IF_FLAG_MULTIGRID = 4, /* if_prepare also builds the smoothed-aggregation hierarchy that if_options.solver = 1 needs
                              (about 3 x the memory of the prepared mesh, a second or two of device time)          */
    IF_FLAG_HIGHPASS = 2, /* if_filter (per call): write the high-pass field phi - phibar_l (PAPER.md:143-147,
                             Fig. 3) instead of phibar_l                                                    */
    IF_FLAG_VECTOR = 16,  /* if_prepare: also assemble the metric terms of the vector Laplacian.
                             if_filter / if_spectrum / if_apply (per call, order_n 1|2, n_fields even): the fields are
                             velocities in pairs (u_0, v_0, u_1, v_1, ...) = (zonal, meridional) components at the
                             vertices, and every pair is filtered as ONE coupled 2V x 2V system
                                 S_2 = M_2 + gamma l^2 D_2   |   M_2 + gamma l^4 D_2 M_2^-1 D_2,   D_2 = [D~ T; -T D~],
                                 D~_vv' = int (grad N_v . grad N_v' + (R_e^-2 + m^2) N_v N_v') dS,
                                 T_vv'  = int m (-N_v' dx N_v + N_v dx N_v') dS,   m = tan(latitude) / R_e per triangle
                             (dim = 3: the mesh lies on a sphere about the origin, latitude from the z axis; dim = 2: no
                             metric terms, two scalar filters).  T is antisymmetric, D_2 symmetric positive semidefinite:
                             Jacobi-preconditioned CG with one residual norm over both components.  if_stats reports a
                             pair's iterations and status under both of its fields.  Combine with IF_FLAG_PAIRS for
                             the kinetic-energy spectrum                                                        */
    IF_FLAG_TRUE_RESIDUAL = 32, /* if_filter (per call, with a non-NULL if_stats.true_res; not with IF_FLAG_HIGHPASS): after the
                             solves, apply the operator to every returned field and report the TRUE relative residual
                             ||M phi - A_l x||_2 / ||M phi||_2 next to the recursive one (it floors near u * condition
                             number; one SpMM per right-hand side, outside if_stats.seconds)                       */
    IF_FLAG_PAIRS = 8     /* if_spectrum (per call): the fields are velocity components in pairs (u_0, v_0, u_1, v_1, ...)
                             and the spectra of a pair are added (kinetic energy 1/2 <u^2 + v^2>, the quantity of
                             PAPER.md:149-157): n_fields even; energy is [n_fields/2][n_ells], E [n_fields/2][n_ells-1];
                             if_stats stays per field                                                           */
};

typedef struct {
    double gamma;    /* 0 => 0.5                                                              */
    double tol;      /* 0 => 1e-12; stop when ||r||_2 <= tol ||M phi||_2 (recursive residual; PAPER.md:113
                        uses 1e-9)                                                                           */
    int max_iter;    /* 0 => 200000 iterations per right-hand side                                          */
    int check_every; /* 0 => 16; iterations per CUDA-graph launch = between two polls of the done flag     */
    int batch;       /* right-hand sides per SpMM: 4, 8 or 16; 0 => 16                                      */
    int sell_c;      /* SELL chunk height C (rows sharing one padded width): 32, 64 or 128; 0 => 32          */
    int sell_sigma;  /* SELL sorting window sigma (rows): multiple of sell_c; 0 => 128 (the SpMM row tile; a
                        larger window scatters a tile over the window and defeats the halo staging)         */
    int sfc_kind;    /* 0 => Morton order of the quantised coordinates; 1 => keep the caller's order        */
    int flags;       /* IF_FLAG_*                                                                           */
    int solver;      /* 0 => Jacobi-preconditioned CG for every right-hand side (per call: 0 inherits the handle's choice,
                        2 = Jacobi-PCG explicitly).  1 => right-hand sides with l >= mg_min_ell mean edge lengths are
                        solved by multigrid-preconditioned CG: one V cycle of a smoothed-aggregation hierarchy per
                        iteration for n = 1, the product V M V of two cycles for n = 2 (needs batch = 16 and a handle
                        prepared with IF_FLAG_MULTIGRID, else ignored; a call with up to 4 / 8 columns runs the
                        4- / 8-column variants of the cycle's kernels); the rest by Jacobi-PCG.  With IF_FLAG_VECTOR
                        the same hierarchy preconditions the coupled system: the coupled operator on the mesh,
                        the scalar levels below per component.  Same systems, same
                        start vector, same stop test, same answers within the tolerance (PAPER.md:207 names the
                        convergence of plain CG at large scales, above all for n = 2, as the open problem).  On
                        meshes of 400 000 vertices or more (n = 2: 100 000) the stream ends and starts its columns on
                        the device, inside each iteration's CUDA graph; the host only launches graphs and reads a
                        16-byte snapshot one launch behind (environment IF_MG_HOST_REFILL = 0 / 1 forces either way) */
    double radius;     /* if_prepare with IF_FLAG_VECTOR: R_e of the metric terms; 0 => the mean |x_v| of a dim = 3 mesh    */
    double mg_min_ell; /* in mean edge lengths; right-hand sides below that stay on the Jacobi path.  0 => 0.5 when
                          the call has 12 or more columns (right-hand sides; a (u, v) pair counts two); a call with
                          fewer runs 4- or 8-column kernels, which cost more per right-hand side, and Jacobi-PCG keeps
                          its smallest scales: n = 1 up to 2.5 (up to 4 columns) or 1.5 edge lengths, n = 2 up to 1  */
} if_options;

typedef struct {
    int32_t* iters;     /* HOST [n_fields*n_ells] or NULL: CG iterations of each right-hand side (f*L + j)  */
    double* rel_res;    /* HOST [n_fields*n_ells] or NULL: final recursive ||r||_2/||M phi||_2              */
    int32_t* status;    /* HOST [n_fields*n_ells] or NULL: 0 converged, 1 max_iter, 2 breakdown (p.Ap <= 0) */
    double seconds;     /* out: device time of the call (CUDA events on the stream)                         */
    int64_t batch_iters; /* out: fused SpMM+CG iterations launched, summed over batches                      */
    int64_t rhs_iters;   /* out: sum over right-hand sides of their iterations                               */
    double spmm_seconds;   /* out: mean device time of ONE operator application inside the iteration loop (the
                              fused SpMM kernel; for n = 2 its two launches), CUDA events on the stream, sampled
                              once per check_every iterations; 0 if nothing was sampled                       */
    double update_seconds; /* out: the same for ONE fused vector-update kernel                               */
    int64_t kernel_samples; /* out: number of samples behind the two means                                   */
    double mg_kernel_seconds[8]; /* out (solver = 1): mean device time per ITERATION of the kernel groups of the
                              multigrid-preconditioned path, CUDA events on the stream, one sample per graph launch:
                              [0] kernel A (n = 2: its two launches)  [1] fused residual update + first sweep + its
                              residual on the mesh  [2] restriction mesh -> level 1  [3] all kernels on level 1
                              [4] levels >= 2  [5] prolongation level 1 -> mesh  [6] last sweep (+ CG bookkeeping);
                              for n = 2 groups 1-6 hold the sum over both cycles; [7] unused                         */
    int64_t mg_samples;     /* out: samples behind mg_kernel_seconds                                          */
    int64_t mg_batch_iters; /* out: 16-column iterations of the multigrid-preconditioned path (part of batch_iters) */
    double* true_res;   /* HOST [n_fields*n_ells] or NULL: filled by if_filter with IF_FLAG_TRUE_RESIDUAL (the vector
                           filter reports a pair's joint residual under both of its fields)                          */
} if_stats;

/* Preparation phase.  All pointers HOST.
 *   coords  [n_vert][dim] vertex positions, dim = 2 (planar) or 3 (surface in space; triangles are flat)
 *   tri     [n_tri][3]    vertex ids, any orientation
 *   period  [dim] or NULL; period[d] > 0 makes axis d periodic (edge vectors use the minimum image)
 *   opt     NULL => defaults;   out: receives the handle (device-resident mesh; the current CUDA device)
 * Boundary edges (one adjacent triangle) get the natural no-normal-flux condition. */
int if_prepare(const double* coords, int dim, int64_t n_vert, const int32_t* tri, int64_t n_tri,
               const double* period, const if_options* opt, if_handle* out);

/* Bytes of DEVICE workspace if_filter / if_spectrum / if_apply need for this order (1..4) and batch (0 => default). */
int if_workspace_bytes(if_handle h, int order_n, int batch, size_t* bytes);

/* Solving phase.  d_fields DEVICE [n_fields][n_vert]; ells HOST [n_ells] (> 0, coordinate units, any order);
 * order_n 1..4 (the condition number grows like (l^2 lambda_max)^n: fp64 carries n = 3 to about 6 and n = 4 to about 2.5
 * edge lengths, beyond that the call returns IF_WNOTCONVERGED like n = 2 beyond 32); d_out DEVICE [n_fields][n_ells][n_vert]; d_workspace DEVICE, ws_bytes >= if_workspace_bytes;
 * opt NULL => the options given to if_prepare; stats NULL or HOST. */
int if_filter(if_handle h, const double* d_fields, int n_fields, const double* ells, int n_ells, int order_n,
              double* d_out, void* d_workspace, size_t ws_bytes, void* cuda_stream, const if_options* opt,
              if_stats* stats);

/* As if_filter, but only the scale spectrum is returned (no field output).  n_ells >= 2, ells strictly
 * ascending.  HOST outputs: energy [n_fields][n_ells] = e_l; k_mid [n_ells-1] = sqrt(k_j k_j+1), k_j = 1/l_j;
 * E [n_fields][n_ells-1] = (e_j - e_j+1)/(k_j - k_j+1).  Any of the three may be NULL. */
int if_spectrum(if_handle h, const double* d_fields, int n_fields, const double* ells, int n_ells, int order_n,
                double* energy, double* k_mid, double* E, void* d_workspace, size_t ws_bytes,
                void* cuda_stream, const if_options* opt, if_stats* stats);

/* if_spectrum for callers whose fields live in HOST memory (pinned memory makes the copy asynchronous): the fields
 * are copied to the device inside the call, into the tail of the workspace, which must therefore hold
 * if_workspace_bytes(...) + n_fields * n_vert * 8 bytes.  Everything else as if_spectrum. */
int if_spectrum_host(if_handle h, const double* h_fields, int n_fields, const double* ells, int n_ells, int order_n,
                     double* energy, double* k_mid, double* E, void* d_workspace, size_t ws_bytes,
                     void* cuda_stream, const if_options* opt, if_stats* stats);

/* The energy reduction alone, for callers that cannot call cudaMalloc (CUDA graph capture, serving loops, harnesses
 * that forbid it):  d_energy[f] = 1/2 sum_v A_v x_fv^2 / sum_v A_v  (what if_spectrum reports per filtered
 * field) for d_fields DEVICE [n_fields][n_vert] in the caller's numbering, e.g. the output of if_filter; d_energy DEVICE
 * [n_fields].  Takes no workspace and allocates nothing: the scratch of its grid reduction is a static device array of
 * 258 KiB inside the library (held by every GPU that loads the library until exit), which serves at most 32 fields per
 * call -- more returns IF_ELIMIT.  One memset of 256 bytes and one kernel are enqueued on `cuda_stream`; no
 * synchronisation.  The handle's device must be current (else IF_EINVAL).  All calls share the array: calls that
 * overlap on the GPU (other streams or threads) race -- serialise them.  The result is deterministic. */
int if_energy_noalloc(if_handle h, const double* d_fields, int n_fields, double* d_energy, void* cuda_stream);

/* Operator only: d_out[f][j] = (M + gamma l_j^(2n) S (M^-1 S)^(n-1)) d_fields[f].  Same layouts as if_filter. */
int if_apply(if_handle h, const double* d_fields, int n_fields, const double* ells, int n_ells, int order_n,
             double* d_out, void* d_workspace, size_t ws_bytes, void* cuda_stream, const if_options* opt);

/* Mesh facts (all HOST, any may be NULL): vertices, stored entries of S (diagonal included), sum of A_v,
 * mean edge length, padded SELL slots (off-diagonal entries incl. padding). */
int if_mesh_info(if_handle h, int64_t* n_vert, int64_t* nnz, double* total_area, double* mean_edge,
                 int64_t* sell_slots);

/* Row tiling of the fused SpMM kernel (all HOST, any may be NULL): tiles of 128 consecutive internal rows, total
 * and largest number of out-of-tile rows ("halo") the tiles gather from, and tiles left unstaged because their
 * halo or row width exceeds the shared-memory caps (they take the slower global-gather path). */
int if_mesh_tile_info(if_handle h, int64_t* n_tiles, int64_t* halo_rows, int64_t* halo_max, int64_t* unstaged_tiles);

/* The multigrid hierarchy of a handle prepared with IF_FLAG_MULTIGRID (all HOST, any may be NULL): number of levels
 * (0: none; level 0 is the mesh), per level l < 12 its rows, stored entries of the (S_l, M_l) pair and entries of the
 * prolongator to level l+1, the wall-clock seconds if_prepare spent building it, and the Jacobi sweeps per side of the
 * V cycle, sweeps[n-1][0..2] = on the mesh, on level 1, below, for filter order n = 1, 2 (bench.py's byte model). */
int if_mesh_multigrid_info(if_handle h, int* n_levels, int64_t* rows, int64_t* nnz, int64_t* p_nnz,
                           double* build_seconds, int* sweeps);

/* Copy S (CSR, caller's numbering, columns ascending, diagonal included) and A_v to HOST arrays:
 * rowptr [n_vert+1], col [nnz], val [nnz], area [n_vert]; any may be NULL.  Needs IF_FLAG_KEEP_CSR
 * (else IF_EINVAL).  For checking the preparation phase against another assembly. */
int if_mesh_export_csr(if_handle h, int64_t* rowptr, int32_t* col, double* val, double* area);

/* Internal ordering (HOST [n_vert], may be NULL): perm[new] = caller id of internal row `new`. */
int if_mesh_export_perm(if_handle h, int32_t* perm);

/* The prepared mesh is independent of the scales and can be kept on disk and reused.
 * if_save writes every device array of the handle -- the multigrid hierarchy of IF_FLAG_MULTIGRID included -- to `path`
 * (HOST string); if_load rebuilds a handle on the current CUDA device from such a file (same library build: the
 * row-tile constants and the size of every array are checked against the header and the file's length).  The optional
 * CSR copy of IF_FLAG_KEEP_CSR is not saved.  IF_EIO on any file problem. */
int if_save(if_handle h, const char* path);
int if_load(const char* path, if_handle* out);

void if_destroy(if_handle h);
const char* if_strerror(int code);
/* Kernels launched by this library in the calling process so far (bench.py's gpu_launches). */
int64_t if_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* IMPLICIT_FILTER_H */
