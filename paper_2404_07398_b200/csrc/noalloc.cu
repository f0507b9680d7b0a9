// An entry point that allocates nothing: if_energy_noalloc (include/implicit_filter.h).
//
// Some callers cannot call cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that forbid it.
// The solving calls of this library take their scratch from the caller's workspace; this file offers the one kernel
// whose scratch is small and fixed -- the energy reduction H6b, e = 1/2 sum_v A_v x_v^2 / sum_v A_v, a
// single-pass deterministic grid reduction that needs per-block partial sums and a ticket -- with that scratch in a
// file-scope device array of a stated maximum size instead.  Every GPU that loads the library holds the array
// (NA_SCRATCH_BYTES = 258 KiB) until the process exits.
//
// In host code the array's NAME is a host-side stand-in, not a device address: its address is looked up once per
// handle (= once per device, with that device current) by cudaGetSymbolAddress in na_setup, which if_prepare and
// if_load call, and the kernel is given that pointer.  The entry point itself calls no cudaMalloc, cudaFree or
// allocating library routine: one cudaMemsetAsync of the ticket, one launch.
//
// All calls share the array and it keeps the last call's contents: the ticket is cleared before every launch (in
// stream order), the partial sums are fully rewritten by every launch.  Calls that overlap on the GPU (different
// streams, or different host threads) race on it; serialise them.
#include "common.cuh"

namespace ifl {
namespace {

constexpr int NA_MAX_FIELDS = 32;      // fields per call
constexpr int NA_MAX_BLOCKS = 1024;    // blocks of the reduction grid (148 SMs x 4 = 592 on B200)
constexpr int NA_BLOCK = 256;
constexpr size_t NA_PARTIAL_BYTES = (size_t)NA_MAX_BLOCKS * NA_MAX_FIELDS * sizeof(double);
constexpr size_t NA_SCRATCH_BYTES = NA_PARTIAL_BYTES + 256;     // + the ticket (its own 256-byte line)

static __device__ __align__(256) unsigned char g_na_scratch[NA_SCRATCH_BYTES];

// e[f] = 1/2 sum_v A_v x_fv^2 / total_area for f < n_fields; fields [n_fields][nv] in the CALLER's vertex numbering,
// area in the internal order (iperm: caller -> internal).  Fixed-order sums: thread -> block (shared memory, in thread
// order) -> grid (the last block to take a ticket adds the blocks' partial sums in block order), so the result does
// not depend on scheduling.  scratch = [gridDim.x][NA_MAX_FIELDS] doubles, then the ticket.
__global__ void __launch_bounds__(NA_BLOCK) k_energy_static(const double* __restrict__ area, const int32_t* __restrict__ iperm,
                                                            int64_t nv, const double* __restrict__ fields, int n_fields,
                                                            double total_area, unsigned char* __restrict__ scratch,
                                                            double* __restrict__ energy) {
    constexpr int FC = 4;                          // fields per pass over the vertices
    __shared__ double red[NA_BLOCK];
    __shared__ bool is_last;
    double* partials = reinterpret_cast<double*>(scratch);
    unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch + NA_PARTIAL_BYTES);
    const int tid = threadIdx.x;
    for (int f0 = 0; f0 < n_fields; f0 += FC) {
        double acc[FC] = {0.0, 0.0, 0.0, 0.0};
        for (int64_t v = (int64_t)blockIdx.x * NA_BLOCK + tid; v < nv; v += (int64_t)gridDim.x * NA_BLOCK) {
            const double a = area[iperm[v]];
#pragma unroll
            for (int k = 0; k < FC; ++k)
                if (f0 + k < n_fields) {
                    const double x = fields[(int64_t)(f0 + k) * nv + v];
                    acc[k] = fma(a * x, x, acc[k]);
                }
        }
        for (int k = 0; k < FC && f0 + k < n_fields; ++k) {
            red[tid] = acc[k];
            __syncthreads();
            if (tid == 0) {
                double s = 0.0;
                for (int i = 0; i < NA_BLOCK; ++i) s += red[i];
                partials[(size_t)blockIdx.x * NA_MAX_FIELDS + f0 + k] = s;
            }
            __syncthreads();
        }
    }
    if (tid == 0) {
        __threadfence();
        is_last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    if (tid < n_fields) {
        double s = 0.0;
        for (unsigned b = 0; b < gridDim.x; ++b) s += __ldcg(&partials[(size_t)b * NA_MAX_FIELDS + tid]);
        energy[tid] = 0.5 * s / total_area;
    }
}

}  // namespace

// set-up, once per handle (the handle's device is current): the device address of the scratch array
int na_setup(if_mesh_s* h) {
    void* p = nullptr;
    IF_CUDA_TRY(cudaGetSymbolAddress(&p, g_na_scratch));
    h->na_scratch = p;
    return IF_OK;
}

}  // namespace ifl

using namespace ifl;

extern "C" int if_energy_noalloc(if_handle h, const double* d_fields, int n_fields, double* d_energy, void* cuda_stream) {
    if (!h || !d_fields || !d_energy || n_fields < 1) return IF_EINVAL;
    if (n_fields > NA_MAX_FIELDS) {
        fprintf(stderr, "[implicit_filter] if_energy_noalloc: %d fields exceed the fixed maximum of %d per call "
                        "(the scratch array is static; split the call)\n", n_fields, NA_MAX_FIELDS);
        return IF_ELIMIT;
    }
    if (!h->na_scratch) return IF_ECUDA;           // set-up failed in if_prepare / if_load
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return IF_ECUDA; }
    if (dev != h->device) return IF_EINVAL;        // the handle's device must be current (nothing is switched here)
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    unsigned char* scratch = static_cast<unsigned char*>(h->na_scratch);
    const int64_t want = (h->n_vert + NA_BLOCK - 1) / NA_BLOCK;
    const int grid = (int)(want < 1 ? 1 : (want > 4LL * h->n_sm ? 4LL * h->n_sm : want));
    const int g = grid > NA_MAX_BLOCKS ? NA_MAX_BLOCKS : grid;
    // the array keeps the last call's contents: the ticket must start at zero, the partial sums are all rewritten
    IF_CUDA_TRY(cudaMemsetAsync(scratch + NA_PARTIAL_BYTES, 0, 256, st));
    k_energy_static<<<g, NA_BLOCK, 0, st>>>(h->area, h->iperm, h->n_vert, d_fields, n_fields, h->total_area, scratch, d_energy);
    IF_LAUNCH_CHECK();
    return IF_OK;
}
