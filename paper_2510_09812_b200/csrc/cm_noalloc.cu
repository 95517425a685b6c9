// cm_volume_average_noalloc: the volume average of S2 (Eq. 16-17) for callers that must not allocate.
//
// Who this is for.  cm_volume_average keeps a library-order staging copy of the field inside the mesh and grows it
// with cudaFree + cudaMalloc when a larger field arrives.  That is a problem for two kinds of caller:
//   * a host program that hands the whole device to its own memory pool at start-up (a simulation framework with
//     a fixed memory budget, an arena allocator, a tensor library's caching allocator grown to the limit): there
//     is nothing left for cudaMalloc to give, so the first average of a reordered mesh fails with out-of-memory;
//   * a time loop that monitors <m> every step while other streams are busy: cudaMalloc and cudaFree may
//     synchronise the whole device and take an unbounded time, which stalls every stream of the process.
// This entry point allocates nothing, frees nothing, calls no allocating library routine and does not synchronise.
// The caller passes the field and the place for the result (both device memory); the only scratch memory, one
// partial sum per tile of nodes, lives in a file-scope device array of fixed size that every GPU which loads the
// library holds until the process exits (NA_MAX_TILES x NA_MAX_NC doubles = 96 KiB per GPU).
//
// What the fixed array costs the caller:
//   * sizes: at most CM_NOALLOC_MAX_NODES nodes (2048 tiles of 8192 nodes = 16,777,216) and 1, 3 or 6 components;
//     anything larger is refused with CM_E_BADARG and a message, nothing is launched;
//   * sharing: every call on a GPU uses the SAME array, whatever mesh or stream it is given.  Two calls that can
//     overlap on the GPU (different streams, or different host threads with different streams) race on it and both
//     results are garbage.  Put them on one stream, or order them with events;
//   * contents: the array keeps the last call's partial sums.  Nothing in it has to start at zero: the first kernel
//     of a call writes every row the second kernel of that call reads (rows 0 .. tiles-1), and rows beyond are
//     never read, so there is nothing to clear between calls (tests/test_zz_no_alloc.py calls it twice in a row
//     with a larger and then a smaller problem for exactly this reason);
//   * set-up: host code cannot use the array's name as a device address, so the first call on each GPU asks the
//     runtime for the address (cudaGetSymbolAddress, with that GPU current) and caches it per device ordinal.  That
//     first call is a set-up call: make it once per GPU before any stream capture begins.
#include "cm_internal.h"

namespace {

constexpr int NA_BS = 256;          // threads per CTA
constexpr int NA_TILE = 8192;       // nodes summed by one CTA (32 per thread)
constexpr int NA_MAX_TILES = 2048;  // rows of the scratch array
constexpr int NA_MAX_NC = 6;        // components per row (a symmetric tensor field)
constexpr int NA_MAX_DEV = 64;      // device ordinals the address cache covers
static_assert((long)NA_TILE * NA_MAX_TILES == CM_NOALLOC_MAX_NODES, "header and scratch size disagree");

// The scratch: row t holds the NC partial sums of tile t, packed [t * NC + c] for the NC of the current call.
// In HOST code this name is only a handle for cudaGetSymbolAddress; it is never passed to a kernel.
static __device__ __align__(256) double g_na_partial[NA_MAX_TILES * NA_MAX_NC];

// partial[t][c] = sum over the nodes i of tile t (library order) of w_i * g[order[i]][c]; fixed summation order:
// thread-strided within the tile, shuffle tree within a warp, warps in ascending order.
template <typename T, int NC>
__global__ void __launch_bounds__(NA_BS) na_tile_sum_kernel(long N, const double *__restrict__ w, const int *__restrict__ order,
                                                            const T *__restrict__ g_user, double *__restrict__ partial)
{
    __shared__ double sh[NC][NA_BS / 32];
    const long lo = (long)blockIdx.x * NA_TILE;
    const long hi = lo + NA_TILE < N ? lo + NA_TILE : N;
    double acc[NC];
#pragma unroll
    for (int c = 0; c < NC; c++) acc[c] = 0;
    for (long i = lo + threadIdx.x; i < hi; i += NA_BS) {
        const double wi = w[i];
        const long j = order ? (long)order[i] : i;
#pragma unroll
        for (int c = 0; c < NC; c++) acc[c] += wi * (double)g_user[j * NC + c];
    }
#pragma unroll
    for (int c = 0; c < NC; c++)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc[c] += __shfl_xor_sync(0xffffffffu, acc[c], o);
    if ((threadIdx.x & 31) == 0)
#pragma unroll
        for (int c = 0; c < NC; c++) sh[c][threadIdx.x >> 5] = acc[c];
    __syncthreads();
    if (threadIdx.x < NC) {
        double s = 0;
        for (int k = 0; k < NA_BS / 32; k++) s += sh[threadIdx.x][k];
        partial[(long)blockIdx.x * NC + threadIdx.x] = s;
    }
}

// one CTA: out[c] = sum_t partial[t][c], t < ntiles (ntiles == 0 writes zeros)
__global__ void __launch_bounds__(NA_BS) na_final_kernel(int ntiles, int nc, const double *__restrict__ partial, double *__restrict__ out)
{
    __shared__ double sh[NA_BS];
    for (int c = 0; c < nc; c++) {
        double s = 0;
        for (int t = threadIdx.x; t < ntiles; t += NA_BS) s += partial[(long)t * nc + c];
        sh[threadIdx.x] = s;
        __syncthreads();
        for (int o = NA_BS / 2; o > 0; o >>= 1) {
            if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
            __syncthreads();
        }
        if (threadIdx.x == 0) out[c] = sh[0];
        __syncthreads();
    }
}

std::mutex g_na_lock;
double *g_na_addr[NA_MAX_DEV] = {}; // device address of g_na_partial on each GPU, filled on that GPU's first call

// Device address of the scratch array on the CURRENT device (asked for once per device, then cached).
int na_scratch_address(double **out)
{
    int dev = -1;
    CM_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= NA_MAX_DEV) {
        cm_set_error("cm_volume_average_noalloc: device ordinal %d is outside the %d this entry point keeps an address for", dev, NA_MAX_DEV);
        return CM_E_BADARG;
    }
    std::lock_guard<std::mutex> hold(g_na_lock);
    if (!g_na_addr[dev]) {
        double *p = nullptr;
        CM_CUDA(cudaGetSymbolAddress((void **)&p, g_na_partial));
        if (!p) { cm_set_error("cm_volume_average_noalloc: cudaGetSymbolAddress returned a null address"); return CM_E_CUDA; }
        g_na_addr[dev] = p;
    }
    *out = g_na_addr[dev];
    return CM_OK;
}

template <typename T>
int na_launch(const cm_mesh *M, const T *g, int nc, double *scratch, double *out_dev, cudaStream_t st)
{
    const int ntiles = (int)((M->N + NA_TILE - 1) / NA_TILE);
    const int *order = M->identity ? nullptr : M->d_order;
    if (ntiles > 0) {
        switch (nc) {
        case 1: na_tile_sum_kernel<T, 1><<<ntiles, NA_BS, 0, st>>>(M->N, M->d_wvol, order, g, scratch); break;
        case 3: na_tile_sum_kernel<T, 3><<<ntiles, NA_BS, 0, st>>>(M->N, M->d_wvol, order, g, scratch); break;
        default: na_tile_sum_kernel<T, 6><<<ntiles, NA_BS, 0, st>>>(M->N, M->d_wvol, order, g, scratch); break;
        }
    }
    na_final_kernel<<<1, NA_BS, 0, st>>>(ntiles, nc, scratch, out_dev);
    CM_CUDA(cudaGetLastError());
    return CM_OK;
}

} // namespace

extern "C" int cm_volume_average_noalloc(const cm_mesh *mesh, cm_dtype dtype, const void *g_dev, int ncomp, double *out_dev, void *stream)
{
    if (!mesh || !g_dev || !out_dev) { cm_set_error("cm_volume_average_noalloc: null argument"); return CM_E_BADARG; }
    if (dtype != CM_F64 && dtype != CM_F32) { cm_set_error("cm_volume_average_noalloc: unknown dtype"); return CM_E_BADARG; }
    if (ncomp != 1 && ncomp != 3 && ncomp != 6) {
        cm_set_error("cm_volume_average_noalloc: ncomp = %d, but the fixed scratch array is laid out for 1, 3 or 6 components", ncomp);
        return CM_E_BADARG;
    }
    if (mesh->N > CM_NOALLOC_MAX_NODES) {
        cm_set_error("cm_volume_average_noalloc: the mesh has %ld nodes, the fixed scratch array covers at most %ld "
                     "(use cm_volume_average, which allocates)", mesh->N, (long)CM_NOALLOC_MAX_NODES);
        return CM_E_BADARG;
    }
    double *scratch = nullptr;
    CM_TRY(na_scratch_address(&scratch));
    cudaStream_t st = (cudaStream_t)stream;
    if (dtype == CM_F64) return na_launch<double>(mesh, (const double *)g_dev, ncomp, scratch, out_dev, st);
    return na_launch<float>(mesh, (const float *)g_dev, ncomp, scratch, out_dev, st);
}
