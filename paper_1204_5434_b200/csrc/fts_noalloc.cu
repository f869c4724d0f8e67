// fts_noalloc.cu — fts_mean_noalloc (include/fts.h): the mean of a complex field, i.e. Q = mean_x q(x,1) of
// PAPER.md:65 Eq. 4 when the field is the last contour slice, for callers that cannot give the library ANY device
// memory to work in.
//
// Who that is.  Every other entry point computes inside a workspace the caller cudaMalloc'ed for fts_create.  Some
// callers have nothing of the kind to hand over at the moment they need a number:
//   * an observer hooked into somebody else's running simulation (a convergence monitor, a checkpoint writer) that is
//     given device pointers to slices but owns no context, and whose host application has already partitioned all of
//     HBM among its own workspaces (a 256^3 store_both run holds 58 GB) — a cudaMalloc there can fail outright;
//   * code on a latency-critical path where marches are in flight on other streams: cudaMalloc and cudaFree may
//     synchronise the whole device, which would stall every one of those marches for one scalar;
//   * a process whose memory is managed by a pool (PyTorch's caching allocator, an MPI runtime) that must not see raw
//     runtime allocations appear beside it.
// For them the per-CTA partial sums of the two-stage reduction live in g_mean_partials below, a fixed array in the
// library's own device image, instead of in a workspace.  The caller passes only the input field and the 16-byte output.
//
// The arithmetic is that of the workspace path (reduce_partial_kernel / reduce_final_kernel<RED_SUM> in
// fts_kernels.cuh, launched by reduce() in fts_api.cu): same grid, same per-thread order, same shared-memory trees,
// same 1/npoints scaling, so the two agree bit for bit.  The kernels here are this file's own copies, restricted to
// the plain sum; nothing in the existing path was changed or is called.
//
// What a user must know (also in fts.h):
//   * Limit: npoints <= FTS_MEAN_NOALLOC_MAX_POINTS (2^24 = 256^3, the largest grid the library accepts); larger
//     inputs are refused with FTS_EUNSUPPORTED and a message, nothing is launched.
//   * Cost: 592 double2 = 9472 bytes of device memory on every GPU that loads libfts.so, held until the process exits,
//     whether or not this entry point is ever called.
//   * Set-up: the FIRST call on each device looks up the array's device address (cudaGetSymbolAddress, which may
//     initialise the CUDA context and load the library's device image).  Make that first call during start-up, before
//     any stream capture begins on that device.  Later calls on that device only launch two kernels.
//   * No cudaMalloc, cudaFree, or allocating library routine is called, on any call.
//   * Sharing: all calls on a device use the one array.  Nothing in it has to start at zero — the second kernel reads
//     only the partials the first kernel of the SAME call wrote, never more (a short field after a long one does not
//     see the long one's leftovers) — so there is nothing to clear between calls.  But two calls whose kernels can
//     run at the same time on one GPU (different streams, or different host threads on different streams) overwrite
//     each other's partials and give wrong means: issue the calls on one stream, or order them with events.
#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "../../include/fts.h"

namespace {

constexpr int NA_BLOCKS = 592, NA_THREADS = 256;    // the workspace path's RED_BLOCKS / RED_THREADS (4 CTAs per SM, 148 SMs)
constexpr int NA_MAX_DEVICES = 64;

// The scratch.  In host code this name is only a handle for cudaGetSymbolAddress — it is NOT a device address and must
// never be passed to a kernel; scratch_for_current_device() below turns it into one.
static __device__ __align__(256) double2 g_mean_partials[NA_BLOCKS];

template <class C2>     // C2 = double2 (complex128) or float2 (complex64); sums are fp64 in both
__global__ void __launch_bounds__(NA_THREADS) mean_partial_noalloc_kernel(const C2* __restrict__ a, int M, double2* __restrict__ partial) {
    __shared__ double2 sm[NA_THREADS];
    double2 acc = make_double2(0.0, 0.0);
    for (int i = blockIdx.x * NA_THREADS + threadIdx.x; i < M; i += gridDim.x * NA_THREADS) {
        const C2 v = a[i];
        acc.x += (double)v.x; acc.y += (double)v.y;
    }
    sm[threadIdx.x] = acc;
    __syncthreads();
    for (int s = NA_THREADS / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s) { sm[threadIdx.x].x += sm[threadIdx.x + s].x; sm[threadIdx.x].y += sm[threadIdx.x + s].y; }
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sm[0];      // every partial the second stage reads is written here, in this call
}

__global__ void __launch_bounds__(1024) mean_final_noalloc_kernel(const double2* __restrict__ partial, int n, double scale, double* __restrict__ out) {
    __shared__ double2 sm[1024];
    sm[threadIdx.x] = (int)threadIdx.x < n ? partial[threadIdx.x] : make_double2(0.0, 0.0);   // entries >= n may be stale: not read
    __syncthreads();
    for (int s = 512; s > 0; s >>= 1) {
        if (threadIdx.x < s) { sm[threadIdx.x].x += sm[threadIdx.x + s].x; sm[threadIdx.x].y += sm[threadIdx.x + s].y; }
        __syncthreads();
    }
    if (threadIdx.x == 0) { out[0] = sm[0].x * scale; out[1] = sm[0].y * scale; }
}

std::mutex g_setup_mutex;
double2* g_partials_addr[NA_MAX_DEVICES] = {};      // device address of g_mean_partials, per device ordinal; nullptr = not looked up yet

void say(char* errbuf, size_t len, const char* fmt, ...) {       // error text into the caller's buffer (may be NULL)
    if (!errbuf || !len) return;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(errbuf, len, fmt, ap);
    va_end(ap);
}

// Once per device, with that device current: the device address of the scratch array.
cudaError_t scratch_for_current_device(double2** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= NA_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_partials_addr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_mean_partials);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_partials_addr[dev] = static_cast<double2*>(p);
    }
    *out = g_partials_addr[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" fts_status fts_mean_noalloc(const void* field_dev, size_t npoints, fts_precision prec, double* mean_dev, void* stream,
                                       char* errbuf, size_t errbuf_len) {
    if (errbuf && errbuf_len) errbuf[0] = 0;
    if (!field_dev || !mean_dev || npoints == 0 || (prec != FTS_F64 && prec != FTS_F32)) {
        say(errbuf, errbuf_len, "fts_mean_noalloc: NULL pointer, npoints = 0 or unknown precision");
        return FTS_EINVAL;
    }
    if (npoints > (size_t)FTS_MEAN_NOALLOC_MAX_POINTS) {
        say(errbuf, errbuf_len, "fts_mean_noalloc: npoints = %llu exceeds the limit of %llu points (FTS_MEAN_NOALLOC_MAX_POINTS = 256^3); "
            "nothing was launched", (unsigned long long)npoints, (unsigned long long)FTS_MEAN_NOALLOC_MAX_POINTS);
        return FTS_EUNSUPPORTED;
    }
    double2* partial = nullptr;
    cudaError_t e = scratch_for_current_device(&partial);
    if (e != cudaSuccess) {
        say(errbuf, errbuf_len, "fts_mean_noalloc: looking up the static scratch array failed: %s", cudaGetErrorString(e));
        return FTS_ECUDA;
    }
    const int M = (int)npoints;
    int nb = (M + NA_THREADS - 1) / NA_THREADS; if (nb > NA_BLOCKS) nb = NA_BLOCKS;
    cudaStream_t st = (cudaStream_t)stream;
    if (prec == FTS_F64) mean_partial_noalloc_kernel<double2><<<nb, NA_THREADS, 0, st>>>((const double2*)field_dev, M, partial);
    else mean_partial_noalloc_kernel<float2><<<nb, NA_THREADS, 0, st>>>((const float2*)field_dev, M, partial);
    mean_final_noalloc_kernel<<<1, 1024, 0, st>>>(partial, nb, 1.0 / (double)M, mean_dev);
    e = cudaGetLastError();
    if (e != cudaSuccess) {
        say(errbuf, errbuf_len, "fts_mean_noalloc: kernel launch failed: %s", cudaGetErrorString(e));
        return FTS_ECUDA;
    }
    return FTS_OK;
}
