// gpe_norm_noalloc (include/gpe.h): the particle-number reduction h^3 sum |psi|^2 (Eq. 3; the paper's
// kernel K3) for callers that must not trigger a device allocation.
//
// Who that is.  gpe_norm() needs a gpe_sim, and creating a sim calls cudaMalloc four times and cudaMallocHost once
// (work records, block partial sums, the sums, a pinned flag).  Three kinds of users of this library cannot afford
// that:
//   - a process whose framework allocator (torch's caching allocator is the usual one) has already reserved nearly
//     all of the GPU's memory for state blocks -- the 1e8 to 3e8-point shells take tens of GB each -- so a raw
//     cudaMalloc from inside a library fails although the framework itself still has free blocks to hand out;
//   - a monitoring call placed between time steps while other streams are running: cudaMalloc and cudaFree wait for
//     the whole device, so a "cheap" norm check would stall every stream once per call;
//   - code that holds nothing but an array of wavefunction values (a checkpoint reader, a diagnostic thread) and
//     has no grid or sim to ask.
// For them the block partial sums -- the only scratch the reduction needs -- live in the file-scope device array
// below.  It is part of the library image: every GPU on which the library's kernels are loaded carries its
// GPE_NORM_NOALLOC_SCRATCH_BYTES (512 KiB) until the process exits, whether or not this call is ever made.  The
// price is a size limit (one slot per block of NOALLOC_CHUNK values, GPE_NORM_NOALLOC_MAX_VALUES in all) and no
// concurrency: all calls on a device use the same slots.
//
// The kernels are a variant of norm_kernel / finalize_kernel in gpe_kernels.cu (same per-block chunking, same
// fixed-order tree, fp64 accumulation), kept in this file because the scratch array, the code that resolves its
// device address and the launches that receive that address have to be in one translation unit.  Nothing in the
// existing paths calls into this file.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <mutex>

#include "gpe_internal.h"

namespace {

constexpr int NOALLOC_THREADS = 256;
constexpr int NOALLOC_CHUNK = 8192;     // values per block, at most (the same figure as gpe_kernels.cu's NORM_CHUNK)
constexpr int64_t NOALLOC_SLOTS = GPE_NORM_NOALLOC_SCRATCH_BYTES / sizeof(double);
static_assert(NOALLOC_SLOTS * NOALLOC_CHUNK == GPE_NORM_NOALLOC_MAX_VALUES, "gpe.h states the limit the scratch gives");

// The scratch: one partial sum per block.  In HOST code this name is only a handle for cudaGetSymbolAddress; it is
// not a device address and must never be handed to a kernel (scratch_of_current_device() below does the
// translation).  Contents survive from call to call; no slot has to start at zero, because a call writes every
// slot it will read (slots 0..nb-1) before the finishing kernel reads them, on the same stream.
static __device__ __align__(256) double g_norm_scratch[NOALLOC_SLOTS];

constexpr int MAX_DEVICES = 64;
std::mutex g_setup_mutex;
double* g_scratch_addr[MAX_DEVICES] = {};   // device address of g_norm_scratch on device d, once resolved

// Set-up, once per device, with that device current: ask the runtime where g_norm_scratch lives on it.  (This is
// also the moment the runtime loads the library's kernels onto the device if nothing has run there yet.)
int scratch_of_current_device(double** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return gpe::api_cuda_fail((int)e, "cudaGetDevice");
    if (dev < 0 || dev >= MAX_DEVICES) return gpe::api_fail(GPE_ERR_UNSUPPORTED, "gpe_norm_noalloc: device ordinal above 63");
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_addr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_norm_scratch);
        if (e != cudaSuccess) return gpe::api_cuda_fail((int)e, "cudaGetSymbolAddress(norm scratch)");
        if (!p) return gpe::api_fail(GPE_ERR_CUDA, "gpe_norm_noalloc: the runtime returned a null scratch address");
        g_scratch_addr[dev] = static_cast<double*>(p);
    }
    *out = g_scratch_addr[dev];
    return GPE_OK;
}

__device__ __forceinline__ double abs2(const double2 v) { return v.x * v.x + v.y * v.y; }
__device__ __forceinline__ double abs2(const float2 v) { return (double)v.x * (double)v.x + (double)v.y * (double)v.y; }
__device__ __forceinline__ double abs2(const double v) { return v * v; }

// slot[b] = sum of |psi_k|^2 over block b's contiguous chunk; thread t takes k = lo+t, lo+t+256, ... then a fixed
// shuffle / shared-memory tree (scheduling cannot change the result)
template <typename E>
__global__ void __launch_bounds__(NOALLOC_THREADS) noalloc_partial_kernel(const E* __restrict__ psi, int64_t n, int64_t chunk,
                                                                          double* __restrict__ slot) {
    __shared__ double red[NOALLOC_THREADS / 32];
    const int64_t lo = blockIdx.x * chunk, hi = (lo + chunk < n) ? lo + chunk : n;
    double acc = 0.0;
    for (int64_t k = lo + threadIdx.x; k < hi; k += NOALLOC_THREADS) acc += abs2(psi[k]);
    for (int off = 16; off > 0; off >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, off);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int wv = 0; wv < NOALLOC_THREADS / 32; ++wv) s += red[wv];
        slot[blockIdx.x] = s;
    }
}

constexpr int NOALLOC_FIN_THREADS = 1024;
// out[0] = cell_volume * sum_b slot[b], one block, fixed order: thread t sums b = t, t+1024, ..., then the tree.
// nb = 0 (an empty array) writes 0.
__global__ void __launch_bounds__(NOALLOC_FIN_THREADS) noalloc_finish_kernel(const double* __restrict__ slot, int64_t nb,
                                                                             double cell_volume, double* __restrict__ out) {
    __shared__ double red[NOALLOC_FIN_THREADS / 32];
    double acc = 0.0;
    for (int64_t b = threadIdx.x; b < nb; b += NOALLOC_FIN_THREADS) acc += slot[b];
    for (int off = 16; off > 0; off >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, off);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int wv = 0; wv < NOALLOC_FIN_THREADS / 32; ++wv) s += red[wv];
        out[0] = cell_volume * s;
    }
}

// true iff p is memory the current device's kernels may touch directly (its own device memory or managed memory)
bool on_current_device(const void* p) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return false;
    cudaPointerAttributes attr;
    if (cudaPointerGetAttributes(&attr, p) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    if (attr.type == cudaMemoryTypeManaged) return true;
    return attr.type == cudaMemoryTypeDevice && attr.device == dev;
}

}  // namespace

extern "C" int gpe_norm_noalloc(const void* dev_psi, int64_t n, int dtype, double cell_volume, double* dev_out, void* stream) {
    using gpe::api_fail;
    if (dtype != GPE_C64 && dtype != GPE_C128 && dtype != GPE_R64) return api_fail(GPE_ERR_INVALID_ARG, "gpe_norm_noalloc: unknown dtype");
    if (n < 0) return api_fail(GPE_ERR_INVALID_ARG, "gpe_norm_noalloc: n < 0");
    if (n > GPE_NORM_NOALLOC_MAX_VALUES)
        return api_fail(GPE_ERR_UNSUPPORTED,
                        "gpe_norm_noalloc: n exceeds GPE_NORM_NOALLOC_MAX_VALUES (536870912 values): the static scratch has one "
                        "slot per 8192 values and cannot grow; use gpe_norm on a sim, or reduce the array in pieces");
    if (!dev_out || (n > 0 && !dev_psi)) return api_fail(GPE_ERR_INVALID_ARG, "gpe_norm_noalloc: null pointer");
    if (!(cell_volume > 0.0) || !std::isfinite(cell_volume)) return api_fail(GPE_ERR_INVALID_ARG, "gpe_norm_noalloc: cell_volume must be finite and > 0");
    const size_t esize = dtype == GPE_C128 ? 16 : 8;
    if (((uintptr_t)dev_psi % esize) != 0 || ((uintptr_t)dev_out % sizeof(double)) != 0)
        return api_fail(GPE_ERR_INVALID_ARG, "gpe_norm_noalloc: dev_psi must be aligned to its element size and dev_out to 8 bytes");
    if (!on_current_device(dev_out) || (n > 0 && !on_current_device(dev_psi)))
        return api_fail(GPE_ERR_INVALID_ARG, "gpe_norm_noalloc: dev_psi / dev_out are not memory of the current CUDA device");
    double* slot = nullptr;
    const int rc = scratch_of_current_device(&slot);
    if (rc) return rc;

    cudaStream_t st = (cudaStream_t)stream;
    const int64_t nb = (n + NOALLOC_CHUNK - 1) / NOALLOC_CHUNK;   // <= NOALLOC_SLOTS by the check above
    if (nb > 0) {
        const int64_t chunk = (n + nb - 1) / nb;
        if (dtype == GPE_C128)
            noalloc_partial_kernel<double2><<<(unsigned)nb, NOALLOC_THREADS, 0, st>>>((const double2*)dev_psi, n, chunk, slot);
        else if (dtype == GPE_C64)
            noalloc_partial_kernel<float2><<<(unsigned)nb, NOALLOC_THREADS, 0, st>>>((const float2*)dev_psi, n, chunk, slot);
        else
            noalloc_partial_kernel<double><<<(unsigned)nb, NOALLOC_THREADS, 0, st>>>((const double*)dev_psi, n, chunk, slot);
        const cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return gpe::api_cuda_fail((int)e, "gpe_norm_noalloc: partial-sum launch");
    }
    noalloc_finish_kernel<<<1, NOALLOC_FIN_THREADS, 0, st>>>(slot, nb, cell_volume, dev_out);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return gpe::api_cuda_fail((int)e, "gpe_norm_noalloc: finishing launch");
    return GPE_OK;
}
