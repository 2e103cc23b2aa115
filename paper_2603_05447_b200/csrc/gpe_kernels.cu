// Small CUDA kernels (sm_100a) of the sparse-grid Gross-Pitaevskii path: canonical <-> storage order
// (pack / unpack), the norm reduction and the fixed-order final pass of every
// reduction (row a6; PAPER.md:87 kernel K3), the flush of the lazy renormalisation scale.  The fused stage
// kernels are in gpe_stage.cu.
#include <cuda_runtime.h>

#include <cstdint>

#include "gpe_internal.h"

namespace gpe {

namespace {

template <typename T> struct CxOf;
template <> struct CxOf<double> { using type = double2; };
template <> struct CxOf<float> { using type = float2; };

// ---- small kernels ------------------------------------------------------------------------------
template <typename C>
__global__ void pack_kernel(const C* __restrict__ canonical, C* __restrict__ storage, const int64_t* __restrict__ perm, int64_t n) {
    for (int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; s < n; s += (int64_t)gridDim.x * blockDim.x)
        storage[s] = canonical[perm[s]];
}
template <typename C>
__global__ void unpack_kernel(const C* __restrict__ storage, C* __restrict__ canonical, const int64_t* __restrict__ perm, int64_t n) {
    for (int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; s < n; s += (int64_t)gridDim.x * blockDim.x)
        canonical[perm[s]] = storage[s];
}

// re-gridding: dst[i] = src[map[i]] or 0 where the new point was not in the old grid (canonical order)
template <typename C>
__global__ void remap_kernel(const C* __restrict__ src, C* __restrict__ dst, const int64_t* __restrict__ map, int64_t n) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t m = map[i];
        C v;
        v.x = 0; v.y = 0;
        if (m >= 0) v = src[m];
        dst[i] = v;
    }
}

constexpr int NORM_THREADS = 256;
constexpr int NORM_CHUNK = 8192;   // elements per block
constexpr int NORM_MAX_BLOCKS = 148 * 16;

template <typename C>
__global__ void __launch_bounds__(NORM_THREADS) norm_kernel(const C* __restrict__ psi, int64_t n, int64_t chunk, double* partials) {
    __shared__ double red[NORM_THREADS / 32];
    const int64_t lo = blockIdx.x * chunk, hi = (lo + chunk < n) ? lo + chunk : n;
    double acc = 0.0;
    for (int64_t k = lo + threadIdx.x; k < hi; k += NORM_THREADS) {
        const C v = psi[k];
        acc += (double)v.x * (double)v.x + (double)v.y * (double)v.y;
    }
    for (int off = 16; off > 0; off >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, off);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int wv = 0; wv < NORM_THREADS / 32; ++wv) s += red[wv];
        partials[(size_t)blockIdx.x * NACC + 0] = s;
        partials[(size_t)blockIdx.x * NACC + 1] = 0.0;
        partials[(size_t)blockIdx.x * NACC + 2] = 0.0;
        partials[(size_t)blockIdx.x * NACC + 3] = 0.0;
    }
}

constexpr int FIN_THREADS = 1024;
// out[k] = sum over blocks, fixed order: thread t sums b = t, t+1024, ... then a fixed shuffle/shared tree
__global__ void __launch_bounds__(FIN_THREADS) finalize_kernel(const double* __restrict__ partials, int64_t nblk, double* out,
                                                                double* scale_out, double n_target, double h3) {
    __shared__ double red[FIN_THREADS / 32][NACC];
    double acc[NACC] = {0.0, 0.0, 0.0, 0.0};
    for (int64_t b = threadIdx.x; b < nblk; b += FIN_THREADS) {
        const double4 v = *reinterpret_cast<const double4*>(partials + b * NACC);
        acc[0] += v.x; acc[1] += v.y; acc[2] += v.z; acc[3] += v.w;
    }
#pragma unroll
    for (int k = 0; k < NACC; ++k)
        for (int off = 16; off > 0; off >>= 1) acc[k] += __shfl_down_sync(0xffffffffu, acc[k], off);
    if ((threadIdx.x & 31) == 0)
        for (int k = 0; k < NACC; ++k) red[threadIdx.x >> 5][k] = acc[k];
    __syncthreads();
    if (threadIdx.x < NACC) {
        double s = 0.0;
        for (int wv = 0; wv < FIN_THREADS / 32; ++wv) s += red[wv][threadIdx.x];
        out[threadIdx.x] = s;
        if (threadIdx.x == 0 && scale_out) {
            // a zero or non-finite particle number has no renormalisation: keep the values as they are (scale 1)
            // and raise the sticky flag next to the scale; the host turns it into GPE_ERR_STATE at the flush
            const bool ok = s > 0.0 && isfinite(s);
            scale_out[0] = ok ? sqrt(n_target / (h3 * s)) : 1.0;
            if (!ok) scale_out[1] = 1.0;
        }
    }
}

template <typename T>
__global__ void scale_kernel(typename CxOf<T>::type* psi, int64_t n, const double* scale) {
    const T s = (T)(*scale);
    for (int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) {
        auto v = psi[k];
        v.x *= s;
        v.y *= s;
        psi[k] = v;
    }
}

__global__ void set_scalar_kernel(double* dst, double v) { *dst = v; }

inline int grid_for(int64_t n, int threads) {
    int64_t b = (n + threads - 1) / threads;
    const int64_t cap = 148 * 32;
    if (b > cap) b = cap;
    if (b < 1) b = 1;
    return (int)b;
}

}  // namespace

int launch_pack(int dtype, const void* canonical, void* storage, const int64_t* perm, int64_t n, void* stream) {
    if (n <= 0) return 0;
    cudaStream_t st = (cudaStream_t)stream;
    if (dtype == GPE_C128)
        pack_kernel<double2><<<grid_for(n, 256), 256, 0, st>>>((const double2*)canonical, (double2*)storage, perm, n);
    else
        pack_kernel<float2><<<grid_for(n, 256), 256, 0, st>>>((const float2*)canonical, (float2*)storage, perm, n);
    return (int)cudaGetLastError();
}

int launch_unpack(int dtype, const void* storage, void* canonical, const int64_t* perm, int64_t n, void* stream) {
    if (n <= 0) return 0;
    cudaStream_t st = (cudaStream_t)stream;
    if (dtype == GPE_C128)
        unpack_kernel<double2><<<grid_for(n, 256), 256, 0, st>>>((const double2*)storage, (double2*)canonical, perm, n);
    else
        unpack_kernel<float2><<<grid_for(n, 256), 256, 0, st>>>((const float2*)storage, (float2*)canonical, perm, n);
    return (int)cudaGetLastError();
}

int launch_remap(int dtype, const void* src_canonical, void* dst_canonical, const int64_t* map, int64_t n_dst, void* stream) {
    if (n_dst <= 0) return 0;
    cudaStream_t st = (cudaStream_t)stream;
    if (dtype == GPE_C128)
        remap_kernel<double2><<<grid_for(n_dst, 256), 256, 0, st>>>((const double2*)src_canonical, (double2*)dst_canonical, map, n_dst);
    else
        remap_kernel<float2><<<grid_for(n_dst, 256), 256, 0, st>>>((const float2*)src_canonical, (float2*)dst_canonical, map, n_dst);
    return (int)cudaGetLastError();
}

int norm_blocks(int64_t n) {
    int64_t b = (n + NORM_CHUNK - 1) / NORM_CHUNK;
    if (b > NORM_MAX_BLOCKS) b = NORM_MAX_BLOCKS;
    if (b < 1) b = 1;
    return (int)b;
}

int launch_norm_partials(int dtype, const void* storage, int64_t n, double* partials, void* stream) {
    cudaStream_t st = (cudaStream_t)stream;
    const int nb = norm_blocks(n);
    const int64_t chunk = (n + nb - 1) / nb;
    if (dtype == GPE_C128)
        norm_kernel<double2><<<nb, NORM_THREADS, 0, st>>>((const double2*)storage, n, chunk, partials);
    else
        norm_kernel<float2><<<nb, NORM_THREADS, 0, st>>>((const float2*)storage, n, chunk, partials);
    return (int)cudaGetLastError();
}

int launch_finalize(const double* partials, int64_t nblk, double* out, double* scale_out, double n_target, double h3,
                    void* stream) {
    finalize_kernel<<<1, FIN_THREADS, 0, (cudaStream_t)stream>>>(partials, nblk, out, scale_out, n_target, h3);
    return (int)cudaGetLastError();
}

int launch_scale(int dtype, void* storage, int64_t n, const double* scale, void* stream) {
    if (n <= 0) return 0;
    cudaStream_t st = (cudaStream_t)stream;
    if (dtype == GPE_C128)
        scale_kernel<double><<<grid_for(n, 256), 256, 0, st>>>((double2*)storage, n, scale);
    else
        scale_kernel<float><<<grid_for(n, 256), 256, 0, st>>>((float2*)storage, n, scale);
    return (int)cudaGetLastError();
}

int launch_set_scalar(double* dst, double v, void* stream) {
    set_scalar_kernel<<<1, 1, 0, (cudaStream_t)stream>>>(dst, v);
    return (int)cudaGetLastError();
}

}  // namespace gpe
