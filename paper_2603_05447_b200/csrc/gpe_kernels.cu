// CUDA kernels (sm_100a) for the sparse-grid Gross-Pitaevskii hot path: fused stencil + potential +
// nonlinear term + Runge-Kutta / imaginary-time combination over the 8x8-column-tile layout.
//
//   H[psi;t] psi = -1/2 lap_h psi + V(r,t) psi + g|psi|^2 psi      PAPER.md:27 Eq. 2, :71 Eq. 8
//   psi = 0 outside the region of interest
//   RK4 in stage-state form                                        PAPER.md:276-281 Eq. A6-A7, :315-319 A10-A11
//   imaginary time: Euler step + particle-number partial sums,
//   renormalisation applied lazily at the next load                PAPER.md:60 Eq. 6, :87 (kernels K1-K3)
//
// One thread block = one WorkRec: nz <= kz consecutive z-planes of one tile.
//   phase 0: the slab entries (mask, base) of the own tile and its 4 neighbours -> shared memory
//   phase 1: (nz+2R) planes of (8+2R)x(8+2R) star-halo tile -> shared memory with cp.async; absent
//            points are zero-filled by cp.async's src-size = 0 (Dirichlet psi = 0); the same pass
//            writes the compact list of (plane, bit) codes of the block's own points
//   phase 2: one thread per ACTIVE point (compact index j = storage position - pos0, so the aux
//            loads and the stores are dense and coalesced): stencil from shared memory, V analytic,
//            nonlinear term, stage combination
//   phase 3 (IMAG / ENERGY): fixed-order block reduction -> partials[block]
#include <cuda_runtime.h>

#include <cstdint>

#include "gpe_internal.h"

namespace gpe {

namespace {

template <typename T> struct CxOf;
template <> struct CxOf<double> { using type = double2; };
template <> struct CxOf<float> { using type = float2; };

template <typename T> __device__ __forceinline__ typename CxOf<T>::type mk(T a, T b);
template <> __device__ __forceinline__ double2 mk<double>(double a, double b) { return make_double2(a, b); }
template <> __device__ __forceinline__ float2 mk<float>(float a, float b) { return make_float2(a, b); }

__device__ __forceinline__ void cp_async_zfill(void* smem_dst, const double2* src, bool valid) {
    unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    int sz = valid ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(d), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_zfill(void* smem_dst, const float2* src, bool valid) {
    unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    int sz = valid ? 8 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(d), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() {
    asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;\n" ::: "memory");
}

template <int R> struct Geo {
    static constexpr int PX = 8 + 2 * R;      // rows (x) of the shared tile
    static constexpr int PY = 8 + 2 * R;      // row pitch (y), elements
    static constexpr int PLANE = PX * PY;     // plane pitch, elements
    static constexpr int SLOTS = 64 + 32 * R; // lanes loaded per plane: own 64 + 4 star halos of 8R
};

// shared-memory carve-up (bytes), common to host and device
template <typename T, int R> struct Smem {
    using C = typename CxOf<T>::type;
    __host__ __device__ static constexpr size_t np(int kz) { return (size_t)(kz + 2 * R); }
    __host__ __device__ static constexpr size_t tile_off() { return 0; }
    __host__ __device__ static constexpr size_t slab_off(int kz) { return np(kz) * Geo<R>::PLANE * sizeof(C); }
    __host__ __device__ static constexpr size_t q_off(int kz) { return slab_off(kz) + 5 * np(kz) * sizeof(Slab); }
    __host__ __device__ static constexpr size_t red_off(int kz) { return q_off(kz) + (size_t)(16 + kz) * sizeof(double); }
    __host__ __device__ static constexpr size_t code_off(int kz) {
        return red_off(kz) + (size_t)(STAGE_THREADS / 32) * NACC * sizeof(double);
    }
    __host__ __device__ static constexpr size_t total(int kz) { return code_off(kz) + (size_t)64 * kz * sizeof(uint16_t); }
};

template <typename T, int R, int MODE>
__global__ void __launch_bounds__(STAGE_THREADS) stage_kernel(const StageParams p) {
    using C = typename CxOf<T>::type;
    using G = Geo<R>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int kz = p.kz;
    C* tile = reinterpret_cast<C*>(smem_raw + Smem<T, R>::tile_off());
    Slab* sslab = reinterpret_cast<Slab*>(smem_raw + Smem<T, R>::slab_off(kz));
    double* qx = reinterpret_cast<double*>(smem_raw + Smem<T, R>::q_off(kz));
    double* qy = qx + 8;
    double* qz = qx + 16;
    double* red = reinterpret_cast<double*>(smem_raw + Smem<T, R>::red_off(kz));
    uint16_t* codes = reinterpret_cast<uint16_t*>(smem_raw + Smem<T, R>::code_off(kz));

    const int tid = threadIdx.x;
    const WorkRec* __restrict__ w = p.work + blockIdx.x;
    const int z0 = w->z0, nz = w->nz;
    const int np = nz + 2 * R;
    const int npmax = kz + 2 * R;

    // ---- phase 0: slab entries and coordinate tables -------------------------------------------
    for (int idx = tid; idx < 5 * np; idx += STAGE_THREADS) {
        const int q = idx / np, zi = idx - q * np;
        const int zp = z0 - R + zi;
        Slab s;
        s.mask = 0ull;
        s.base = 0;
        if (zp >= w->zlo[q] && zp < w->zhi[q]) s = p.slabs[w->eoff[q] + zp];
        sslab[q * npmax + zi] = s;
    }
    {
        // ax x^2, ay y^2, az z^2 with one rounding per operation (same order as the mask, R2)
        if (tid < 8) {
            double x = __dadd_rn(__dmul_rn((double)(w->ix0 + tid) - 0.5 * (double)(p.pot.nx - 1), p.pot.h), p.pot.cx);
            qx[tid] = __dmul_rn(p.pot.ax, __dmul_rn(x, x));
        } else if (tid < 16) {
            double y = __dadd_rn(__dmul_rn((double)(w->iy0 + tid - 8) - 0.5 * (double)(p.pot.ny - 1), p.pot.h), p.pot.cy);
            qy[tid - 8] = __dmul_rn(p.pot.ay, __dmul_rn(y, y));
        } else if (tid >= 32 && tid < 32 + nz) {
            double z = __dadd_rn(__dmul_rn((double)(z0 + tid - 32) - 0.5 * (double)(p.pot.nz - 1), p.pot.h), p.pot.cz);
            qz[tid - 32] = __dmul_rn(p.pot.az, __dmul_rn(z, z));
        }
    }
    __syncthreads();

    // ---- phase 1: star-halo tile -> shared memory ----------------------------------------------
    const C* __restrict__ in = reinterpret_cast<const C*>(p.in);
    const long long pos0 = w->pos0;
    for (int it = tid; it < np * G::SLOTS; it += STAGE_THREADS) {
        const int zi = it / G::SLOTS;
        const int s = it - zi * G::SLOTS;
        int q, bit, dx, dy;  // source tile, source bit, destination (x, y) in the shared tile
        if (s < 64) {
            q = 0; bit = s; dx = (s >> 3) + R; dy = (s & 7) + R;
        } else {
            const int hh = s - 64;
            q = 1 + hh / (8 * R);
            const int r = hh - (q - 1) * (8 * R);
            if (q <= 2) {                       // -x / +x neighbour: R columns of 8
                const int ex = r >> 3, ly = r & 7;
                const int lx = (q == 1) ? (8 - R + ex) : ex;
                bit = lx * 8 + ly;
                dx = (q == 1) ? ex : (8 + R + ex);
                dy = ly + R;
            } else {                            // -y / +y neighbour: 8 rows of R
                const int lx = r / R, ey = r - lx * R;
                const int ly = (q == 3) ? (8 - R + ey) : ey;
                bit = lx * 8 + ly;
                dx = lx + R;
                dy = (q == 3) ? ey : (8 + R + ey);
            }
        }
        const Slab sl = sslab[q * npmax + zi];
        const bool on = (sl.mask >> bit) & 1ull;
        const long long pos = sl.base + __popcll(sl.mask & ((1ull << bit) - 1ull));
        cp_async_zfill(&tile[(zi * G::PX + dx) * G::PY + dy], on ? (in + pos) : in, on);
        if (q == 0 && on && zi >= R && zi < R + nz) codes[pos - pos0] = (uint16_t)(((zi - R) << 6) | bit);
    }
    cp_async_wait_all();
    __syncthreads();

    // ---- phase 2: one thread per active point --------------------------------------------------
    const T kw0 = (T)(-0.5 / (p.pot.h * p.pot.h) * 3.0 * (R == 1 ? -2.0 : -2.5));
    const T kw1 = (T)(-0.5 / (p.pot.h * p.pot.h) * (R == 1 ? 1.0 : 4.0 / 3.0));
    const T kw2 = (T)(-0.5 / (p.pot.h * p.pot.h) * (-1.0 / 12.0));
    const C* __restrict__ aux = reinterpret_cast<const C*>(p.aux);
    C* __restrict__ out1 = reinterpret_cast<C*>(p.out1);
    C* __restrict__ out2 = reinterpret_cast<C*>(p.out2);
    double sc = 1.0;
    if (MODE == MODE_IMAG) sc = *p.scale_in;
    double acc[NACC] = {0.0, 0.0, 0.0, 0.0};

    const int npts = w->npts;
    for (int j = tid; j < npts; j += STAGE_THREADS) {
        C a = mk<T>((T)0, (T)0);
        if (MODE == MODE_S2 || MODE == MODE_S3 || MODE == MODE_S4) a = aux[pos0 + j];
        const int code = codes[j];
        const int zl = code >> 6, lx = (code >> 3) & 7, ly = code & 7;
        const int ci = ((zl + R) * G::PX + lx + R) * G::PY + ly + R;
        const C c = tile[ci];
        C s1;
        {
            const C a0 = tile[ci - 1], a1 = tile[ci + 1], a2 = tile[ci - G::PY], a3 = tile[ci + G::PY];
            const C a4 = tile[ci - G::PLANE], a5 = tile[ci + G::PLANE];
            s1 = mk<T>(((a0.x + a1.x) + (a2.x + a3.x)) + (a4.x + a5.x), ((a0.y + a1.y) + (a2.y + a3.y)) + (a4.y + a5.y));
        }
        C tc = mk<T>(kw0 * c.x + kw1 * s1.x, kw0 * c.y + kw1 * s1.y);
        if (R == 2) {
            const C a0 = tile[ci - 2], a1 = tile[ci + 2], a2 = tile[ci - 2 * G::PY], a3 = tile[ci + 2 * G::PY];
            const C a4 = tile[ci - 2 * G::PLANE], a5 = tile[ci + 2 * G::PLANE];
            const C s2 = mk<T>(((a0.x + a1.x) + (a2.x + a3.x)) + (a4.x + a5.x), ((a0.y + a1.y) + (a2.y + a3.y)) + (a4.y + a5.y));
            tc.x += kw2 * s2.x;
            tc.y += kw2 * s2.y;
        }
        // V(r, t) analytically (Eq. 10 dressed form via BASELINE configs; R2)
        double v = 0.5 * ((qx[lx] + qy[ly]) + qz[zl]);
        if (p.pot.kind == GPE_POT_DRESSED) {
            const double d = v - p.pot.delta;
            v = sqrt(d * d + p.pot.omega * p.pot.omega) - p.pot.omega;
        }
        const T a2 = c.x * c.x + c.y * c.y;
        if (MODE == MODE_ENERGY) {
            acc[0] += (double)(c.x * tc.x + c.y * tc.y);
            acc[1] += v * (double)a2;
            acc[2] += (double)a2 * (double)a2;
            acc[3] += (double)a2;
            continue;
        }
        const T diag = (T)(v + p.g * (sc * sc) * (double)a2);
        const C hc = mk<T>(tc.x + diag * c.x, tc.y + diag * c.y);
        const T ca = (T)p.ca;
        C o;
        if (MODE == MODE_APPLY) {
            o = hc;
        } else if (MODE == MODE_IMAG) {
            const T s = (T)sc;
            o = mk<T>(s * (c.x - ca * hc.x), s * (c.y - ca * hc.y));
            acc[0] += (double)o.x * (double)o.x + (double)o.y * (double)o.y;
        } else {
            // f = -i H c = (hc.y, -hc.x)
            const C base = (MODE == MODE_S1) ? c : a;
            o = mk<T>(base.x + ca * hc.y, base.y - ca * hc.x);
            if (MODE == MODE_S4) {
                const T third = (T)(1.0 / 3.0);
                o.x += third * c.x;
                o.y += third * c.y;
            }
            if (MODE == MODE_S2) {
                const T third = (T)(1.0 / 3.0), tt = (T)(2.0 / 3.0);
                out2[pos0 + j] = mk<T>(third * (c.x - a.x) + tt * o.x, third * (c.y - a.y) + tt * o.y);
            }
        }
        out1[pos0 + j] = o;
    }

    // ---- phase 3: fixed-order block reduction ---------------------------------------------------
    if (MODE == MODE_IMAG || MODE == MODE_ENERGY) {
#pragma unroll
        for (int k = 0; k < NACC; ++k) {
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) acc[k] += __shfl_down_sync(0xffffffffu, acc[k], off);
        }
        if ((tid & 31) == 0) {
#pragma unroll
            for (int k = 0; k < NACC; ++k) red[(tid >> 5) * NACC + k] = acc[k];
        }
        __syncthreads();
        if (tid < NACC) {
            double s = 0.0;
            for (int wv = 0; wv < STAGE_THREADS / 32; ++wv) s += red[wv * NACC + tid];
            p.partials[(size_t)blockIdx.x * NACC + tid] = s;
        }
    }
}

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
        if (threadIdx.x == 0 && scale_out) scale_out[0] = sqrt(n_target / (h3 * s));
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

template <typename T, int R, int MODE>
cudaError_t launch_one(const StageParams& p, cudaStream_t st) {
    const size_t smem = Smem<T, R>::total(p.kz);
    stage_kernel<T, R, MODE><<<p.n_work, STAGE_THREADS, smem, st>>>(p);
    return cudaGetLastError();
}

template <typename T, int R>
cudaError_t launch_mode(int mode, const StageParams& p, cudaStream_t st) {
    switch (mode) {
        case MODE_APPLY: return launch_one<T, R, MODE_APPLY>(p, st);
        case MODE_S1: return launch_one<T, R, MODE_S1>(p, st);
        case MODE_S2: return launch_one<T, R, MODE_S2>(p, st);
        case MODE_S3: return launch_one<T, R, MODE_S3>(p, st);
        case MODE_S4: return launch_one<T, R, MODE_S4>(p, st);
        case MODE_IMAG: return launch_one<T, R, MODE_IMAG>(p, st);
        case MODE_ENERGY: return launch_one<T, R, MODE_ENERGY>(p, st);
    }
    return cudaErrorInvalidValue;
}

template <typename T, int R, int MODE>
cudaError_t set_attr() {
    return cudaFuncSetAttribute(stage_kernel<T, R, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
}
template <typename T, int R>
cudaError_t set_attr_modes() {
    cudaError_t e;
    if ((e = set_attr<T, R, MODE_APPLY>())) return e;
    if ((e = set_attr<T, R, MODE_S1>())) return e;
    if ((e = set_attr<T, R, MODE_S2>())) return e;
    if ((e = set_attr<T, R, MODE_S3>())) return e;
    if ((e = set_attr<T, R, MODE_S4>())) return e;
    if ((e = set_attr<T, R, MODE_IMAG>())) return e;
    if ((e = set_attr<T, R, MODE_ENERGY>())) return e;
    return cudaSuccess;
}

inline int grid_for(int64_t n, int threads) {
    int64_t b = (n + threads - 1) / threads;
    const int64_t cap = 148 * 32;
    if (b > cap) b = cap;
    if (b < 1) b = 1;
    return (int)b;
}

}  // namespace

size_t stage_smem_bytes(int dtype, int radius, int kz) {
    if (dtype == GPE_C128) return radius == 1 ? Smem<double, 1>::total(kz) : Smem<double, 2>::total(kz);
    return radius == 1 ? Smem<float, 1>::total(kz) : Smem<float, 2>::total(kz);
}

int kernels_configure() {
    cudaError_t e;
    if ((e = set_attr_modes<double, 1>())) return (int)e;
    if ((e = set_attr_modes<double, 2>())) return (int)e;
    if ((e = set_attr_modes<float, 1>())) return (int)e;
    if ((e = set_attr_modes<float, 2>())) return (int)e;
    return 0;
}

int launch_stage(int dtype, int radius, int mode, const StageParams& p, void* stream) {
    cudaStream_t st = (cudaStream_t)stream;
    if (p.n_work <= 0) return 0;
    if (dtype == GPE_C128) return (int)(radius == 1 ? launch_mode<double, 1>(mode, p, st) : launch_mode<double, 2>(mode, p, st));
    return (int)(radius == 1 ? launch_mode<float, 1>(mode, p, st) : launch_mode<float, 2>(mode, p, st));
}

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
