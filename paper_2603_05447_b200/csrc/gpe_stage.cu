// Fused stage kernels (sm_100a) of the sparse-grid Gross-Pitaevskii hot path: stencil + V(r,t) + nonlinear
// term + Runge-Kutta / imaginary-time combination over the 8x8-column-tile layout, one launch per stage.
//
//   H[psi;t] psi = -1/2 lap_h psi + V(r,t) psi + g|psi|^2 psi      PAPER.md:27 Eq. 2, :71 Eq. 8
//   psi = 0 outside the region of interest
//   RK4 in stage-state form                                        PAPER.md:276-281 Eq. A6-A7, :315-319 A10-A11
//   imaginary time: Euler step + particle-number partial sums,
//   renormalisation applied lazily at the next load                PAPER.md:60 Eq. 6, :87 (kernels K1-K3)
//
// Work decomposition: a STREAM is one WorkRec = nz <= 32 consecutive z-planes of one
// 8x8 column tile.  A warp marches one stream along z (PR = 2 rows per lane).  Lane t = (g, ly) = (t / 8, t % 8)
// owns the PRx1 patch rows lx = PR g .. PR g + PR-1 of column ly of every plane, so
//   - for a fixed patch element the 8 lanes of a row touch CONSECUTIVE storage positions: every global
//     load / store and every shared-memory access of a row group is a run of contiguous values
//     (full 32-byte sectors, no bank conflicts),
//   - z neighbours never leave registers (accumulate-forward form: psi(k-1..k-R) and the partial sums of
//     T psi for planes k-1..k-R are the only state),
//   - the x neighbours inside the patch are the lane's own registers.
// Tables: the slab entries (64-bit mask + storage base) of the own tile and of the four neighbour tiles for
// the planes the stream touches are copied to shared memory once at stream start; no table load sits on the
// per-plane critical path.
// Per plane: cp.async (zero-filled where the mask bit is clear: Dirichlet psi = 0) of the own patch, of the
// lane's share of the star halo (edge rows / columns of the four neighbour tiles) and of the aux operand
// (y0 or p) into rings of plane slots, PF planes in flight; one __syncwarp per plane, no block-level barrier.
// Plane c = k-R is finished when plane k has arrived: V(r,t) analytic, nonlinear term, stage combination,
// row-contiguous stores.  IMAG / ENERGY: per-stream partial sums in a fixed order -> partials[stream].
//
// Variants of the one kernel template: R = 1 / 2 (7- and 13-point stars), HOC (the paper's 19-point compact
// stencil, PAPER.md:341-343 Eq. B2: diagonal-tile tables, corner halo, in-plane face / diagonal sums carried
// along z), per-axis weights for anisotropic grids (Eq. B1), T = float / double, REAL (8-byte real-valued
// state for ground states), and the MODEs of gpe_internal.h: operator, RK stages S1-S4 and the
// general stage LC of Eq. A6-A7 (RKHE3, RKCK), Euler imaginary time, the paper's split iteration (K1 = KINP: the
// Eq. 7 half step applied to every staged value inside the kinetic kernel; K2 = SPLITB), energy sums.
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdlib>

#include "gpe_internal.h"

namespace gpe {

namespace {

template <typename T> struct CxOf;
template <> struct CxOf<double> { using type = double2; };
template <> struct CxOf<float> { using type = float2; };

template <typename T> __device__ __forceinline__ typename CxOf<T>::type mk(T a, T b);
template <> __device__ __forceinline__ double2 mk<double>(double a, double b) { return make_double2(a, b); }
template <> __device__ __forceinline__ float2 mk<float>(float a, float b) { return make_float2(a, b); }

// Storage element of a REAL-valued state (ground states by imaginary time need no imaginary part):
// 8 bytes in memory and in shared memory, widened to (x, 0) in registers, so every kernel below runs unchanged
// on half the bytes.
struct Re8 { double x; };
template <typename T, bool REAL> struct ElemOf { using type = typename CxOf<T>::type; };
template <> struct ElemOf<double, true> { using type = Re8; };
__device__ __forceinline__ double2 to_elem(double2 v, double2*) { return v; }
__device__ __forceinline__ float2 to_elem(float2 v, float2*) { return v; }
__device__ __forceinline__ Re8 to_elem(double2 v, Re8*) { Re8 r; r.x = v.x; return r; }

// cp.async of one complex value with zero fill (src-size 0 reads nothing and writes zeros: Dirichlet psi = 0)
__device__ __forceinline__ void cp_async_zfill(unsigned smem_dst, const double2* src, bool valid) {
    const int sz = valid ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(smem_dst), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_zfill(unsigned smem_dst, const float2* src, bool valid) {
    const int sz = valid ? 8 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(smem_dst), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_zfill(unsigned smem_dst, const Re8* src, bool valid) {
    const int sz = valid ? 8 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(smem_dst), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory");
}
__device__ __forceinline__ double2 lds_c(unsigned addr, double2*) {
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];\n" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ float2 lds_c(unsigned addr, float2*) {
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];\n" : "=f"(v.x), "=f"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ double2 lds_c(unsigned addr, Re8*) {
    double2 v;
    asm volatile("ld.shared.f64 %0, [%1];\n" : "=d"(v.x) : "r"(addr));
    v.y = 0.0;
    return v;
}
__device__ __forceinline__ void sts_c(unsigned addr, double2 v, double2*) {
    asm volatile("st.shared.v2.f64 [%0], {%1, %2};\n" ::"r"(addr), "d"(v.x), "d"(v.y) : "memory");
}
__device__ __forceinline__ void sts_c(unsigned addr, float2 v, float2*) {
    asm volatile("st.shared.v2.f32 [%0], {%1, %2};\n" ::"r"(addr), "f"(v.x), "f"(v.y) : "memory");
}
__device__ __forceinline__ void sts_c(unsigned addr, double2 v, Re8*) {
    asm volatile("st.shared.f64 [%0], %1;\n" ::"r"(addr), "d"(v.x) : "memory");
}
__device__ __forceinline__ uint2 lds_u2(unsigned addr) {
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];\n" : "=r"(v.x), "=r"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ unsigned lds_u1(unsigned addr) {
    unsigned v;
    asm volatile("ld.shared.u32 %0, [%1];\n" : "=r"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts_u2(unsigned addr, unsigned a, unsigned b) {
    asm volatile("st.shared.v2.u32 [%0], {%1, %2};\n" ::"r"(addr), "r"(a), "r"(b) : "memory");
}
__device__ __forceinline__ void sts_u1(unsigned addr, unsigned a) {
    asm volatile("st.shared.u32 [%0], %1;\n" ::"r"(addr), "r"(a) : "memory");
}

// sqrt(s) for s >= 0 from the hardware reciprocal-square-root seed (about 2^-23 relative), one coupled
// Newton step for g ~ sqrt(s) and h ~ 1/(2 sqrt(s)) (2^-45) and the residual correction g + (s - g^2) h, whose
// error is second order in the 2^-45 (relative error a few 1e-16 from rounding only; the IEEE-rounded sqrt()
// costs about three times the FP64 instructions).
__device__ __forceinline__ double fast_sqrt(double s) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;\n" : "=d"(y) : "d"(s));
    double g = s * y, h = 0.5 * y;
    double r = fma(-g, h, 0.5);
    g = fma(g, r, g);
    h = fma(h, r, h);
    r = fma(-g, g, s);          // residual s - g^2
    g = fma(r, h, g);
    return s > 0.0 ? g : 0.0;
}

// exp(-x) of the Eq. 7 propagator, x = V dt/2.  Ground-state runs have x of a few 1e-2 at most (cfg 2: V < 60,
// dt/2 = 2.5e-4), where the degree-8 Taylor polynomial is exact to the last bit or two (x^9/9! < 4e-17 for
// |x| < 1/16) at 8 FMAs; anything larger takes the library routine (a branch, uniform in practice).
__device__ __forceinline__ double exp_neg(double x) {
    if (fabs(x) < 0.0625) {
        const double r = -x;
        double q = 1.0 / 40320.0;
        q = fma(q, r, 1.0 / 5040.0);
        q = fma(q, r, 1.0 / 720.0);
        q = fma(q, r, 1.0 / 120.0);
        q = fma(q, r, 1.0 / 24.0);
        q = fma(q, r, 1.0 / 6.0);
        q = fma(q, r, 0.5);
        q = fma(q, r, 1.0);
        return fma(q, r, 1.0);
    }
    return exp(-x);
}

constexpr int KZMAX = 32;                 // planes per stream (host splits work items to at most this)
// planes in flight per stream (cp.async groups): the 7-point kernels are bound by global-load latency (84
// registers, small slots: three planes ahead), the 13-point ones by the shared-memory pipe (two)
#ifndef GPE_PF_R1
#define GPE_PF_R1 3
#endif
__host__ __device__ constexpr int pf_of(int radius) { return radius == 1 ? GPE_PF_R1 : 3; }
constexpr int STAGE_WARPS = STAGE_THREADS / 32;


// Shared memory of one stream.  Plane slot: (8+2R) rows (x) of PY values, the tile at rows/cols R..R+7 and
// the star halo around it.
template <typename T, int R, bool AUX, bool HOC = false, bool REAL = false> struct Geo {
    static constexpr int NT = HOC ? NTILE : 5;               // tiles whose slab tables are staged
    static constexpr int ES = (REAL ? 1 : 2) * (int)sizeof(T);
    static constexpr int ROWS = 8 + 2 * R;
    // row pitch in values; 8-byte values are read by half-warps (two rows, 2 apart): 2 PY 8 = 64 (mod 128) bytes
    static constexpr int PY = ES == 8 ? 12 : 8 + 2 * R;
    static constexpr int PLANE = ROWS * PY;                 // values per slot
    static constexpr int NE = KZMAX + 2 * R;                // table entries per tile
    static constexpr int NSLOT = pf_of(R) + 1;              // ring of plane slots per stream
    static constexpr int NAUX = pf_of(R) + 1;               // ring of aux-plane slots per stream
    static constexpr int RING_BYTES = NSLOT * PLANE * ES;
    static constexpr int AUX_BYTES = AUX ? NAUX * 64 * ES : 0;
    static constexpr int MASK_OFF = RING_BYTES + AUX_BYTES;  // [NT][NE] (lo, hi)
    static constexpr int BASE_OFF = MASK_OFF + NT * NE * 8;  // [NT][NE] storage base
    static constexpr int STREAM_BYTES = (BASE_OFF + NT * NE * 4 + 15) / 16 * 16;
    __host__ __device__ static constexpr int at(int r, int c) { return (r + R) * PY + (c + R); }
};

template <typename T> struct KW;   // stencil weights of the right type straight from the parameter block
template <> struct KW<double> {
    static __device__ __forceinline__ double w(const StageParams& p, int axis, int s) { return p.kw[axis][s]; }
    static __device__ __forceinline__ double c(const StageParams& p) { return p.kw[0][0]; }
    static __device__ __forceinline__ double e(const StageParams& p, int pair) { return p.ke[pair]; }
    static __device__ __forceinline__ double cn(const StageParams& p) { return p.kcn; }
};
template <> struct KW<float> {
    static __device__ __forceinline__ float w(const StageParams& p, int axis, int s) { return p.kwf[axis][s]; }
    static __device__ __forceinline__ float c(const StageParams& p) { return p.kwf[0][0]; }
    static __device__ __forceinline__ float e(const StageParams& p, int pair) { return p.kef[pair]; }
    static __device__ __forceinline__ float cn(const StageParams& p) { return p.kcnf; }
};

// imaginary part of a value: identically zero for a real-valued state (REAL), where it is not computed at all
#define YV(expr) (REAL ? (T)0 : (T)(expr))

// acc += w * v for a real weight and a complex value: complex64 uses Blackwell's packed FP32 FMA (FFMA2: both
// components in one instruction, same rounding as two FFMAs)
template <bool REAL> __device__ __forceinline__ void caxpy(double2& acc, double w, const double2& v) {
    acc.x = fma(w, v.x, acc.x);
    if (!REAL) acc.y = fma(w, v.y, acc.y);
}
template <bool REAL> __device__ __forceinline__ void caxpy(float2& acc, float w, const float2& v) {
    acc = __ffma2_rn(make_float2(w, w), v, acc);
}

__host__ __device__ constexpr bool mode_has_aux(int mode) { return mode == MODE_S2 || mode == MODE_S3 || mode == MODE_S4; }

template <typename T, int R, int MODE, int PR, bool HOC, bool REAL>
__global__ void __launch_bounds__(STAGE_THREADS, 16)
stage_kernel(const __grid_constant__ StageParams p) {
    static_assert(!HOC || (R == 1 && PR == 2), "the 19-point stencil has radius 1 and runs with a warp per stream");
    static_assert(!REAL || sizeof(T) == 8, "the real-valued state is fp64");
    static_assert(MODE != MODE_KINP || pf_of(R) >= 2, "K1 works on the plane after the current one: two planes must have landed");
    using C = typename CxOf<T>::type;                      // value in registers
    using EL = typename ElemOf<T, REAL>::type;             // value in memory
    constexpr bool HAS_AUX = mode_has_aux(MODE);
    using G = Geo<T, R, HAS_AUX, HOC, REAL>;
    constexpr int NT = G::NT;
    constexpr int PF = pf_of(R), NSLOT = G::NSLOT, NAUX = G::NAUX;
    constexpr unsigned ES = G::ES;
    constexpr int LPS = 64 / PR;                           // lanes per stream (16: half-warp, 32: warp)
    constexpr int SPW = 32 / LPS;                          // streams per warp
    constexpr int LPH = LPS / 4;                           // lanes per halo side
    constexpr int NHE = 8 * R / LPH;                       // halo values per lane and plane
    constexpr unsigned SLOT_BYTES = (unsigned)G::PLANE * ES;
    constexpr unsigned ROW_BYTES = (unsigned)G::PY * ES;
    extern __shared__ __align__(16) unsigned char smem_raw[];

    // Programmatic dependent launch: the next stage kernel of the stream may be scheduled as soon as every block of
    // this one has started (i.e. into the slots this kernel's tail leaves idle); it stages its tables, which no
    // kernel writes, and waits below (griddepcontrol.wait) for this kernel to complete before it touches psi.
    asm volatile("griddepcontrol.launch_dependents;\n" ::: "memory");
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int half = lane / LPS, t = lane % LPS;
    const int g = t >> 3, ly = t & 7;                      // row group and column of the PRx1 patch
    const int sidx = (blockIdx.x * STAGE_WARPS + warp) * SPW + half;   // this (half-)warp's stream
    const bool valid = sidx < p.n_work;
    const WorkRec* __restrict__ w = p.work + (valid ? sidx : 0);

    const int z0 = w->z0, nz = valid ? w->nz : 0;
    const int lead = w->lead;                              // overlap planes read below z0 (R, or 0: nothing there)
    const int kstart = z0 - lead;
    const int ne = nz > 0 ? nz + lead + R : 0;             // planes kstart .. kstart+ne-1 are touched

    const unsigned sb = (unsigned)__cvta_generic_to_shared(smem_raw) + (unsigned)((warp * SPW + half) * G::STREAM_BYTES);
    const unsigned ring = sb, auxring = sb + G::RING_BYTES, smask = sb + G::MASK_OFF, sbase = sb + G::BASE_OFF;

    // ---- slab tables of the five tiles -> shared memory (all loads in flight at once) ----------------
    {
        constexpr int NM = (G::NE + LPS - 1) / LPS;
        unsigned tl[NT * NM], th[NT * NM], tb[NT * NM];
#pragma unroll
        for (int q = 0; q < NT; ++q) {
            const int zl = w->zlo[q], zh = w->zhi[q];
            const Slab* __restrict__ tab = p.slabs + w->eoff[q];
#pragma unroll
            for (int m = 0; m < NM; ++m) {
                const int i = t + LPS * m, zp = kstart + i;
                tl[q * NM + m] = 0u; th[q * NM + m] = 0u; tb[q * NM + m] = 0u;
                if (i < ne && zp >= zl && zp < zh) {
                    const uint4 s = __ldg(reinterpret_cast<const uint4*>(tab + zp));
                    tl[q * NM + m] = s.x; th[q * NM + m] = s.y; tb[q * NM + m] = s.z;
                }
            }
        }
#pragma unroll
        for (int q = 0; q < NT; ++q)
#pragma unroll
            for (int m = 0; m < NM; ++m) {
                const int i = t + LPS * m;
                if (i < G::NE) {
                    sts_u2(smask + (unsigned)((q * G::NE + i) * 8), tl[q * NM + m], th[q * NM + m]);
                    sts_u1(sbase + (unsigned)((q * G::NE + i) * 4), tb[q * NM + m]);
                }
            }
    }

    // ---- lane constants ---------------------------------------------------------------------------------
    const bool ghi = PR * g >= 4;                          // own rows live in the high mask word
    const int rb0 = ((PR * g) & 3) * 8 + ly;               // bit of own element 0 inside its word
    unsigned bm[PR];                                       // bits below own element e inside its word
#pragma unroll
    for (int e = 0; e < PR; ++e) bm[e] = (1u << (rb0 + 8 * e)) - 1u;
    const unsigned own_off = (unsigned)G::at(PR * g, ly) * ES;         // + e * ROW_BYTES
    const unsigned aux_off = (unsigned)(8 * PR * g + ly) * ES;         // + e * 8 * ES
    // halo duty: neighbour tile hq (0..3 = -x,+x,-y,+y), values LPH*e + hj of its 8R-value edge
    const int hq = t / LPH, hj = t % LPH;
    unsigned hbm[NHE], hoff[NHE];
    int hdr[NHE], hdc[NHE];                                // position of halo value e relative to the tile's (0, 0) column
    bool hhi[NHE];                                         // value e lives in the high mask word
#pragma unroll
    for (int e = 0; e < NHE; ++e) {
        const int idx = LPH * e + hj;
        int nlx, nly, drow, dcol;
        if (hq < 2) {
            const int rr = idx >> 3, cc = idx & 7;
            nlx = hq == 0 ? 8 - R + rr : rr; nly = cc;
            drow = hq == 0 ? rr - R : 8 + rr; dcol = cc;
        } else {
            const int rr = idx / R, cc = idx % R;
            nlx = rr; nly = hq == 2 ? 8 - R + cc : cc;
            drow = rr; dcol = hq == 2 ? cc - R : 8 + cc;
        }
        hdr[e] = drow; hdc[e] = dcol;
        hbm[e] = (1u << ((nlx * 8 + nly) & 31)) - 1u;
        hhi[e] = nlx >= 4;
        hoff[e] = (unsigned)((drow + R) * G::PY + (dcol + R)) * ES;
    }

    // 19-point: lanes 0..3 fetch the corner (-x,-y), (-x,+y), (+x,-y), (+x,+y): local point (7,7), (7,0), (0,7), (0,0)
    // of the diagonal tile, bit cbit of its high (t < 2) or low mask word
    const int cbit = t == 0 ? 31 : (t == 1 ? 24 : (t == 2 ? 7 : 0));
    const unsigned coff = (unsigned)G::at((t & 2) ? 8 : -1, (t & 1) ? 8 : -1) * ES;
    const EL* __restrict__ in = reinterpret_cast<const EL*>(p.in);
    const EL* __restrict__ auxp = reinterpret_cast<const EL*>(p.aux);

    // potential: u = qxy[e] + qz(plane); qxy = 1/2 (ax x^2 + ay y^2) of the patch points
    double qxy[PR];
    {
        const double y = ((double)(w->iy0 + ly) - p.yc) * p.pot.hy + p.pot.cy;
        const double qy = p.hay * (y * y);
#pragma unroll
        for (int e = 0; e < PR; ++e) {
            const double x = ((double)(w->ix0 + PR * g + e) - p.xc) * p.pot.h + p.pot.cx;
            qxy[e] = fma(p.hax, x * x, qy);
        }
    }
    // K1: the same for the halo values (and the 19-point corner) this lane copies: it applies the Eq. 7 half step to them
    double qxh[NHE], qxc = 0.0;
    if (MODE == MODE_KINP) {
#pragma unroll
        for (int e = 0; e < NHE; ++e) {
            const double x = ((double)(w->ix0 + hdr[e]) - p.xc) * p.pot.h + p.pot.cx;
            const double y = ((double)(w->iy0 + hdc[e]) - p.yc) * p.pot.hy + p.pot.cy;
            qxh[e] = fma(p.hax, x * x, p.hay * (y * y));
        }
        if (HOC) {
            const double x = ((double)(w->ix0 + ((t & 2) ? 8 : -1)) - p.xc) * p.pot.h + p.pot.cx;
            const double y = ((double)(w->iy0 + ((t & 1) ? 8 : -1)) - p.yc) * p.pot.hy + p.pot.cy;
            qxc = fma(p.hax, x * x, p.hay * (y * y));
        }
    }
    // everything above read the work record and the slab tables only; psi, the aux operand and the lazy scale are
    // written by the kernels before this one
    asm volatile("griddepcontrol.wait;\n" ::: "memory");
    double sc = 1.0, gsc = p.g;
    if (MODE == MODE_IMAG || MODE == MODE_PREP || MODE == MODE_KINP) { sc = *p.scale_in; gsc = p.g * (sc * sc); }

    int niter = ne;
    if (SPW == 2) niter = max(niter, __shfl_xor_sync(0xffffffffu, niter, 16));   // both halves run the same loop
    __syncwarp();                                                  // tables visible to the half-warp

    // ---- producer: plane index i (plane kstart + i) -> slot sp; aux of plane i - R -> aux slot ap ------
    auto produce = [&](const int i, const unsigned sp, const unsigned ap) {
        if (i < ne) {
            {
                const uint2 m = lds_u2(smask + (unsigned)i * 8u);
                const unsigned word = ghi ? m.y : m.x;
                const unsigned bc = lds_u1(sbase + (unsigned)i * 4u) + (ghi ? (unsigned)__popc(m.x) : 0u);
                const unsigned dst = ring + sp * SLOT_BYTES + own_off;
#pragma unroll
                for (int e = 0; e < PR; ++e) {
                    const bool on = (word >> (rb0 + 8 * e)) & 1u;
                    cp_async_zfill(dst + (unsigned)e * ROW_BYTES, in + (bc + (unsigned)__popc(word & bm[e])), on);
                }
            }
            // 19-point: the overlap planes need their in-plane face sums too (they are the xz / yz edge neighbours)
            if (MODE != MODE_PREP && (HOC || (i >= lead && i < ne - R))) {
                const unsigned ti = (unsigned)((1 + hq) * G::NE + i);
                const uint2 m = lds_u2(smask + ti * 8u);
                const unsigned b = lds_u1(sbase + ti * 4u);
                const unsigned pl = (unsigned)__popc(m.x);
                const unsigned dst = ring + sp * SLOT_BYTES;
#pragma unroll
                for (int e = 0; e < NHE; ++e) {
                    const unsigned ww = hhi[e] ? m.y : m.x, bb = b + (hhi[e] ? pl : 0u);
                    const bool on = (ww & (hbm[e] + 1u)) != 0u;
                    cp_async_zfill(dst + hoff[e], in + (bb + (unsigned)__popc(ww & hbm[e])), on);
                }
            }
            if (HOC && MODE != MODE_PREP && t < 4) {
                // corner of the star-plus-diagonals halo: one point of the diagonal tile 5 + t
                const unsigned ti = (unsigned)((5 + t) * G::NE + i);
                const uint2 m = lds_u2(smask + ti * 8u);
                const unsigned ww = t < 2 ? m.y : m.x;
                const unsigned pos = lds_u1(sbase + ti * 4u) + (t < 2 ? (unsigned)__popc(m.x) : 0u) + (unsigned)__popc(ww & ((1u << cbit) - 1u));
                cp_async_zfill(ring + sp * SLOT_BYTES + coff, in + pos, (ww >> cbit) & 1u);
            }
            if (HAS_AUX) {
                const int ia = i - R;
                if (ia >= lead && ia < ne - R) {
                    const uint2 m = lds_u2(smask + (unsigned)ia * 8u);
                    const unsigned word = ghi ? m.y : m.x;
                    const unsigned bc = lds_u1(sbase + (unsigned)ia * 4u) + (ghi ? (unsigned)__popc(m.x) : 0u);
                    const unsigned dst = auxring + ap * (64u * ES) + aux_off;
#pragma unroll
                    for (int e = 0; e < PR; ++e)
                        if ((word >> (rb0 + 8 * e)) & 1u)
                            cp_async_zfill(dst + (unsigned)e * (8u * ES), auxp + (bc + (unsigned)__popc(word & bm[e])), true);
                }
            }
        }
        cp_async_commit();
    };

    // state (accumulate-forward form): set s holds psi and the partial T psi of one earlier plane
    C SP[R][PR], SA[R][PR];
#pragma unroll
    for (int s = 0; s < R; ++s)
#pragma unroll
        for (int e = 0; e < PR; ++e) { SP[s][e] = mk<T>((T)0, (T)0); SA[s][e] = mk<T>((T)0, (T)0); }
    double acc[NACC] = {0.0, 0.0, 0.0, 0.0};
    C GPV[PR];                                             // 19-point: edge contribution G of the previous plane
#pragma unroll
    for (int e = 0; e < PR; ++e) GPV[e] = mk<T>((T)0, (T)0);

    // ---- prologue: planes 0 .. PF-1 in flight ----------------------------------------------------------------
#pragma unroll
    for (int i = 0; i < PF; ++i) produce(i, (unsigned)i, (unsigned)((i + NAUX - (R % NAUX)) % NAUX));

    // K1: every value this lane copied for plane index j -- its patch, its share of the halo, its
    // corner -- is replaced in the slot by a = s c exp(-V ca) (1 - g ca |s c|^2) (Eq. 7 with the linearised interaction
    // factor, the lazy scale s of the previous iteration): the arithmetic of MODE_PREP at the point itself, so the result
    // does not depend on which tile stages the value; zero-filled points stay zero.  Done one plane step ahead of the
    // stencil (the copies of plane j have landed for THIS lane after its wait_group; the other lanes see the result
    // after the next __syncwarp), so that the dependent chain load -> V -> exp -> store overlaps the previous plane's work.
    auto half_step_plane = [&](const int j, const unsigned sj) {
        if (j >= ne) return;
        const double zk = ((double)(kstart + j) - p.zc) * p.pot.hz + p.pot.cz;
        const double qzk = p.haz * (zk * zk) - p.delta_eff;
        auto half_step = [&](const C c, const double q) -> C {
            double vp = q + qzk;
            if (p.pot.kind == GPE_POT_DRESSED) vp = fast_sqrt(fma(vp, vp, p.om2)) - p.pot.omega;
            const double c2 = (double)c.x * (double)c.x + (double)c.y * (double)c.y;
            const T f = (T)(sc * exp_neg(vp * p.ca) * fma(-gsc * p.ca, c2, 1.0));
            return mk<T>(c.x * f, YV(c.y * f));
        };
        const unsigned sa = ring + sj * SLOT_BYTES;
#pragma unroll
        for (int e = 0; e < PR; ++e) {
            const C c = lds_c(sa + own_off + (unsigned)e * ROW_BYTES, (EL*)nullptr);
            sts_c(sa + own_off + (unsigned)e * ROW_BYTES, half_step(c, qxy[e]), (EL*)nullptr);
        }
        if (HOC || (j >= lead && j < ne - R)) {
#pragma unroll
            for (int e = 0; e < NHE; ++e) {
                const C c = lds_c(sa + hoff[e], (EL*)nullptr);
                sts_c(sa + hoff[e], half_step(c, qxh[e]), (EL*)nullptr);
            }
            if (HOC && t < 4) {
                const C c = lds_c(sa + coff, (EL*)nullptr);
                sts_c(sa + coff, half_step(c, qxc), (EL*)nullptr);
            }
        }
    };
    if (MODE == MODE_KINP) {
        cp_async_wait<PF - 1>();
        half_step_plane(0, 0u);
    }

    // one plane step at plane index i (plane k = kstart + i).  (PN, AN) = set of plane k-1, (PO, AO) = set of
    // plane k-R (the same set for R = 1).  sl = ring slot of plane i; al = aux slot of plane i - R.
    auto step = [&](C (&PN)[PR], C (&AN)[PR], C (&PO)[PR], C (&AO)[PR], const int i, const unsigned sl, const unsigned al) {
        if (MODE == MODE_KINP) cp_async_wait<PF - 2>(); else cp_async_wait<PF - 1>();
        __syncwarp();
        {
            unsigned sp = sl + PF, ap = al + PF;
            if (sp >= NSLOT) sp -= NSLOT;
            if (ap >= NAUX) ap -= NAUX;
            produce(i + PF, sp, ap);
        }
        if (i >= ne) return;
        if (MODE == MODE_KINP) half_step_plane(i + 1, sl + 1 == NSLOT ? 0u : sl + 1);
        const unsigned so = ring + sl * SLOT_BYTES + own_off;   // own patch in the slot of plane k
        const int ic = i - R;                                   // plane finished in this step
        // ---- output plane: activity bits and storage positions --------------------------------------------
        unsigned cword = 0u, cbase = 0u;
        bool cany = false;                                      // the slab of plane c holds points (stream-uniform)
        if (ic >= lead) {
            const uint2 m = lds_u2(smask + (unsigned)ic * 8u);
            cword = ghi ? m.y : m.x;
            cbase = lds_u1(sbase + (unsigned)ic * 4u) + (ghi ? (unsigned)__popc(m.x) : 0u);
            cany = (m.x | m.y) != 0u;
        }
        // ---- MODE_LC: the earlier stage states of plane c, plain loads issued before anything else of the step ----
        C lcs[PR];
        if (MODE == MODE_LC) {
#pragma unroll
            for (int e = 0; e < PR; ++e) lcs[e] = mk<T>((T)0, (T)0);
            if (cany && !REAL) {
#pragma unroll
                for (int j = 0; j < MAX_LC_AUX; ++j) {
                    if (j < p.n_aux) {
                        // the last RKCK stage writes y_new over y^(1) = auxn[0]: plain loads, no read-only path, no restrict
                        const C* aj = reinterpret_cast<const C*>(p.auxn[j]);
                        const T cj = (T)p.coef[j];
#pragma unroll
                        for (int e = 0; e < PR; ++e) {
                            if ((cword >> (rb0 + 8 * e)) & 1u) {
                                const C a = aj[REAL ? 0u : cbase + (unsigned)__popc(cword & bm[e])];
                                lcs[e].x = fma(cj, a.x, lcs[e].x);
                                lcs[e].y = fma(cj, a.y, lcs[e].y);
                            }
                        }
                    }
                }
            }
        }
        // ---- MODE_LC: warm the L2 with the earlier stage states of the plane finished two steps from now (the
        //      loads above are consumed within their own step: from DRAM they would stall it) -------------------
        if (MODE == MODE_LC && !REAL) {
            const int ip = ic + 2;
            if (ip >= lead && ip < ne - R) {
                const uint2 m = lds_u2(smask + (unsigned)ip * 8u);
                const unsigned wd = ghi ? m.y : m.x;
                const unsigned bs = lds_u1(sbase + (unsigned)ip * 4u) + (ghi ? (unsigned)__popc(m.x) : 0u);
#pragma unroll
                for (int j = 0; j < MAX_LC_AUX; ++j) {
                    if (j < p.n_aux) {
                        const C* aj = reinterpret_cast<const C*>(p.auxn[j]);
#pragma unroll
                        for (int e = 0; e < PR; ++e)
                            if ((wd >> (rb0 + 8 * e)) & 1u)
                                asm volatile("prefetch.global.L2 [%0];\n" ::"l"(aj + (bs + (unsigned)__popc(wd & bm[e]))));
                    }
                }
            }
        }
        // ---- psi(k) of the patch ------------------------------------------------------------------------
        C v[PR];
#pragma unroll
        for (int e = 0; e < PR; ++e) v[e] = lds_c(so + (unsigned)e * ROW_BYTES, (EL*)nullptr);
        // ---- V(r,t) of plane c: depends on coordinates only, so its dependency chains (one per patch point,
        //      interleaved) are issued here and overlap the shared-memory latency of psi(k) --------------------
        double vpot[PR];
        if (cany && MODE != MODE_KIN && MODE != MODE_KINP) {
            const double zc = ((double)(kstart + ic) - p.zc) * p.pot.hz + p.pot.cz;
            const double qz = p.haz * (zc * zc) - p.delta_eff;
#pragma unroll
            for (int e = 0; e < PR; ++e) vpot[e] = qxy[e] + qz;
            if (p.pot.kind == GPE_POT_DRESSED) {
#pragma unroll
                for (int e = 0; e < PR; ++e) vpot[e] = fast_sqrt(fma(vpot[e], vpot[e], p.om2)) - p.pot.omega;
            }
        }
        // ---- 19-point: in-plane face sums (x and y) and diagonal sum E of the patch points in plane k; G = the
        //      part of plane k that the neighbouring planes see as their xz / yz edge neighbours ----------------
        C Fx[PR], Fy[PR], E[PR], G[PR];
        if (HOC && MODE != MODE_PREP) {
            C Lc[4], Rc[4], Mc[4];                              // columns ly-1, ly+1, ly of rows -1 .. 2 of the patch
#pragma unroll
            for (int r = -1; r <= 2; ++r) {
                Lc[r + 1] = lds_c(so + (unsigned)(r * (int)ROW_BYTES - (int)ES), (EL*)nullptr);
                Rc[r + 1] = lds_c(so + (unsigned)(r * (int)ROW_BYTES + (int)ES), (EL*)nullptr);
                Mc[r + 1] = (r == 0 || r == 1) ? v[r == 1 ? 1 : 0] : lds_c(so + (unsigned)(r * (int)ROW_BYTES), (EL*)nullptr);
            }
#pragma unroll
            for (int a = 0; a < PR; ++a) {
                Fx[a] = mk<T>(Mc[a].x + Mc[a + 2].x, YV(Mc[a].y + Mc[a + 2].y));
                Fy[a] = mk<T>(Lc[a + 1].x + Rc[a + 1].x, YV(Lc[a + 1].y + Rc[a + 1].y));
                E[a] = mk<T>((Lc[a].x + Rc[a].x) + (Lc[a + 2].x + Rc[a + 2].x), YV((Lc[a].y + Rc[a].y) + (Lc[a + 2].y + Rc[a + 2].y)));
                // what planes k-1 and k+1 see of plane k: xz / yz edge neighbours and (27-point) the corners
                G[a] = mk<T>(fma(KW<T>::e(p, 1), Fx[a].x, fma(KW<T>::e(p, 2), Fy[a].x, KW<T>::cn(p) * E[a].x)),
                             YV(fma(KW<T>::e(p, 1), Fx[a].y, fma(KW<T>::e(p, 2), Fy[a].y, KW<T>::cn(p) * E[a].y))));
            }
        }
        // ---- psi(k) completes the z part of planes k-1 .. k-R -------------------------------------------
#pragma unroll
        for (int e = 0; e < PR; ++e) {
            caxpy<REAL>(AO[e], KW<T>::w(p, 2, R), v[e]);
            if (R == 2) {
                caxpy<REAL>(AN[e], KW<T>::w(p, 2, 1), v[e]);
            }
            if (HOC && MODE != MODE_PREP) {                     // the xz / yz edge neighbours of plane k-1 in plane k
                AO[e].x += G[e].x;
                AO[e].y = YV(AO[e].y + G[e].y);
            }
        }
        // ---- finish plane c = k - R: nonlinear term, stage combination (branch-free; stores predicated) ----
        if (cany) {
            C av[PR];
#pragma unroll
            for (int e = 0; e < PR; ++e) {
                av[e] = mk<T>((T)0, (T)0);
                if (HAS_AUX) av[e] = lds_c(auxring + al * (64u * ES) + aux_off + (unsigned)e * (8u * ES), (EL*)nullptr);
            }
#pragma unroll
            for (int e = 0; e < PR; ++e) {
                const bool on = (cword >> (rb0 + 8 * e)) & 1u;
                const unsigned pos = cbase + (unsigned)__popc(cword & bm[e]);
                const C cv = PO[e];
                const C tc = AO[e];
                const T a2 = REAL ? cv.x * cv.x : fma(cv.x, cv.x, cv.y * cv.y);
                if (MODE == MODE_ENERGY) {
                    // inactive lanes hold cv = 0 and finite tc: they add exact zeros
                    acc[0] += (double)(cv.x * tc.x + cv.y * tc.y);
                    acc[1] += vpot[e] * (double)a2;
                    acc[2] += (double)a2 * (double)a2;
                    acc[3] += (double)a2;
                    continue;
                }
                if (MODE == MODE_PREP || MODE == MODE_KIN || MODE == MODE_KINP || MODE == MODE_SPLITB) {
                    // the paper's split iteration: Euler half step of the kinetic part and / or the diagonal
                    // propagator exp(-V ca) (1 - g ca |u|^2) of Eq. 7 with the linearised interaction factor
                    const T ca = (T)p.ca;
                    C u = cv;
                    if (MODE != MODE_PREP) u = mk<T>(fma(-ca, tc.x, cv.x), YV(fma(-ca, tc.y, cv.y)));
                    C o = u;
                    if (MODE != MODE_KIN && MODE != MODE_KINP) {
                        const double u2 = (double)u.x * (double)u.x + (double)u.y * (double)u.y;
                        const T f = (T)(sc * exp_neg(vpot[e] * p.ca) * fma(-gsc * p.ca, u2, 1.0));
                        o = mk<T>(u.x * f, YV(u.y * f));
                    }
                    if (MODE == MODE_SPLITB) {
                        const double o2 = (double)o.x * (double)o.x + (double)o.y * (double)o.y;
                        acc[0] += on ? o2 : 0.0;
                    }
                    if (on) reinterpret_cast<EL*>(p.out1)[pos] = to_elem(o, (EL*)nullptr);
                    continue;
                }
                const T diag = (T)fma(gsc, (double)a2, vpot[e]);
                const C hc = mk<T>(fma(diag, cv.x, tc.x), YV(fma(diag, cv.y, tc.y)));
                const T ca = (T)p.ca;
                C o;
                if (MODE == MODE_APPLY) {
                    o = hc;
                } else if (MODE == MODE_IMAG) {
                    const T s = (T)sc;
                    o = mk<T>(s * fma(-ca, hc.x, cv.x), YV(s * fma(-ca, hc.y, cv.y)));
                    const double o2 = (double)o.x * (double)o.x + (double)o.y * (double)o.y;
                    acc[0] += on ? o2 : 0.0;
                } else if (MODE == MODE_LC) {
                    const T cc = (T)p.coefc;
                    o = mk<T>(fma(ca, hc.y, fma(cc, cv.x, lcs[e].x)), fma(-ca, hc.x, fma(cc, cv.y, lcs[e].y)));
                } else {
                    // f = -i H c = (hc.y, -hc.x)
                    const C base = (MODE == MODE_S1) ? cv : av[e];
                    o = mk<T>(fma(ca, hc.y, base.x), fma(-ca, hc.x, base.y));
                    if (MODE == MODE_S4) {
                        const T third = (T)(1.0 / 3.0);
                        o.x = fma(third, cv.x, o.x);
                        o.y = fma(third, cv.y, o.y);
                    }
                    if (MODE == MODE_S2) {
                        const T b0 = (T)p.comb[0], b1 = (T)p.comb[1], b2 = (T)p.comb[2];
                        const C o2 = mk<T>(fma(b2, o.x, fma(b1, cv.x, b0 * av[e].x)), fma(b2, o.y, fma(b1, cv.y, b0 * av[e].y)));
                        if (on) reinterpret_cast<EL*>(p.out2)[pos] = to_elem(o2, (EL*)nullptr);
                    }
                }
                if (on) reinterpret_cast<EL*>(p.out1)[pos] = to_elem(o, (EL*)nullptr);
            }
        }
        // ---- the oldest set becomes the set of plane k: z-backward part, centre ---------------------------------
#pragma unroll
        for (int e = 0; e < PR; ++e) {
            C an;
            if (R == 2) {
                an.x = KW<T>::w(p, 2, 2) * PO[e].x;
                an.y = YV(KW<T>::w(p, 2, 2) * PO[e].y);
                caxpy<REAL>(an, KW<T>::w(p, 2, 1), PN[e]);
            } else {
                an.x = KW<T>::w(p, 2, 1) * PO[e].x;
                an.y = YV(KW<T>::w(p, 2, 1) * PO[e].y);
            }
            AO[e] = an;
            caxpy<REAL>(AO[e], KW<T>::c(p), v[e]);
            PO[e] = v[e];
            if (HOC && MODE != MODE_PREP) {
                // faces and diagonals of plane k, and plane k-1's share of the xz / yz edges
                AO[e].x = fma(KW<T>::w(p, 0, 1), Fx[e].x, fma(KW<T>::w(p, 1, 1), Fy[e].x, fma(KW<T>::e(p, 0), E[e].x, AO[e].x + GPV[e].x)));
                AO[e].y = YV(fma(KW<T>::w(p, 0, 1), Fx[e].y, fma(KW<T>::w(p, 1, 1), Fy[e].y, fma(KW<T>::e(p, 0), E[e].y, AO[e].y + GPV[e].y))));
                GPV[e] = G[e];
            }
        }
        // ---- in-plane part (only planes of the stream itself are ever finished) ----------------------------------
        if (!HOC && MODE != MODE_PREP && i >= lead && i < ne - R) {
            // x direction: source rows r = -R .. PR-1+R of column ly; rows 0..PR-1 are the patch itself
#pragma unroll
            for (int r = -R; r <= PR - 1 + R; ++r) {
                const C val = (r >= 0 && r < PR) ? v[r < 0 ? 0 : (r < PR ? r : 0)] : lds_c(so + (unsigned)(r * (int)ROW_BYTES), (EL*)nullptr);
#pragma unroll
                for (int a = 0; a < PR; ++a) {
                    const int d = r > a ? r - a : a - r;
                    if (d >= 1 && d <= R) {
                        caxpy<REAL>(AO[a], KW<T>::w(p, 0, d), val);
                    }
                }
            }
            // y direction: columns ly +- 1 .. R of each patch row
#pragma unroll
            for (int a = 0; a < PR; ++a) {
#pragma unroll
                for (int cc = -R; cc <= R; ++cc) {
                    if (cc == 0) continue;
                    const C val = lds_c(so + (unsigned)(a * (int)ROW_BYTES + cc * (int)ES), (EL*)nullptr);
                    const int d = cc > 0 ? cc : -cc;
                    caxpy<REAL>(AO[a], KW<T>::w(p, 1, d), val);
                }
            }
        }
    };

    unsigned sl = 0, al = (unsigned)((NAUX - (R % NAUX)) % NAUX);   // slots of plane index i and of plane i - R
    for (int it = 0; it < niter; it += R) {
        if (R == 1) {
            step(SP[0], SA[0], SP[0], SA[0], it, sl, al);
            sl = (sl + 1 == NSLOT) ? 0 : sl + 1;
            al = (al + 1 == NAUX) ? 0 : al + 1;
        } else {
            step(SP[0], SA[0], SP[R - 1], SA[R - 1], it, sl, al);
            sl = (sl + 1 == NSLOT) ? 0 : sl + 1;
            al = (al + 1 == NAUX) ? 0 : al + 1;
            if (it + 1 < niter) {
                step(SP[R - 1], SA[R - 1], SP[0], SA[0], it + 1, sl, al);
                sl = (sl + 1 == NSLOT) ? 0 : sl + 1;
                al = (al + 1 == NAUX) ? 0 : al + 1;
            }
        }
    }
    cp_async_wait<0>();

    // ---- per-stream partial sums in a fixed order (bit-reproducible, independent of scheduling) -------
    if (MODE == MODE_IMAG || MODE == MODE_ENERGY || MODE == MODE_SPLITB) {
#pragma unroll
        for (int kq = 0; kq < NACC; ++kq)
#pragma unroll
            for (int off = LPS / 2; off > 0; off >>= 1) acc[kq] += __shfl_down_sync(0xffffffffu, acc[kq], off, LPS);
        if (t == 0 && valid) {
#pragma unroll
            for (int kq = 0; kq < NACC; ++kq) p.partials[(size_t)sidx * NACC + kq] = acc[kq];
        }
    }
}

// rows per lane: complex128 lanes carry 2 rows (a warp per stream: half the registers, twice the resident
// warps).  complex64 runs the same way: 4 rows per lane (a half-warp per stream, two streams per warp) measured
// 9.8e10 stage updates/s on cfg 4 against 1.2e11 with 2 rows (twice the shared memory per warp: 11 warps per SM)
template <typename T> constexpr int rows_per_lane() { return 2; }

template <typename T, int R, int MODE, bool HOC, bool REAL> constexpr size_t stage_smem() {
    return (size_t)(STAGE_WARPS * rows_per_lane<T>() / 2) * Geo<T, R, mode_has_aux(MODE), HOC, REAL>::STREAM_BYTES;
}

// where a stage launch goes: the stream, and whether it may start under programmatic dependent launch
// (gpe_sim_set_option GPE_OPT_PDL; 0 = plain stream-ordered launches)
struct LaunchAt {
    cudaStream_t stream;
    int pdl;
};

template <typename T, int R, int MODE, bool HOC, bool REAL>
cudaError_t launch_one(const StageParams& p, LaunchAt st) {
    constexpr int spb = STAGE_WARPS * rows_per_lane<T>() / 2;   // streams per block
    const int nblk = (p.n_work + spb - 1) / spb;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)nblk);
    cfg.blockDim = dim3(STAGE_THREADS);
    cfg.dynamicSmemBytes = stage_smem<T, R, MODE, HOC, REAL>();
    cfg.stream = st.stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = st.pdl ? 1 : 0;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, stage_kernel<T, R, MODE, rows_per_lane<T>(), HOC, REAL>, p);
}

template <typename T, int R, bool HOC>
cudaError_t launch_mode(int mode, const StageParams& p, LaunchAt st) {
    switch (mode) {
        case MODE_APPLY: return launch_one<T, R, MODE_APPLY, HOC, false>(p, st);
        case MODE_S1: return launch_one<T, R, MODE_S1, HOC, false>(p, st);
        case MODE_S2: return launch_one<T, R, MODE_S2, HOC, false>(p, st);
        case MODE_S3: return launch_one<T, R, MODE_S3, HOC, false>(p, st);
        case MODE_S4: return launch_one<T, R, MODE_S4, HOC, false>(p, st);
        case MODE_IMAG: return launch_one<T, R, MODE_IMAG, HOC, false>(p, st);
        case MODE_ENERGY: return launch_one<T, R, MODE_ENERGY, HOC, false>(p, st);
        case MODE_PREP: return launch_one<T, R, MODE_PREP, HOC, false>(p, st);
        case MODE_KIN: return launch_one<T, R, MODE_KIN, HOC, false>(p, st);
        case MODE_SPLITB: return launch_one<T, R, MODE_SPLITB, HOC, false>(p, st);
        case MODE_LC: return launch_one<T, R, MODE_LC, HOC, false>(p, st);
        case MODE_KINP: return launch_one<T, R, MODE_KINP, HOC, false>(p, st);
    }
    return cudaErrorInvalidValue;
}

// real-valued fp64 state: the operator and the imaginary-time modes only (real time needs the imaginary part)
template <int R, bool HOC>
cudaError_t launch_mode_real(int mode, const StageParams& p, LaunchAt st) {
    switch (mode) {
        case MODE_APPLY: return launch_one<double, R, MODE_APPLY, HOC, true>(p, st);
        case MODE_IMAG: return launch_one<double, R, MODE_IMAG, HOC, true>(p, st);
        case MODE_ENERGY: return launch_one<double, R, MODE_ENERGY, HOC, true>(p, st);
        case MODE_PREP: return launch_one<double, R, MODE_PREP, HOC, true>(p, st);
        case MODE_KIN: return launch_one<double, R, MODE_KIN, HOC, true>(p, st);
        case MODE_SPLITB: return launch_one<double, R, MODE_SPLITB, HOC, true>(p, st);
        case MODE_KINP: return launch_one<double, R, MODE_KINP, HOC, true>(p, st);
    }
    return cudaErrorInvalidValue;
}

template <typename T, int R, int MODE, bool HOC, bool REAL>
cudaError_t set_attr() {
    return cudaFuncSetAttribute(stage_kernel<T, R, MODE, rows_per_lane<T>(), HOC, REAL>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)stage_smem<T, R, MODE, HOC, REAL>());
}
template <typename T, int R, bool HOC>
cudaError_t set_attr_modes() {
    cudaError_t e;
    if ((e = set_attr<T, R, MODE_APPLY, HOC, false>())) return e;
    if ((e = set_attr<T, R, MODE_S1, HOC, false>())) return e;
    if ((e = set_attr<T, R, MODE_S2, HOC, false>())) return e;
    if ((e = set_attr<T, R, MODE_S3, HOC, false>())) return e;
    if ((e = set_attr<T, R, MODE_S4, HOC, false>())) return e;
    if ((e = set_attr<T, R, MODE_IMAG, HOC, false>())) return e;
    if ((e = set_attr<T, R, MODE_ENERGY, HOC, false>())) return e;
    if ((e = set_attr<T, R, MODE_PREP, HOC, false>())) return e;
    if ((e = set_attr<T, R, MODE_KIN, HOC, false>())) return e;
    if ((e = set_attr<T, R, MODE_SPLITB, HOC, false>())) return e;
    if ((e = set_attr<T, R, MODE_LC, HOC, false>())) return e;
    if ((e = set_attr<T, R, MODE_KINP, HOC, false>())) return e;
    return cudaSuccess;
}
template <int R, bool HOC>
cudaError_t set_attr_modes_real() {
    cudaError_t e;
    if ((e = set_attr<double, R, MODE_APPLY, HOC, true>())) return e;
    if ((e = set_attr<double, R, MODE_IMAG, HOC, true>())) return e;
    if ((e = set_attr<double, R, MODE_ENERGY, HOC, true>())) return e;
    if ((e = set_attr<double, R, MODE_PREP, HOC, true>())) return e;
    if ((e = set_attr<double, R, MODE_KIN, HOC, true>())) return e;
    if ((e = set_attr<double, R, MODE_SPLITB, HOC, true>())) return e;
    if ((e = set_attr<double, R, MODE_KINP, HOC, true>())) return e;
    return cudaSuccess;
}

}  // namespace

int stage_max_planes() { return KZMAX; }

// variant: 1 = 7-point, 2 = 13-point, 3 = 19-point (gpe_internal.h)
size_t stage_smem_bytes(int dtype, int variant) {   // largest over the modes (the aux-carrying RK stages)
    if (dtype == GPE_C128)
        return variant == 1 ? stage_smem<double, 1, MODE_S2, false, false>()
                            : (variant == 2 ? stage_smem<double, 2, MODE_S2, false, false>() : stage_smem<double, 1, MODE_S2, true, false>());
    return variant == 1 ? stage_smem<float, 1, MODE_S2, false, false>()
                        : (variant == 2 ? stage_smem<float, 2, MODE_S2, false, false>() : stage_smem<float, 1, MODE_S2, true, false>());
}

int kernels_configure() {
    cudaError_t e;
    if ((e = set_attr_modes<double, 1, false>())) return (int)e;
    if ((e = set_attr_modes<double, 2, false>())) return (int)e;
    if ((e = set_attr_modes<double, 1, true>())) return (int)e;
    if ((e = set_attr_modes<float, 1, false>())) return (int)e;
    if ((e = set_attr_modes<float, 2, false>())) return (int)e;
    if ((e = set_attr_modes<float, 1, true>())) return (int)e;
    if ((e = set_attr_modes_real<1, false>())) return (int)e;
    if ((e = set_attr_modes_real<2, false>())) return (int)e;
    if ((e = set_attr_modes_real<1, true>())) return (int)e;
    return 0;
}

template <typename T>
cudaError_t launch_variant(int variant, int mode, const StageParams& p, LaunchAt st) {
    if (variant == 1) return launch_mode<T, 1, false>(mode, p, st);
    if (variant == 2) return launch_mode<T, 2, false>(mode, p, st);
    if (variant == 3) return launch_mode<T, 1, true>(mode, p, st);
    return cudaErrorInvalidValue;
}

int launch_stage(int dtype, int variant, int mode, const StageParams& p, void* stream, int pdl) {
    const LaunchAt st{(cudaStream_t)stream, pdl};
    if (p.n_work <= 0) return 0;
    if (dtype == GPE_R64) {
        if (variant == 1) return (int)launch_mode_real<1, false>(mode, p, st);
        if (variant == 2) return (int)launch_mode_real<2, false>(mode, p, st);
        if (variant == 3) return (int)launch_mode_real<1, true>(mode, p, st);
        return (int)cudaErrorInvalidValue;
    }
    return (int)(dtype == GPE_C128 ? launch_variant<double>(variant, mode, p, st) : launch_variant<float>(variant, mode, p, st));
}

}  // namespace gpe
