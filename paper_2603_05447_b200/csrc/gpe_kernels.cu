// CUDA kernels (sm_100a) for the sparse-grid Gross-Pitaevskii hot path: fused stencil + potential +
// nonlinear term + Runge-Kutta / imaginary-time combination over the 8x8-column-tile layout.
//
//   H[psi;t] psi = -1/2 lap_h psi + V(r,t) psi + g|psi|^2 psi      PAPER.md:27 Eq. 2, :71 Eq. 8
//   psi = 0 outside the region of interest
//   RK4 in stage-state form                                        PAPER.md:276-281 Eq. A6-A7, :315-319 A10-A11
//   imaginary time: Euler step + particle-number partial sums,
//   renormalisation applied lazily at the next load                PAPER.md:60 Eq. 6, :87 (kernels K1-K3)
//
// Work decomposition: a STREAM is one WorkRec = nz consecutive z-planes of one 8x8
// column tile.  A half-warp (16 threads) marches one stream along z; thread t owns the 2x2 patch
// (lx, ly) = (2*(t/4) + {0,1}, 2*(t%4) + {0,1}) of every plane, so
//   - z neighbours never leave registers (accumulate-forward form: psi(k-1..k-R) and the partial sums of
//     T psi for planes k-1..k-R are the only state),
//   - half of the in-plane neighbours are the thread's own patch values,
//   - per point only 1 + 2R/2 + 2R/2 shared-memory reads remain (5 for the 13-point stencil instead of 13).
// Per plane: cp.async (zero-filled where the mask bit is clear: Dirichlet psi = 0) of the own patch and of one
// patch of the star halo (the edge patches of the four neighbour tiles) into a 3-slot ring of plane buffers,
// two planes in flight; one __syncwarp per plane, no block-level barrier.  Plane c = k-R is finished when
// plane k has arrived: V(r,t) analytic, nonlinear term, stage combination, coalesced-by-rank stores.
// IMAG / ENERGY: per-stream partial sums in a fixed order -> partials[stream].
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

// cp.async of one complex value with zero fill (src-size 0 reads nothing and writes zeros: Dirichlet psi = 0)
__device__ __forceinline__ void cp_async_zfill(unsigned smem_dst, const double2* src, bool valid) {
    const int sz = valid ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(smem_dst), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_zfill(unsigned smem_dst, const float2* src, bool valid) {
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

// sqrt(s) for s >= 0 from the hardware reciprocal-square-root seed and two coupled Newton steps
// (relative error a few 1e-16; the IEEE-rounded sqrt() costs about twice the FP64 instructions).
__device__ __forceinline__ double fast_sqrt(double s) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;\n" : "=d"(y) : "d"(s));
    double g = s * y, h = 0.5 * y;
    double r = fma(-g, h, 0.5);
    g = fma(g, r, g);
    h = fma(h, r, h);
    r = fma(-g, h, 0.5);
    g = fma(g, r, g);
    h = fma(h, r, h);
    r = fma(-g, g, s);          // residual s - g^2
    g = fma(r, h, g);
    return s > 0.0 ? g : 0.0;
}

// Geometry of one plane slot in shared memory: (8+2R) rows (x) of PY elements; a row stores its even
// columns first and its odd columns HALFP elements later, so that the stride-2 column accesses of the
// 2x2 patches are bank-conflict free for 16-byte and 8-byte elements (PY = 2 mod 4).
template <int R> struct Geo {
    static constexpr int ROWS = 8 + 2 * R;
    static constexpr int PY = (R == 1) ? 10 : 14;
    static constexpr int HALFP = PY / 2;
    static constexpr int PLANE = ROWS * PY;                 // elements per slot
    // position inside a row of column (2*py + c) relative to py, c in [-R, 2+R)
    __host__ __device__ static constexpr int cpos(int c) { return ((c + R) & 1) * HALFP + ((c + R) >> 1); }
};

constexpr int PF = 2;                     // planes in flight per stream (cp.async groups)
constexpr int NSLOT = PF + 1;             // ring of plane slots per stream
constexpr int STAGE_WARPS = STAGE_THREADS / 32;
constexpr int STREAMS_PER_BLOCK = 2 * STAGE_WARPS;

// ranks and activity bits of the four points of patch (ppx, ppy) in a slab mask.
// bit = lx*8 + ly; the patch's bits 16*ppx + 2*ppy + {0, 1, 8, 9} all lie in one 32-bit word.
struct PatchBits {
    unsigned w0;       // bit position of element (0,0) inside its word
    unsigned bm0, bm1; // masks of the bits below elements (0,0) and (1,0) inside the word
    bool hiword;
    __device__ __forceinline__ void init(int ppx, int ppy) {
        w0 = 16u * (ppx & 1) + 2u * ppy;
        bm0 = (1u << w0) - 1u;
        bm1 = (1u << (w0 + 8u)) - 1u;
        hiword = (ppx >> 1) != 0;
    }
    // rank[e], e = a*2+b; returns the 4 activity bits (bit e)
    __device__ __forceinline__ unsigned ranks(unsigned lo, unsigned hi, unsigned rank[4]) const {
        const unsigned word = hiword ? hi : lo;
        const unsigned bc = hiword ? (unsigned)__popc(lo) : 0u;
        const unsigned nib = word >> w0;
        rank[0] = bc + (unsigned)__popc(word & bm0);
        rank[1] = rank[0] + (nib & 1u);
        rank[2] = bc + (unsigned)__popc(word & bm1);
        rank[3] = rank[2] + ((nib >> 8) & 1u);
        return (nib & 3u) | ((nib >> 6) & 12u);
    }
};

struct Entry {          // slab entry in registers: 64-bit mask + 32-bit storage position of the first lane
    unsigned lo, hi, base;
};

template <typename T> struct KW;   // stencil weights of the right type straight from the parameter block
template <> struct KW<double> {
    static __device__ __forceinline__ double w(const StageParams& p, int s) { return p.kw[s]; }
};
template <> struct KW<float> {
    static __device__ __forceinline__ float w(const StageParams& p, int s) { return p.kwf[s]; }
};

template <typename T, int R, int MODE>
__global__ void __launch_bounds__(STAGE_THREADS, (R == 1 ? 4 : 3)) stage_kernel(const __grid_constant__ StageParams p) {
    using C = typename CxOf<T>::type;
    using G = Geo<R>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr unsigned ES = sizeof(C);
    constexpr bool HAS_AUX = (MODE == MODE_S2 || MODE == MODE_S3 || MODE == MODE_S4);

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int half = lane >> 4, t = lane & 15;
    const int px = t >> 2, py = t & 3;
    const int sidx = (blockIdx.x * STAGE_WARPS + warp) * 2 + half;   // this half-warp's stream
    const bool valid = sidx < p.n_work;
    const WorkRec* __restrict__ w = p.work + (valid ? sidx : 0);

    // ---- per-stream constants -------------------------------------------------------------------
    const int z0 = w->z0, nz = valid ? w->nz : 0;
    const int z1 = z0 + nz;
    const int hq = 1 + (t >> 2), hj = t & 3;              // halo duty: neighbour tile hq, patch hj of its edge
    const Slab* __restrict__ slab0 = p.slabs + w->eoff[0];   // + plane index = own tile's entry
    const Slab* __restrict__ slabh = p.slabs + w->eoff[hq];
    const int zlo0 = w->zlo[0], zhi0 = w->zhi[0], zloh = w->zlo[hq], zhih = w->zhi[hq];
    int pxh, pyh, hb;                                     // neighbour patch and its slot base (elements)
    if (hq == 1) { pxh = 3; pyh = hj; hb = (6 - 8 + R) * G::PY + hj; }
    else if (hq == 2) { pxh = 0; pyh = hj; hb = (8 + R) * G::PY + hj; }
    else if (hq == 3) { pxh = hj; pyh = 3; hb = (2 * hj + R) * G::PY + 3 - 4; }
    else { pxh = hj; pyh = 0; hb = (2 * hj + R) * G::PY + 4; }
    // which of the neighbour patch's elements lie within R of this tile (all four for R = 2)
    const unsigned hen = (R == 2) ? 15u : (hq == 1 ? 12u : hq == 2 ? 3u : hq == 3 ? 10u : 5u);
    PatchBits pbo, pbh;
    pbo.init(px, py);
    pbh.init(pxh, pyh);
    const int ob = (2 * px + R) * G::PY + py;             // own patch base in a slot (elements)
    const unsigned ring = (unsigned)__cvta_generic_to_shared(smem_raw) +
                          (unsigned)((warp * 2 + half) * NSLOT * G::PLANE) * ES;
    const unsigned ring_own = ring + (unsigned)ob * ES, ring_halo = ring + (unsigned)hb * ES;
    constexpr int CB0 = G::cpos(0), CB1 = G::cpos(1);
    constexpr unsigned SLOT_BYTES = (unsigned)G::PLANE * ES;

    const C* __restrict__ in = reinterpret_cast<const C*>(p.in);

    // potential: u = qxy[e] + qz(plane); qxy = 1/2 (ax x^2 + ay y^2) of the patch points
    double qxy[4];
    {
        double qx[2], qy[2];
#pragma unroll
        for (int a = 0; a < 2; ++a) {
            const double x = ((double)(w->ix0 + 2 * px + a) - p.xc) * p.pot.h + p.pot.cx;
            const double y = ((double)(w->iy0 + 2 * py + a) - p.yc) * p.pot.h + p.pot.cy;
            qx[a] = p.hax * (x * x);
            qy[a] = p.hay * (y * y);
        }
#pragma unroll
        for (int e = 0; e < 4; ++e) qxy[e] = qx[e >> 1] + qy[e & 1];
    }
    double sc = 1.0, gsc = p.g;
    if (MODE == MODE_IMAG) { sc = *p.scale_in; gsc = p.g * (sc * sc); }

    // slab entry of plane zp; zero mask outside the tile's z-range
    auto load_entry = [&](const Slab* __restrict__ tab, int zlo, int zhi, int zp) {
        Entry en;
        en.lo = 0u; en.hi = 0u; en.base = 0u;
        if (zp >= zlo && zp < zhi) {
            const uint4 s = __ldg(reinterpret_cast<const uint4*>(tab + zp));
            en.lo = s.x; en.hi = s.y; en.base = s.z;
        }
        return en;
    };
    // cp.async the enabled points of one patch of one slab into a slot, zero-filling absent points
    auto fetch_patch = [&](const PatchBits& pb, const Entry& en, unsigned dst, unsigned enable) {
        unsigned rk[4];
        const unsigned act = pb.ranks(en.lo, en.hi, rk);
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            if ((enable >> e) & 1u) {
                const bool on = (act >> e) & 1u;
                cp_async_zfill(dst + (unsigned)(((e >> 1) * G::PY + ((e & 1) ? CB1 : CB0)) * (int)ES),
                               in + (on ? en.base + rk[e] : 0u), on);
            }
        }
    };

    const int kstart = z0 - R, kend = nz > 0 ? z1 + R : kstart;   // planes this stream touches
    int niter = nz > 0 ? nz + 2 * R : 0;
    niter = max(niter, __shfl_xor_sync(0xffffffffu, niter, 16));   // both halves run the same loop

    // state (accumulate-forward form): set s holds psi and the partial T psi of one earlier plane
    C SP[R][4], SA[R][4];
#pragma unroll
    for (int s = 0; s < R; ++s)
#pragma unroll
        for (int e = 0; e < 4; ++e) { SP[s][e] = mk<T>((T)0, (T)0); SA[s][e] = mk<T>((T)0, (T)0); }
    double acc[NACC] = {0.0, 0.0, 0.0, 0.0};

    // ---- prologue: planes kstart .. kstart+PF-1 in flight, entries of plane kstart+PF in registers --
    Entry pe0, peh;          // producer: entries of the next plane to fetch
#pragma unroll
    for (int i = 0; i < PF; ++i) {
        const int kp = kstart + i;
        pe0 = load_entry(slab0, zlo0, zhi0, kp);
        fetch_patch(pbo, pe0, ring_own + i * SLOT_BYTES, kp < kend ? 15u : 0u);
        peh = load_entry(slabh, zloh, zhih, kp);
        fetch_patch(pbh, peh, ring_halo + i * SLOT_BYTES, (kp >= z0 && kp < z1) ? hen : 0u);
        cp_async_commit();
    }
    pe0 = load_entry(slab0, zlo0, zhi0, kstart + PF);
    peh = load_entry(slabh, zloh, zhih, kstart + PF);
    Entry ce = load_entry(slab0, zlo0, zhi0, kstart - R);   // consumer: entry of the plane finished next (c = k-R)

    // one plane step.  (PN, AN) = set of plane k-1, (PO, AO) = set of plane k-R (the same set for R = 1).
    auto step = [&](C (&PN)[4], C (&AN)[4], C (&PO)[4], C (&AO)[4], const int k, const unsigned sl) {
        cp_async_wait<PF - 1>();
        __syncwarp();
        // ---- producer: plane k+PF -> slot (sl+PF) % NSLOT; entries of plane k+PF+1 -> registers ------
        {
            const int kp = k + PF;
            unsigned sp = sl + PF;
            if (sp >= NSLOT) sp -= NSLOT;
            fetch_patch(pbo, pe0, ring_own + sp * SLOT_BYTES, kp < kend ? 15u : 0u);
            fetch_patch(pbh, peh, ring_halo + sp * SLOT_BYTES, (kp >= z0 && kp < z1) ? hen : 0u);
            cp_async_commit();
            pe0 = load_entry(slab0, zlo0, zhi0, kp + 1);
            peh = load_entry(slabh, zloh, zhih, kp + 1);
        }
        if (k >= kend) return;
        const unsigned so = ring_own + sl * SLOT_BYTES;   // own patch in the slot of plane k
        const int c = k - R;
        const bool fin = c >= z0;
        // ---- output plane c: positions; aux loads issued early; next plane's entry and aux prefetched -----
        unsigned rk[4];
        unsigned cact = pbo.ranks(ce.lo, ce.hi, rk);
        if (!fin) cact = 0u;
        const unsigned cbase = ce.base;
        ce = load_entry(slab0, zlo0, zhi0, c + 1);
        C av[4];
        if (HAS_AUX) {
            const C* __restrict__ aux = reinterpret_cast<const C*>(p.aux);
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                av[e] = mk<T>((T)0, (T)0);
                if ((cact >> e) & 1u) av[e] = aux[cbase + rk[e]];
            }
        }
        // ---- psi(k) of the patch ------------------------------------------------------------------------
        C v[4];
#pragma unroll
        for (int e = 0; e < 4; ++e)
            v[e] = lds_c(so + (unsigned)(((e >> 1) * G::PY + ((e & 1) ? CB1 : CB0)) * (int)ES), (C*)nullptr);
        // ---- psi(k) completes the z part of planes k-1 .. k-R -------------------------------------------
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            AO[e].x = fma(KW<T>::w(p, R), v[e].x, AO[e].x);
            AO[e].y = fma(KW<T>::w(p, R), v[e].y, AO[e].y);
            if (R == 2) {
                AN[e].x = fma(KW<T>::w(p, 1), v[e].x, AN[e].x);
                AN[e].y = fma(KW<T>::w(p, 1), v[e].y, AN[e].y);
            }
        }
        // ---- finish plane c: V(r,t), nonlinear term, stage combination ------------------------------------
        if (cact) {
            const double zc = ((double)c - p.zc) * p.pot.h + p.pot.cz;
            const double qz = p.haz * (zc * zc) - p.delta_eff;
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const bool on = (cact >> e) & 1u;
                const C cv = PO[e];
                const C tc = AO[e];
                double vpot = qxy[e] + qz;
                if (p.pot.kind == GPE_POT_DRESSED) vpot = fast_sqrt(fma(vpot, vpot, p.om2)) - p.pot.omega;
                const T a2 = fma(cv.x, cv.x, cv.y * cv.y);
                const unsigned pos = cbase + rk[e];
                if (MODE == MODE_ENERGY) {
                    if (on) {
                        acc[0] += (double)(cv.x * tc.x + cv.y * tc.y);
                        acc[1] += vpot * (double)a2;
                        acc[2] += (double)a2 * (double)a2;
                        acc[3] += (double)a2;
                    }
                    continue;
                }
                const T diag = (T)fma(gsc, (double)a2, vpot);
                const C hc = mk<T>(fma(diag, cv.x, tc.x), fma(diag, cv.y, tc.y));
                const T ca = (T)p.ca;
                C o;
                if (MODE == MODE_APPLY) {
                    o = hc;
                } else if (MODE == MODE_IMAG) {
                    const T s = (T)sc;
                    o = mk<T>(s * fma(-ca, hc.x, cv.x), s * fma(-ca, hc.y, cv.y));
                    if (on) acc[0] += (double)o.x * (double)o.x + (double)o.y * (double)o.y;
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
                        const T third = (T)(1.0 / 3.0), tt = (T)(2.0 / 3.0);
                        if (on)
                            reinterpret_cast<C*>(p.out2)[pos] =
                                mk<T>(fma(tt, o.x, third * (cv.x - av[e].x)), fma(tt, o.y, third * (cv.y - av[e].y)));
                    }
                }
                if (on) reinterpret_cast<C*>(p.out1)[pos] = o;
            }
        }
        // ---- the oldest set becomes the set of plane k: z-backward part, centre, in-plane part -----------------
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            C an;
            if (R == 2) {
                an.x = KW<T>::w(p, 2) * PO[e].x;
                an.y = KW<T>::w(p, 2) * PO[e].y;
                an.x = fma(KW<T>::w(p, 1), PN[e].x, an.x);
                an.y = fma(KW<T>::w(p, 1), PN[e].y, an.y);
            } else {
                an.x = KW<T>::w(p, 1) * PO[e].x;
                an.y = KW<T>::w(p, 1) * PO[e].y;
            }
            AO[e].x = fma(KW<T>::w(p, 0), v[e].x, an.x);
            AO[e].y = fma(KW<T>::w(p, 0), v[e].y, an.y);
            PO[e] = v[e];
        }
        if (k >= z0 && k < z1) {
            // x direction: source rows r = -R .. 1+R of column b; rows 0, 1 are the patch itself
#pragma unroll
            for (int b = 0; b < 2; ++b) {
#pragma unroll
                for (int r = -R; r <= 1 + R; ++r) {
                    const C val = (r == 0 || r == 1)
                                      ? v[r * 2 + b]
                                      : lds_c(so + (unsigned)((r * G::PY + (b ? CB1 : CB0)) * (int)ES), (C*)nullptr);
#pragma unroll
                    for (int a = 0; a < 2; ++a) {
                        const int d = r > a ? r - a : a - r;
                        if (d >= 1 && d <= R) {
                            AO[a * 2 + b].x = fma(KW<T>::w(p, d), val.x, AO[a * 2 + b].x);
                            AO[a * 2 + b].y = fma(KW<T>::w(p, d), val.y, AO[a * 2 + b].y);
                        }
                    }
                }
            }
            // y direction: source columns cc = -R .. 1+R of row a
#pragma unroll
            for (int a = 0; a < 2; ++a) {
#pragma unroll
                for (int cc = -R; cc <= 1 + R; ++cc) {
                    const C val = (cc == 0 || cc == 1)
                                      ? v[a * 2 + cc]
                                      : lds_c(so + (unsigned)((a * G::PY + G::cpos(cc)) * (int)ES), (C*)nullptr);
#pragma unroll
                    for (int b = 0; b < 2; ++b) {
                        const int d = cc > b ? cc - b : b - cc;
                        if (d >= 1 && d <= R) {
                            AO[a * 2 + b].x = fma(KW<T>::w(p, d), val.x, AO[a * 2 + b].x);
                            AO[a * 2 + b].y = fma(KW<T>::w(p, d), val.y, AO[a * 2 + b].y);
                        }
                    }
                }
            }
        }
    };

    unsigned sl = 0;                                       // ring slot of plane k
    for (int it = 0; it < niter; it += R) {
        const int k = kstart + it;
        if (R == 1) {
            step(SP[0], SA[0], SP[0], SA[0], k, sl);
            sl = (sl + 1 == NSLOT) ? 0 : sl + 1;
        } else {
            step(SP[0], SA[0], SP[R - 1], SA[R - 1], k, sl);
            sl = (sl + 1 == NSLOT) ? 0 : sl + 1;
            if (it + 1 < niter) {
                step(SP[R - 1], SA[R - 1], SP[0], SA[0], k + 1, sl);
                sl = (sl + 1 == NSLOT) ? 0 : sl + 1;
            }
        }
    }
    cp_async_wait<0>();

    // ---- per-stream partial sums in a fixed order (bit-reproducible, independent of scheduling) -------
    if (MODE == MODE_IMAG || MODE == MODE_ENERGY) {
#pragma unroll
        for (int kq = 0; kq < NACC; ++kq)
#pragma unroll
            for (int off = 8; off > 0; off >>= 1) acc[kq] += __shfl_down_sync(0xffffffffu, acc[kq], off, 16);
        if (t == 0 && valid) {
#pragma unroll
            for (int kq = 0; kq < NACC; ++kq) p.partials[(size_t)sidx * NACC + kq] = acc[kq];
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

template <typename T, int R> constexpr size_t stage_smem() {
    return (size_t)STREAMS_PER_BLOCK * NSLOT * Geo<R>::PLANE * sizeof(typename CxOf<T>::type);
}

template <typename T, int R, int MODE>
cudaError_t launch_one(const StageParams& p, cudaStream_t st) {
    const size_t smem = stage_smem<T, R>();
    const int nblk = (p.n_work + STREAMS_PER_BLOCK - 1) / STREAMS_PER_BLOCK;
    stage_kernel<T, R, MODE><<<nblk, STAGE_THREADS, smem, st>>>(p);
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
    return cudaFuncSetAttribute(stage_kernel<T, R, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)stage_smem<T, R>());
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

size_t stage_smem_bytes(int dtype, int radius) {
    if (dtype == GPE_C128) return radius == 1 ? stage_smem<double, 1>() : stage_smem<double, 2>();
    return radius == 1 ? stage_smem<float, 1>() : stage_smem<float, 2>();
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
