// C-ABI glue of libgpe_b200.so (include/gpe.h): handles, argument checks, table upload, and the
// sequences of kernel launches behind each call.  Every step of the path runs in gpe_kernels.cu; there
// is no CPU fallback.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "gpe_internal.h"

using namespace gpe;

struct gpe_grid {
    GridHost h;
    // device tables (uploaded when the first sim is created on the grid)
    bool on_device = false;
    int device = -1;
    Slab* d_slabs = nullptr;
    int64_t* d_perm = nullptr;
    int n_sims = 0;
};

struct gpe_sim {
    gpe_grid* grid = nullptr;
    int dtype = GPE_C128;
    int radius = 1;
    bool hoc = false;       // 19-point higher-order compact stencil (radius 1 plus edge neighbours)
    bool custom27 = false;  // weights of the 3x3x3 stencil supplied by the caller (gpe_sim_set_compact_weights)
    double w27[8] = {0, 0, 0, 0, 0, 0, 0, 0};   // centre, face x y z, edge xy xz yz, corner (absolute, 1/length^2)
    double g = 0.0, n_target = 1.0;
    double t = 0.0;
    int kz = 32;
    size_t csize = 16;      // bytes per complex value
    int64_t n = 0;          // n_active
    void* buf[4] = {nullptr, nullptr, nullptr, nullptr};  // A (psi), B, C, D in storage order
    void* staging = nullptr;                               // canonical staging (host copies, apply_H)
    void* extra[2] = {nullptr, nullptr};                   // library-owned: two more stage states for RKCK (lazy)
    // library-owned scratch
    WorkRec* d_work = nullptr;
    int32_t n_blocks = 0;
    double* d_partials = nullptr;
    int64_t* d_map = nullptr;   // re-gridding table of gpe_remap_psi into this sim (allocated on first use)
    double* h_flag = nullptr;   // pinned copy of the degenerate-norm flag, filled asynchronously at the end of a run
    cudaEvent_t ev_flag = nullptr;
    bool flag_pending = false;
    void* flag_stream = nullptr;   // stream of the run whose flush recorded ev_flag (the device-side reset goes there)
    // CUDA graph of RK4_GRAPH_STEPS steps for runs on small grids in a potential that does not change during the run
    cudaStream_t cap_stream = nullptr;
    cudaGraphExec_t rk4_exec = nullptr;
    bool graph_off = false;     // capture failed once
    // gpe_sim_set_option
    int opt_k1 = 1;             // GPE_OPT_FUSED_K1
    int opt_graph = 1;          // GPE_OPT_RK4_GRAPH
    int opt_pdl = 1;            // GPE_OPT_PDL
    struct GraphKey {
        double dt = 0.0, delta = 0.0, g = 0.0, w27[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        void* buf[4] = {nullptr, nullptr, nullptr, nullptr};
        const void* work = nullptr;
        int32_t n_blocks = 0;
        bool custom27 = false;
        bool operator==(const GraphKey& o) const {
            return dt == o.dt && delta == o.delta && g == o.g && std::memcmp(w27, o.w27, sizeof(w27)) == 0 &&
                   std::memcmp(buf, o.buf, sizeof(buf)) == 0 && work == o.work && n_blocks == o.n_blocks && custom27 == o.custom27;
        }
    } rk4_key;
    double* d_sums = nullptr;   // [NACC] + scale at [NACC] + degenerate-norm flag at [NACC + 1]
    int64_t launches = 0;
    bool counted = false;   // registered in grid->n_sims
    // stage timing
    bool timing = false;
    std::vector<cudaEvent_t> ev[4];  // pairs (start, stop) per stage
    size_t ev_used[4] = {0, 0, 0, 0};
};

namespace {

thread_local std::string g_err;

int fail(int code, const std::string& msg) {
    g_err = msg;
    return code;
}
int cuda_fail(cudaError_t e, const char* what) {
    g_err = std::string(what) + ": " + cudaGetErrorString(e);
    return GPE_ERR_CUDA;
}
#define CU(call)                                           \
    do {                                                   \
        cudaError_t e__ = (call);                          \
        if (e__ != cudaSuccess) return cuda_fail(e__, #call); \
    } while (0)
#define KL(call)                                                       \
    do {                                                               \
        int e__ = (call);                                              \
        if (e__ != 0) return cuda_fail((cudaError_t)e__, #call);       \
    } while (0)

double cell_volume(const gpe_box& b) { return b.h * (b.hy > 0.0 ? b.hy : b.h) * (b.hz > 0.0 ? b.hz : b.h); }

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// GPE_R64: 8-byte elements.  Copies move them with the 8-byte (complex64) kernels; sums of squares and the scaling
// treat the array as ceil(n/2) complex128 values (buffers are zero-filled and 256-byte padded, the odd tail is 0).
int copy_dtype(int dtype) { return dtype == GPE_R64 ? GPE_C64 : dtype; }
int pair_dtype(int dtype) { return dtype == GPE_R64 ? GPE_C128 : dtype; }
int64_t pair_count(int dtype, int64_t n) { return dtype == GPE_R64 ? (n + 1) / 2 : n; }

size_t buf_bytes(int64_t n, int dtype) { return align_up((size_t)(n > 0 ? n : 1) * (dtype == GPE_C128 ? 16 : 8), 256); }

PotDev pot_dev(const gpe_sim* s, double t) {
    const GridHost& h = s->grid->h;
    PotDev p;
    p.kind = h.pot.kind;
    p.nx = h.box.nx; p.ny = h.box.ny; p.nz = h.box.nz;
    p.h = h.box.h; p.hy = h.box.hy > 0.0 ? h.box.hy : h.box.h; p.hz = h.box.hz > 0.0 ? h.box.hz : h.box.h;
    p.cx = h.box.center[0]; p.cy = h.box.center[1]; p.cz = h.box.center[2];
    p.ax = h.pot.ax; p.ay = h.pot.ay; p.az = h.pot.az;
    p.delta = delta_of_t(h.pot, t);
    p.omega = h.pot.omega;
    return p;
}

// Split the grid's work items into pieces of at most kz planes and upload them.
int build_work(gpe_sim* s) {
    const GridHost& h = s->grid->h;
    std::vector<WorkRec> recs;
    const int kz = s->kz;
    for (int64_t wi = 0; wi < h.n_work(); ++wi) {
        const int32_t k = h.wi_tile[wi];
        const int z0 = h.wi_z0[wi], nz = h.wi_nz[wi];
        const int kk = (nz + kz - 1) / kz;
        for (int i = 0; i < kk; ++i) {
            const int s0 = z0 + (int)(((int64_t)i * nz) / kk), s1 = z0 + (int)(((int64_t)(i + 1) * nz) / kk);
            WorkRec r;
            std::memset(&r, 0, sizeof(r));
            r.ix0 = h.tile_xy[2 * k] * h.tx;
            r.iy0 = h.tile_xy[2 * k + 1] * h.ty;
            r.z0 = s0;
            r.nz = s1 - s0;
            r.eoff[0] = h.tile_entry_base[k] - h.tile_zlo[k];
            r.zlo[0] = h.tile_zlo[k];
            r.zhi[0] = h.tile_zhi[k];
            for (int q = 1; q < NTILE; ++q) {
                int32_t nb = -1;
                if (q <= 4) {
                    nb = h.tile_nbr[4 * k + q - 1];
                } else {
                    // diagonal tile (i +- 1, j +- 1): the tile list ascends in (i, j), binary search
                    const int32_t ti = h.tile_xy[2 * k] + (q <= 6 ? -1 : 1), tj = h.tile_xy[2 * k + 1] + ((q & 1) ? -1 : 1);
                    int64_t lo = 0, hi = h.n_tiles();
                    while (lo < hi) {
                        const int64_t mid = (lo + hi) / 2;
                        const int32_t mi = h.tile_xy[2 * mid], mj = h.tile_xy[2 * mid + 1];
                        if (mi < ti || (mi == ti && mj < tj)) lo = mid + 1; else hi = mid;
                    }
                    if (lo < h.n_tiles() && h.tile_xy[2 * lo] == ti && h.tile_xy[2 * lo + 1] == tj) nb = (int32_t)lo;
                }
                if (nb >= 0) {
                    r.eoff[q] = h.tile_entry_base[nb] - h.tile_zlo[nb];
                    r.zlo[q] = h.tile_zlo[nb];
                    r.zhi[q] = h.tile_zhi[nb];
                }
            }
            const int64_t e0 = r.eoff[0] + s0, e1 = r.eoff[0] + s1 - 1;
            r.pos0 = h.slab_base[e0];
            r.npts = (int32_t)(h.slab_base[e1] + __builtin_popcountll(h.slab_mask[e1]) - r.pos0);
            // the R planes below the piece matter through the z direction of the own columns only (star stencils):
            // a piece that starts a run has nothing there and skips them; the 19-/27-point stencils also see the
            // neighbour tiles' points in those planes (xz / yz edges) and always read them
            r.lead = s->radius;
            if (!s->hoc) {
                bool any = false;
                for (int z = std::max(s0 - s->radius, (int)h.tile_zlo[k]); z < s0; ++z) any = any || h.slab_mask[r.eoff[0] + z] != 0;
                if (!any) r.lead = 0;
            }
            recs.push_back(r);
        }
    }
    if (recs.size() > (size_t)0x7fffffff) return fail(GPE_ERR_UNSUPPORTED, "too many work pieces");
    if (s->rk4_exec) { cudaGraphExecDestroy(s->rk4_exec); s->rk4_exec = nullptr; }   // captured with the old work records
    if (s->d_work) { cudaFree(s->d_work); s->d_work = nullptr; }
    if (s->d_partials) { cudaFree(s->d_partials); s->d_partials = nullptr; }
    s->n_blocks = (int32_t)recs.size();
    const size_t nrec = recs.empty() ? 1 : recs.size();
    cudaError_t e = cudaMalloc(&s->d_work, nrec * sizeof(WorkRec));
    if (e == cudaErrorMemoryAllocation) return fail(GPE_ERR_OUT_OF_MEMORY, "cudaMalloc(work records)");
    CU(e);
    if (!recs.empty()) CU(cudaMemcpy(s->d_work, recs.data(), recs.size() * sizeof(WorkRec), cudaMemcpyHostToDevice));
    size_t np = std::max<size_t>(nrec, (size_t)norm_blocks(s->n));
    e = cudaMalloc(&s->d_partials, np * NACC * sizeof(double));
    if (e == cudaErrorMemoryAllocation) return fail(GPE_ERR_OUT_OF_MEMORY, "cudaMalloc(partials)");
    CU(e);
    return GPE_OK;
}

int upload_grid(gpe_grid* g) {
    if (g->on_device) return GPE_OK;
    int dev = 0;
    CU(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    CU(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10) return fail(GPE_ERR_CUDA, "device is not sm_100 (B200): kernels are built for sm_100a only");
    KL(kernels_configure());
    const GridHost& h = g->h;
    const size_t ns = (size_t)std::max<int64_t>(h.n_slabs(), 1), na = (size_t)std::max<int64_t>(h.n_active, 1);
    cudaError_t e = cudaMalloc(&g->d_slabs, ns * sizeof(Slab));
    if (e == cudaErrorMemoryAllocation) return fail(GPE_ERR_OUT_OF_MEMORY, "cudaMalloc(slabs)");
    CU(e);
    e = cudaMalloc(&g->d_perm, na * sizeof(int64_t));
    if (e == cudaErrorMemoryAllocation) { cudaFree(g->d_slabs); g->d_slabs = nullptr; return fail(GPE_ERR_OUT_OF_MEMORY, "cudaMalloc(perm)"); }
    if (e != cudaSuccess) { cudaFree(g->d_slabs); g->d_slabs = nullptr; return cuda_fail(e, "cudaMalloc(perm)"); }
    std::vector<Slab> slabs((size_t)h.n_slabs());
    for (int64_t k = 0; k < h.n_slabs(); ++k) { slabs[k].mask = h.slab_mask[k]; slabs[k].base = h.slab_base[k]; }
    e = cudaSuccess;
    if (!slabs.empty()) e = cudaMemcpy(g->d_slabs, slabs.data(), slabs.size() * sizeof(Slab), cudaMemcpyHostToDevice);
    if (e == cudaSuccess && h.n_active > 0)
        e = cudaMemcpy(g->d_perm, h.storage_to_canonical.data(), (size_t)h.n_active * sizeof(int64_t), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {   // nothing is left allocated on a failed upload (a retry allocates again)
        cudaFree(g->d_slabs); g->d_slabs = nullptr;
        cudaFree(g->d_perm); g->d_perm = nullptr;
        return cuda_fail(e, "cudaMemcpy(layout tables)");
    }
    g->device = dev;
    g->on_device = true;
    return GPE_OK;
}

StageParams base_params(const gpe_sim* s, double t) {
    StageParams p;
    std::memset(&p, 0, sizeof(p));
    p.slabs = s->grid->d_slabs;
    p.work = s->d_work;
    p.n_work = s->n_blocks;
    p.kz = s->kz;
    p.pot = pot_dev(s, t);
    p.g = s->g;
    p.partials = s->d_partials;
    p.scale_in = s->d_sums + NACC;
    const GridHost& h = s->grid->h;
    // Eq. B1: each axis with its own 1/d_a^2; star weights c_0, c_1, c_2 (R5); all times -1/2
    const double c0 = s->radius == 1 ? -2.0 : -2.5, c1 = s->radius == 1 ? 1.0 : 4.0 / 3.0, c2 = s->radius == 1 ? 0.0 : -1.0 / 12.0;
    const double ia[3] = {1.0 / (p.pot.h * p.pot.h), 1.0 / (p.pot.hy * p.pot.hy), 1.0 / (p.pot.hz * p.pot.hz)};
    for (int a = 0; a < 3; ++a) { p.kw[a][0] = 0.0; p.kw[a][1] = -0.5 * c1 * ia[a]; p.kw[a][2] = -0.5 * c2 * ia[a]; }
    p.kw[0][0] = -0.5 * c0 * (ia[0] + ia[1] + ia[2]);
    p.ke[0] = p.ke[1] = p.ke[2] = 0.0;
    if (s->hoc) {
        // Eq. B2: lap_19 = lap_7 + sum_pairs (d_i^2 + d_j^2)/12 d_ii d_jj; (d_i^2 + d_j^2)/(d_i^2 d_j^2) = 1/d_i^2 + 1/d_j^2,
        // so the pair weight is c_ij = (1/d_i^2 + 1/d_j^2)/12: edges c_ij, faces 1/d_i^2 - 2 (c_ij + c_ik),
        // centre -2 sum 1/d_i^2 + 4 sum c_ij  (isotropic: -4, 1/3, 1/6 over h^2)
        const double cxy = (ia[0] + ia[1]) / 12.0, cxz = (ia[0] + ia[2]) / 12.0, cyz = (ia[1] + ia[2]) / 12.0;
        p.kw[0][0] = -0.5 * (-2.0 * (ia[0] + ia[1] + ia[2]) + 4.0 * (cxy + cxz + cyz));
        p.kw[0][1] = -0.5 * (ia[0] - 2.0 * (cxy + cxz));
        p.kw[1][1] = -0.5 * (ia[1] - 2.0 * (cxy + cyz));
        p.kw[2][1] = -0.5 * (ia[2] - 2.0 * (cxz + cyz));
        p.ke[0] = -0.5 * cxy; p.ke[1] = -0.5 * cxz; p.ke[2] = -0.5 * cyz;
    }
    p.kcn = 0.0;
    if (s->hoc && s->custom27) {   // T = -1/2 lap with the caller's Laplacian weights
        p.kw[0][0] = -0.5 * s->w27[0];
        for (int a = 0; a < 3; ++a) { p.kw[a][1] = -0.5 * s->w27[1 + a]; p.ke[a] = -0.5 * s->w27[4 + a]; }
        p.kcn = -0.5 * s->w27[7];
    }
    p.kcnf = (float)p.kcn;
    for (int a = 0; a < 3; ++a) {
        for (int k = 0; k < 3; ++k) p.kwf[a][k] = (float)p.kw[a][k];
        p.kef[a] = (float)p.ke[a];
    }
    p.xc = 0.5 * (double)(h.box.nx - 1);
    p.yc = 0.5 * (double)(h.box.ny - 1);
    p.zc = 0.5 * (double)(h.box.nz - 1);
    p.hax = 0.5 * h.pot.ax; p.hay = 0.5 * h.pot.ay; p.haz = 0.5 * h.pot.az;
    p.om2 = h.pot.omega * h.pot.omega;
    p.delta_eff = h.pot.kind == GPE_POT_DRESSED ? p.pot.delta : 0.0;
    p.comb[0] = -1.0 / 3.0; p.comb[1] = 1.0 / 3.0; p.comb[2] = 2.0 / 3.0;   // RK4 b* (Eq. A11)
    return p;
}

int stage(gpe_sim* s, int mode, double t, double ca, const void* in, const void* aux, void* out1, void* out2,
          void* stream, int timed_slot = -1, const double* comb = nullptr) {
    StageParams p = base_params(s, t);
    if (comb) { p.comb[0] = comb[0]; p.comb[1] = comb[1]; p.comb[2] = comb[2]; }
    p.ca = ca; p.in = in; p.aux = aux; p.out1 = out1; p.out2 = out2;
    cudaStream_t st = (cudaStream_t)stream;
    if (s->timing && timed_slot >= 0) {
        auto& v = s->ev[timed_slot];
        size_t& u = s->ev_used[timed_slot];
        while (v.size() < u + 2) {
            cudaEvent_t e;
            CU(cudaEventCreate(&e));
            v.push_back(e);
        }
        CU(cudaEventRecord(v[u], st));
        KL(launch_stage(s->dtype, s->hoc ? 3 : s->radius, mode, p, stream, s->opt_pdl));
        CU(cudaEventRecord(v[u + 1], st));
        u += 2;
    } else {
        KL(launch_stage(s->dtype, s->hoc ? 3 : s->radius, mode, p, stream, s->opt_pdl));
    }
    if (s->n_blocks > 0) s->launches += 1;
    return GPE_OK;
}

int rk4_step(gpe_sim* s, double t, double dt, void* stream) {
    void *A = s->buf[0], *B = s->buf[1], *C = s->buf[2], *D = s->buf[3];
    int rc;
    // PAPER.md:276-281 Eq. A6-A7 with a*, b* of Eq. A10-A11 (RK4); b* = [-1/3, 1/3, 2/3, 1/3]
    if ((rc = stage(s, MODE_S1, t, 0.5 * dt, A, nullptr, B, nullptr, stream, 0))) return rc;            // y2
    if ((rc = stage(s, MODE_S2, t + 0.5 * dt, 0.5 * dt, B, A, C, D, stream, 1))) return rc;             // y3, p
    if ((rc = stage(s, MODE_S3, t + 0.5 * dt, dt, C, A, B, nullptr, stream, 2))) return rc;             // y4
    if ((rc = stage(s, MODE_S4, t + dt, dt / 6.0, B, D, A, nullptr, stream, 3))) return rc;             // y_new
    return GPE_OK;
}

int rkhe3_step(gpe_sim* s, double t, double dt, void* stream) {
    void *A = s->buf[0], *B = s->buf[1], *C = s->buf[2], *D = s->buf[3];
    int rc;
    // Heun's third-order method, PAPER.md:276-281 Eq. A6-A7 with a* = [[1,0],[1,0]], b* = [1/4, 3/4, 0] (Eq. A8-A9)
    // and a21 = 1/3, a32 = 2/3, b3 = 3/4; the b* terms are pre-summed into p by the second stage
    const double comb[3] = {0.25, 0.75, 0.0};
    if ((rc = stage(s, MODE_S1, t, dt / 3.0, A, nullptr, B, nullptr, stream))) return rc;                           // y2
    if ((rc = stage(s, MODE_S2, t + dt / 3.0, 2.0 * dt / 3.0, B, A, C, D, stream, -1, comb))) return rc;            // y3, p
    if ((rc = stage(s, MODE_S3, t + 2.0 * dt / 3.0, 0.75 * dt, C, D, A, nullptr, stream))) return rc;               // y_new
    return GPE_OK;
}

// general stage of Eq. A6-A7: out = sum_j coef[j] aux[j] + coefc in + ca f(t, in)
int stage_lc(gpe_sim* s, double t, double ca, const void* in, int n_aux, const void* const* aux, const double* coef,
             double coefc, void* out, void* stream) {
    StageParams p = base_params(s, t);
    p.ca = ca; p.in = in; p.out1 = out;
    p.n_aux = n_aux;
    p.coefc = coefc;
    for (int j = 0; j < n_aux; ++j) { p.auxn[j] = aux[j]; p.coef[j] = coef[j]; }
    KL(launch_stage(s->dtype, s->hoc ? 3 : s->radius, MODE_LC, p, stream, s->opt_pdl));
    if (s->n_blocks > 0) s->launches += 1;
    return GPE_OK;
}

int rkck_step(gpe_sim* s, double t, double dt, void* stream) {
    // Cash-Karp in the stage-state form: a*, b* of PAPER.md:321-329 Eq. A12-A13 (two garbled entries of the
    // last row of a* corrected: 253/12288, 1375/1536; R17), a_{i+1,i} and c_i of the Cash-Karp tableau
    void* Y[6] = {s->buf[0], s->buf[1], s->buf[2], s->buf[3], s->extra[0], s->extra[1]};
    static const double c[6] = {0.0, 1.0 / 5.0, 3.0 / 10.0, 3.0 / 5.0, 1.0, 7.0 / 8.0};
    static const double sub[6] = {1.0 / 5.0, 9.0 / 40.0, 6.0 / 5.0, 35.0 / 27.0, 253.0 / 4096.0, 512.0 / 1771.0};
    static const double astar[5][5] = {
        {1.0, 0, 0, 0, 0},
        {5.0 / 8.0, 3.0 / 8.0, 0, 0, 0},
        {2.0, 3.0, -4.0, 0, 0},
        {-49.0 / 81.0, 35.0 / 27.0, 200.0 / 81.0, -175.0 / 81.0, 0},
        {253.0 / 12288.0, -3795.0 / 4096.0, 1375.0 / 1536.0, 2875.0 / 4096.0, 1265.0 / 4096.0}};
    static const double bstar[6] = {-991.0 / 15939.0, -3865.0 / 5313.0, 5000.0 / 5313.0, 3125.0 / 4554.0, 25.0 / 154.0, 0.0};
    int rc;
    for (int i = 0; i < 5; ++i) {   // y^(i+2) = sum_{j<=i} a*_{i,j} y^(j+1) + dt a_{i+2,i+1} f(t + c_{i+1} dt, y^(i+1))
        if ((rc = stage_lc(s, t + c[i] * dt, sub[i] * dt, Y[i], i, Y, astar[i], astar[i][i], Y[i + 1], stream))) return rc;
    }
    // y_new = sum_{j<=5} b*_j y^(j) + dt b_6 f(t + c_6 dt, y^(6)); written over y^(1) (read at the point itself only)
    return stage_lc(s, t + c[5] * dt, sub[5] * dt, Y[5], 5, Y, bstar, bstar[5], Y[0], stream);
}

// End of an imaginary-time run: apply the lazy scale, reset it, and fetch the degenerate-norm flag (the finalise
// kernel kept scale 1 and raised it: the state is left as it is) into pinned memory WITHOUT synchronising: a loop of
// single steps stays asynchronous.  check_flag() reports it at the next call that can know.
int flush_scale(gpe_sim* s, void* stream) {
    KL(launch_scale(pair_dtype(s->dtype), s->buf[0], pair_count(s->dtype, s->n), s->d_sums + NACC, stream));
    KL(launch_set_scalar(s->d_sums + NACC, 1.0, stream));
    s->launches += 2;
    CU(cudaMemcpyAsync(s->h_flag, s->d_sums + NACC + 1, sizeof(double), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    CU(cudaEventRecord(s->ev_flag, (cudaStream_t)stream));
    s->flag_pending = true;
    s->flag_stream = stream;
    return GPE_OK;
}

// The state the deferred degenerate-norm flag referred to has just been replaced (gpe_set_psi, gpe_set_psi_host,
// gpe_remap_psi into this sim) by work enqueued on `stream`: forget the flag, on the host and -- ordered after the
// run on the caller's stream, like the new state itself -- on the device.
int drop_flag(gpe_sim* s, void* stream) {
    if (!s->flag_pending) return GPE_OK;
    s->flag_pending = false;
    CU(cudaMemsetAsync(s->d_sums + NACC + 1, 0, sizeof(double), (cudaStream_t)stream));
    return GPE_OK;
}

// synced = the caller has just synchronised the stream the run was enqueued on
int check_flag(gpe_sim* s, bool synced, void* /*stream of the reporting call*/) {
    if (!s->flag_pending) return GPE_OK;
    if (!synced) {
        cudaError_t q = cudaEventQuery(s->ev_flag);
        if (q == cudaErrorNotReady) return GPE_OK;         // still running: a later call reports it
        CU(q);
    } else {
        CU(cudaEventSynchronize(s->ev_flag));
    }
    s->flag_pending = false;
    if (*s->h_flag != 0.0) {
        *s->h_flag = 0.0;
        CU(cudaMemsetAsync(s->d_sums + NACC + 1, 0, sizeof(double), (cudaStream_t)s->flag_stream));
        return fail(GPE_ERR_STATE, "the particle number became zero or non-finite during an imaginary-time run (no renormalisation was applied)");
    }
    return GPE_OK;
}

constexpr int RK4_GRAPH_STEPS = 8;
constexpr int64_t GRAPH_MAX_POINTS = 4000000;   // above this the stage kernels are long enough for the host to keep ahead

// RK4 steps [0, nfull * RK4_GRAPH_STEPS) of a run in a potential that is the same at every stage time of the run:
// the four launches of a step have the same parameters in every step, so RK4_GRAPH_STEPS steps are captured once
// into a CUDA graph (programmatic dependent launches included) and replayed; the host leaves the loop
// (PAPER.md:87 keeps the iteration on the device for the same reason).  Returns the number of steps done (0 = the
// caller runs everything step by step); results are bit-identical to the step-by-step path (same kernels, same
// parameters, same order).
int64_t rk4_graph_steps(gpe_sim* s, double t0, double dt, int64_t nsteps, void* stream) {
    if (!s->opt_graph || s->graph_off || s->timing || s->n_blocks <= 0 || s->n > GRAPH_MAX_POINTS || nsteps < 2 * RK4_GRAPH_STEPS) return 0;
    {
        // the caller's stream is itself being captured: this call must not open a capture of its own or instantiate a
        // graph in the middle of it; the step-by-step launches below go into the caller's capture like any other work
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing((cudaStream_t)stream, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) {
            cudaGetLastError();
            return 0;
        }
    }
    // The replayed launches carry the parameters of the capture, so everything a stage launch depends on must either be
    // in GraphKey or be constant for the sim's lifetime.  Today the ONLY time dependence of the path is Delta(t) of the
    // dressed potential (delta_of_t), and Delta(t) is monotone in t, so "equal at both ends of the run" means "constant
    // over the run".  Any new time-dependent term of V (or a non-monotone ramp) must join GraphKey and this test.
    const gpe_potential& pot = s->grid->h.pot;
    const double d0 = delta_of_t(pot, t0), d1 = delta_of_t(pot, t0 + (double)nsteps * dt);
    if (pot.kind == GPE_POT_DRESSED && d0 != d1) return 0;   // Delta(t) is monotone: equal ends = constant in between
    gpe_sim::GraphKey key;
    key.dt = dt; key.delta = pot.kind == GPE_POT_DRESSED ? d0 : 0.0; key.g = s->g;
    std::memcpy(key.w27, s->w27, sizeof(key.w27));
    for (int k = 0; k < 4; ++k) key.buf[k] = s->buf[k];
    key.work = s->d_work; key.n_blocks = s->n_blocks; key.custom27 = s->custom27;
    if (!s->rk4_exec || !(key == s->rk4_key)) {
        if (s->rk4_exec) { cudaGraphExecDestroy(s->rk4_exec); s->rk4_exec = nullptr; }
        if (!s->cap_stream && cudaStreamCreateWithFlags(&s->cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
            cudaGetLastError(); s->graph_off = true; return 0;
        }
        const int64_t launches0 = s->launches;
        cudaGraph_t graph = nullptr;
        bool ok = cudaStreamBeginCapture(s->cap_stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
        for (int k = 0; ok && k < RK4_GRAPH_STEPS; ++k) ok = rk4_step(s, t0, dt, s->cap_stream) == GPE_OK;
        cudaError_t ee = cudaStreamEndCapture(s->cap_stream, &graph);
        ok = ok && ee == cudaSuccess && graph != nullptr;
        if (ok) ok = cudaGraphInstantiate(&s->rk4_exec, graph, 0) == cudaSuccess;
        if (graph) cudaGraphDestroy(graph);
        s->launches = launches0;                            // nothing ran during the capture
        if (!ok) { cudaGetLastError(); s->rk4_exec = nullptr; s->graph_off = true; return 0; }
        s->rk4_key = key;
    }
    const int64_t nfull = nsteps / RK4_GRAPH_STEPS;
    for (int64_t k = 0; k < nfull; ++k) {
        if (cudaGraphLaunch(s->rk4_exec, (cudaStream_t)stream) != cudaSuccess) {
            cudaGetLastError();
            s->graph_off = true;
            s->launches += k * RK4_GRAPH_STEPS * 4;
            return k * RK4_GRAPH_STEPS;
        }
    }
    s->launches += nfull * RK4_GRAPH_STEPS * 4;
    return nfull * RK4_GRAPH_STEPS;
}

int sums_to_host(gpe_sim* s, double out[NACC], void* stream) {
    CU(cudaMemcpyAsync(out, s->d_sums, NACC * sizeof(double), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    CU(cudaStreamSynchronize((cudaStream_t)stream));
    return GPE_OK;
}

}  // namespace

namespace gpe {
int api_fail(int code, const char* msg) { return fail(code, msg); }
int api_cuda_fail(int cuda_error, const char* what) { return cuda_fail((cudaError_t)cuda_error, what); }
}  // namespace gpe

extern "C" {

const char* gpe_last_error(void) { return g_err.c_str(); }

int gpe_grid_create(const gpe_box* box, const gpe_potential* pot, double v_cut, int halo_width, gpe_grid** out) {
    if (!box || !pot || !out) return fail(GPE_ERR_INVALID_ARG, "null argument");
    gpe_grid* g = new (std::nothrow) gpe_grid();
    if (!g) return fail(GPE_ERR_OUT_OF_MEMORY, "host allocation");
    std::string err;
    int rc = build_layout_from_potential(*box, *pot, v_cut, halo_width, &g->h, &err);
    if (rc) { delete g; return fail(rc, err); }
    *out = g;
    return GPE_OK;
}

int gpe_grid_create_from_indices(const gpe_box* box, const gpe_potential* pot, const int64_t* active_host, int64_t n,
                                 int halo_width, gpe_grid** out) {
    if (!box || !pot || !out) return fail(GPE_ERR_INVALID_ARG, "null argument");
    gpe_grid* g = new (std::nothrow) gpe_grid();
    if (!g) return fail(GPE_ERR_OUT_OF_MEMORY, "host allocation");
    std::string err;
    int rc = build_layout_from_indices(*box, *pot, active_host, n, halo_width, &g->h, &err);
    if (rc) { delete g; return fail(rc, err); }
    *out = g;
    return GPE_OK;
}

int gpe_grid_destroy(gpe_grid* g) {
    if (!g) return GPE_OK;
    if (g->n_sims > 0) return fail(GPE_ERR_STATE, "destroy the sims created on this grid first");
    if (g->d_slabs) cudaFree(g->d_slabs);
    if (g->d_perm) cudaFree(g->d_perm);
    delete g;
    return GPE_OK;
}

int gpe_grid_num_active(const gpe_grid* g, int64_t* out) {
    if (!g || !out) return fail(GPE_ERR_INVALID_ARG, "null argument");
    *out = g->h.n_active;
    return GPE_OK;
}

int gpe_grid_num_stored(gpe_grid* g, int64_t* out) {
    if (!g || !out) return fail(GPE_ERR_INVALID_ARG, "null argument");
    try {
        build_stored_indices(&g->h);
    } catch (const std::bad_alloc&) {
        return fail(GPE_ERR_OUT_OF_MEMORY, "host allocation (stored indices)");
    }
    *out = (int64_t)g->h.stored_idx.size();
    return GPE_OK;
}

int gpe_grid_layout_info(const gpe_grid* g, gpe_layout_info* out) {
    if (!g || !out) return fail(GPE_ERR_INVALID_ARG, "null argument");
    out->tx = g->h.tx; out->ty = g->h.ty; out->zt = g->h.zt; out->halo_width = g->h.halo_width;
    out->n_active = g->h.n_active;
    out->n_tiles = g->h.n_tiles();
    out->n_slabs = g->h.n_slabs();
    out->n_work = g->h.n_work();
    return GPE_OK;
}

int gpe_grid_active_indices(const gpe_grid* g, int64_t* out_host) {
    if (!g || !out_host) return fail(GPE_ERR_INVALID_ARG, "null argument");
    if (g->h.n_active) std::memcpy(out_host, g->h.active_idx.data(), (size_t)g->h.n_active * sizeof(int64_t));
    return GPE_OK;
}

int gpe_grid_stored_indices(gpe_grid* g, int64_t* out_host) {
    if (!g || !out_host) return fail(GPE_ERR_INVALID_ARG, "null argument");
    try {
        build_stored_indices(&g->h);
    } catch (const std::bad_alloc&) {
        return fail(GPE_ERR_OUT_OF_MEMORY, "host allocation (stored indices)");
    }
    if (!g->h.stored_idx.empty()) std::memcpy(out_host, g->h.stored_idx.data(), g->h.stored_idx.size() * sizeof(int64_t));
    return GPE_OK;
}

int gpe_grid_layout_tables(const gpe_grid* g, const gpe_layout_tables* o) {
    if (!g || !o) return fail(GPE_ERR_INVALID_ARG, "null argument");
    const GridHost& h = g->h;
    auto cp = [](void* dst, const void* src, size_t bytes) { if (dst && bytes) std::memcpy(dst, src, bytes); };
    cp(o->tile_xy, h.tile_xy.data(), h.tile_xy.size() * sizeof(int32_t));
    cp(o->tile_zlo, h.tile_zlo.data(), h.tile_zlo.size() * sizeof(int32_t));
    cp(o->tile_zhi, h.tile_zhi.data(), h.tile_zhi.size() * sizeof(int32_t));
    cp(o->tile_entry_base, h.tile_entry_base.data(), h.tile_entry_base.size() * sizeof(int64_t));
    cp(o->tile_nbr, h.tile_nbr.data(), h.tile_nbr.size() * sizeof(int32_t));
    cp(o->slab_mask, h.slab_mask.data(), h.slab_mask.size() * sizeof(uint64_t));
    cp(o->slab_base, h.slab_base.data(), h.slab_base.size() * sizeof(int64_t));
    cp(o->wi_tile, h.wi_tile.data(), h.wi_tile.size() * sizeof(int32_t));
    cp(o->wi_z0, h.wi_z0.data(), h.wi_z0.size() * sizeof(int32_t));
    cp(o->wi_nz, h.wi_nz.data(), h.wi_nz.size() * sizeof(int32_t));
    cp(o->storage_to_canonical, h.storage_to_canonical.data(), h.storage_to_canonical.size() * sizeof(int64_t));
    return GPE_OK;
}

int gpe_sim_state_bytes(const gpe_grid* g, int dtype, size_t* out) {
    if (!g || !out) return fail(GPE_ERR_INVALID_ARG, "null argument");
    if (dtype != GPE_C64 && dtype != GPE_C128 && dtype != GPE_R64) return fail(GPE_ERR_INVALID_ARG, "unknown dtype");
    *out = 5 * buf_bytes(g->h.n_active, dtype);
    return GPE_OK;
}

int gpe_sim_create(gpe_grid* g, int dtype, int stencil, double g_int, double n_target, void* dev_state,
                   size_t state_bytes, void* stream, gpe_sim** out) {
    if (!g || !dev_state || !out) return fail(GPE_ERR_INVALID_ARG, "null argument");
    if (dtype != GPE_C64 && dtype != GPE_C128 && dtype != GPE_R64) return fail(GPE_ERR_INVALID_ARG, "unknown dtype");
    if (stencil != 7 && stencil != 13 && stencil != 19 && stencil != 27) return fail(GPE_ERR_INVALID_ARG, "stencil must be 7, 13, 19 or 27");
    if (!(n_target > 0.0)) return fail(GPE_ERR_INVALID_ARG, "n_target must be > 0");
    const int radius = stencil == 13 ? 2 : 1;
    if (g->h.tx != 8 || g->h.ty != 8) return fail(GPE_ERR_UNSUPPORTED, "kernels need 8x8 column tiles");
    if (g->h.halo_width < radius) return fail(GPE_ERR_UNSUPPORTED, "grid halo_width is smaller than the stencil radius");
    if (g->h.n_active >= ((int64_t)1 << 32)) return fail(GPE_ERR_UNSUPPORTED, "more than 2^32-1 active points (kernels index storage with 32 bits)");
    if (((uintptr_t)dev_state & 255) != 0) return fail(GPE_ERR_INVALID_ARG, "dev_state must be 256-byte aligned");
    const size_t bb = buf_bytes(g->h.n_active, dtype);
    if (state_bytes < 5 * bb) return fail(GPE_ERR_INVALID_ARG, "state_bytes too small (see gpe_sim_state_bytes)");
    {
        // Checked before anything is allocated.  The grid's tables live on the device that was current when its first
        // sim was created (upload_grid below, if this is the first): every sim on the grid, and its state buffer, must
        // be on that device.  The state may be device memory of that device or managed memory.
        int dev = -1;
        CU(cudaGetDevice(&dev));
        if (g->on_device && dev != g->device) return fail(GPE_ERR_STATE, "the current device is not the one the grid's tables were uploaded to");
        cudaPointerAttributes attr;
        cudaError_t pe = cudaPointerGetAttributes(&attr, dev_state);
        const bool ok = pe == cudaSuccess && (attr.type == cudaMemoryTypeManaged || (attr.type == cudaMemoryTypeDevice && attr.device == dev));
        if (!ok) {
            cudaGetLastError();
            return fail(GPE_ERR_INVALID_ARG, "dev_state is neither device memory of the current (= the grid's) device nor managed memory");
        }
    }
    int rc = upload_grid(g);
    if (rc) return rc;
    gpe_sim* s = new (std::nothrow) gpe_sim();
    if (!s) return fail(GPE_ERR_OUT_OF_MEMORY, "host allocation");
    s->grid = g;
    s->dtype = dtype;
    s->radius = radius;
    s->hoc = stencil == 19 || stencil == 27;
    s->g = g_int;
    s->n_target = n_target;
    s->csize = dtype == GPE_C128 ? 16 : 8;
    s->n = g->h.n_active;
    // planes per stream: small grids are cut into shorter streams so that every SM holds several
    // (measured on B200: 67 k points best at 4, 1.2 M at 8, 1e7 at 16; from 2e7 points on the 13- / 19-point kernels
    // are best at 32, the 7-point kernels, whose streams are long runs of cheap planes, at 24: cfg 3a 0.82 of the copy
    // rate against 0.78 at 32; round-2 builder's notes, variants not in the tree 6.9)
    s->kz = s->n < 300000 ? 4 : s->n < 3000000 ? 8 : s->n < 20000000 ? 16 : 32;
    if (s->kz == 32 && !s->hoc && s->radius == 1) s->kz = 24;
    for (int k = 0; k < 4; ++k) s->buf[k] = (char*)dev_state + k * bb;
    s->staging = (char*)dev_state + 4 * bb;
    cudaError_t e = cudaMalloc(&s->d_sums, (NACC + 2) * sizeof(double));
    if (e != cudaSuccess) { delete s; return e == cudaErrorMemoryAllocation ? fail(GPE_ERR_OUT_OF_MEMORY, "cudaMalloc") : cuda_fail(e, "cudaMalloc"); }
    e = cudaMallocHost(&s->h_flag, sizeof(double));
    if (e == cudaSuccess) { *s->h_flag = 0.0; e = cudaEventCreateWithFlags(&s->ev_flag, cudaEventDisableTiming); }
    if (e != cudaSuccess) { gpe_sim_destroy(s); return cuda_fail(e, "pinned flag / event"); }
    rc = build_work(s);
    if (rc) { gpe_sim_destroy(s); return rc; }
    cudaStream_t st = (cudaStream_t)stream;
    e = cudaMemsetAsync(dev_state, 0, 5 * bb, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(s->d_sums, 0, (NACC + 2) * sizeof(double), st);
    if (e == cudaSuccess) e = (cudaError_t)launch_set_scalar(s->d_sums + NACC, 1.0, stream);
    if (e != cudaSuccess) { gpe_sim_destroy(s); return cuda_fail(e, "state initialisation"); }
    g->n_sims += 1;
    s->counted = true;
    s->launches += 1;
    *out = s;
    return GPE_OK;
}

int gpe_sim_destroy(gpe_sim* s) {
    if (!s) return GPE_OK;
    if (s->d_work) cudaFree(s->d_work);
    if (s->d_partials) cudaFree(s->d_partials);
    if (s->d_sums) cudaFree(s->d_sums);
    if (s->d_map) cudaFree(s->d_map);
    if (s->h_flag) cudaFreeHost(s->h_flag);
    if (s->ev_flag) cudaEventDestroy(s->ev_flag);
    if (s->rk4_exec) cudaGraphExecDestroy(s->rk4_exec);
    if (s->cap_stream) cudaStreamDestroy(s->cap_stream);
    for (int k = 0; k < 2; ++k)
        if (s->extra[k]) cudaFree(s->extra[k]);
    for (int k = 0; k < 4; ++k)
        for (cudaEvent_t e : s->ev[k]) cudaEventDestroy(e);
    if (s->counted && s->grid && s->grid->n_sims > 0) s->grid->n_sims -= 1;
    delete s;
    return GPE_OK;
}

int gpe_set_psi(gpe_sim* s, const void* dev_psi_canonical, void* stream) {
    if (!s || (!dev_psi_canonical && s->n > 0)) return fail(GPE_ERR_INVALID_ARG, "null argument");
    KL(launch_pack(copy_dtype(s->dtype), dev_psi_canonical, s->buf[0], s->grid->d_perm, s->n, stream));
    if (s->n > 0) s->launches += 1;
    return drop_flag(s, stream);
}

int gpe_get_psi(gpe_sim* s, void* dev_psi_canonical, void* stream) {
    if (!s || (!dev_psi_canonical && s->n > 0)) return fail(GPE_ERR_INVALID_ARG, "null argument");
    KL(launch_unpack(copy_dtype(s->dtype), s->buf[0], dev_psi_canonical, s->grid->d_perm, s->n, stream));
    if (s->n > 0) s->launches += 1;
    return GPE_OK;
}

int gpe_remap_psi(gpe_sim* src, gpe_sim* dst, void* stream) {
    if (!src || !dst || src == dst) return fail(GPE_ERR_INVALID_ARG, "null or identical simulations");
    if (src->dtype != dst->dtype) return fail(GPE_ERR_INVALID_ARG, "source and destination precisions differ");
    const gpe_box &a = src->grid->h.box, &b = dst->grid->h.box;
    if (a.nx != b.nx || a.ny != b.ny || a.nz != b.nz || a.h != b.h || a.hy != b.hy || a.hz != b.hz || a.center[0] != b.center[0] ||
        a.center[1] != b.center[1] || a.center[2] != b.center[2])
        return fail(GPE_ERR_INVALID_ARG, "the two grids must be post-selected from the same bounding box");
    {
        // the index table is built on the host and copied from pageable memory: that cannot go into a stream capture
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing((cudaStream_t)stream, &cs) != cudaSuccess) { cudaGetLastError(); cs = cudaStreamCaptureStatusNone; }
        if (cs != cudaStreamCaptureStatusNone)
            return fail(GPE_ERR_UNSUPPORTED, "gpe_remap_psi cannot be part of a stream capture (it uploads a host-built index table)");
    }
    dst->t = src->t;
    if (dst->n == 0) return GPE_OK;
    // new canonical rank -> old canonical rank (both index lists ascend: one merge pass), -1 = new point
    const std::vector<int64_t>&ia = src->grid->h.active_idx, &ib = dst->grid->h.active_idx;
    std::vector<int64_t> map((size_t)dst->n);
    size_t j = 0;
    for (size_t i = 0; i < ib.size(); ++i) {
        while (j < ia.size() && ia[j] < ib[i]) ++j;
        map[i] = (j < ia.size() && ia[j] == ib[i]) ? (int64_t)j : -1;
    }
    if (!dst->d_map) {   // kept for the life of the destination sim: a ramp re-grids after every stage
        cudaError_t em = cudaMalloc(&dst->d_map, map.size() * sizeof(int64_t));
        if (em == cudaErrorMemoryAllocation) return fail(GPE_ERR_OUT_OF_MEMORY, "cudaMalloc(remap table)");
        CU(em);
    }
    cudaStream_t st = (cudaStream_t)stream;
    // pageable source: the call returns once the host vector has been staged, the device copy is stream-ordered
    CU(cudaMemcpyAsync(dst->d_map, map.data(), map.size() * sizeof(int64_t), cudaMemcpyHostToDevice, st));
    if (src->n > 0) KL(launch_unpack(copy_dtype(src->dtype), src->buf[0], src->staging, src->grid->d_perm, src->n, stream));
    KL(launch_remap(copy_dtype(dst->dtype), src->staging, dst->staging, dst->d_map, dst->n, stream));
    KL(launch_pack(copy_dtype(dst->dtype), dst->staging, dst->buf[0], dst->grid->d_perm, dst->n, stream));
    src->launches += src->n > 0 ? 1 : 0;
    dst->launches += 2;
    return drop_flag(dst, stream);
}

int gpe_set_psi_host(gpe_sim* s, const void* host_psi_canonical, void* stream) {
    if (!s || (!host_psi_canonical && s->n > 0)) return fail(GPE_ERR_INVALID_ARG, "null argument");
    if (s->n == 0) return GPE_OK;
    CU(cudaMemcpyAsync(s->staging, host_psi_canonical, (size_t)s->n * s->csize, cudaMemcpyHostToDevice, (cudaStream_t)stream));
    int rc = gpe_set_psi(s, s->staging, stream);
    if (rc) return rc;
    CU(cudaStreamSynchronize((cudaStream_t)stream));
    return GPE_OK;
}

int gpe_get_psi_host(gpe_sim* s, void* host_psi_canonical, void* stream) {
    if (!s || (!host_psi_canonical && s->n > 0)) return fail(GPE_ERR_INVALID_ARG, "null argument");
    if (s->n == 0) return GPE_OK;
    int rc = gpe_get_psi(s, s->staging, stream);
    if (rc) return rc;
    CU(cudaMemcpyAsync(host_psi_canonical, s->staging, (size_t)s->n * s->csize, cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    CU(cudaStreamSynchronize((cudaStream_t)stream));
    return check_flag(s, true, stream);
}

int gpe_set_time(gpe_sim* s, double t) {
    if (!s) return fail(GPE_ERR_INVALID_ARG, "null argument");
    if (!std::isfinite(t)) return fail(GPE_ERR_INVALID_ARG, "t must be finite");
    s->t = t;
    return GPE_OK;
}

int gpe_get_time(const gpe_sim* s, double* t) {
    if (!s || !t) return fail(GPE_ERR_INVALID_ARG, "null argument");
    *t = s->t;
    return GPE_OK;
}

int gpe_apply_H(gpe_sim* s, double t, const void* dev_in_canonical, void* dev_out_canonical, void* stream) {
    if (!s || ((!dev_in_canonical || !dev_out_canonical) && s->n > 0)) return fail(GPE_ERR_INVALID_ARG, "null argument");
    if (s->n == 0) return GPE_OK;
    const char* a = (const char*)dev_in_canonical;
    const char* b = (const char*)dev_out_canonical;
    const size_t bytes = (size_t)s->n * s->csize;
    if (a < b + bytes && b < a + bytes) return fail(GPE_ERR_INVALID_ARG, "in and out overlap");
    // scratch: C holds the packed input, D the packed result; the sim's psi (A) is untouched
    KL(launch_pack(copy_dtype(s->dtype), dev_in_canonical, s->buf[2], s->grid->d_perm, s->n, stream));
    s->launches += 1;
    int rc = stage(s, MODE_APPLY, t, 0.0, s->buf[2], nullptr, s->buf[3], nullptr, stream);
    if (rc) return rc;
    KL(launch_unpack(copy_dtype(s->dtype), s->buf[3], dev_out_canonical, s->grid->d_perm, s->n, stream));
    s->launches += 1;
    return GPE_OK;
}

int gpe_run_rk4(gpe_sim* s, double dt, int64_t nsteps, void* stream) {
    if (!s) return fail(GPE_ERR_INVALID_ARG, "null argument");
    if (s->dtype == GPE_R64) return fail(GPE_ERR_UNSUPPORTED, "real-time evolution needs a complex state (GPE_C64 / GPE_C128)");
    if (!std::isfinite(dt) || nsteps < 0) return fail(GPE_ERR_INVALID_ARG, "bad dt or nsteps");
    const double t0 = s->t;
    for (int64_t n = rk4_graph_steps(s, t0, dt, nsteps, stream); n < nsteps; ++n) {
        int rc = rk4_step(s, t0 + (double)n * dt, dt, stream);
        if (rc) return rc;
    }
    s->t = t0 + (double)nsteps * dt;
    return GPE_OK;
}

int gpe_step_rk4(gpe_sim* s, double dt, void* stream) { return gpe_run_rk4(s, dt, 1, stream); }

int gpe_run_rkhe3(gpe_sim* s, double dt, int64_t nsteps, void* stream) {
    if (!s) return fail(GPE_ERR_INVALID_ARG, "null argument");
    if (s->dtype == GPE_R64) return fail(GPE_ERR_UNSUPPORTED, "real-time evolution needs a complex state (GPE_C64 / GPE_C128)");
    if (!std::isfinite(dt) || nsteps < 0) return fail(GPE_ERR_INVALID_ARG, "bad dt or nsteps");
    const double t0 = s->t;
    for (int64_t n = 0; n < nsteps; ++n) {
        int rc = rkhe3_step(s, t0 + (double)n * dt, dt, stream);
        if (rc) return rc;
    }
    s->t = t0 + (double)nsteps * dt;
    return GPE_OK;
}

int gpe_step_rkhe3(gpe_sim* s, double dt, void* stream) { return gpe_run_rkhe3(s, dt, 1, stream); }

int gpe_run_rkck(gpe_sim* s, double dt, int64_t nsteps, void* stream) {
    if (!s) return fail(GPE_ERR_INVALID_ARG, "null argument");
    if (s->dtype == GPE_R64) return fail(GPE_ERR_UNSUPPORTED, "real-time evolution needs a complex state (GPE_C64 / GPE_C128)");
    if (!std::isfinite(dt) || nsteps < 0) return fail(GPE_ERR_INVALID_ARG, "bad dt or nsteps");
    if (s->n > 0 && nsteps > 0) {
        for (int k = 0; k < 2; ++k) {
            if (s->extra[k]) continue;
            cudaError_t e = cudaMalloc(&s->extra[k], buf_bytes(s->n, s->dtype));
            if (e == cudaErrorMemoryAllocation) return fail(GPE_ERR_OUT_OF_MEMORY, "cudaMalloc(RKCK stage states)");
            CU(e);
            CU(cudaMemsetAsync(s->extra[k], 0, buf_bytes(s->n, s->dtype), (cudaStream_t)stream));
        }
    }
    const double t0 = s->t;
    for (int64_t n = 0; n < nsteps; ++n) {
        int rc = rkck_step(s, t0 + (double)n * dt, dt, stream);
        if (rc) return rc;
    }
    s->t = t0 + (double)nsteps * dt;
    return GPE_OK;
}

int gpe_step_rkck(gpe_sim* s, double dt, void* stream) { return gpe_run_rkck(s, dt, 1, stream); }

int gpe_run_imag(gpe_sim* s, double dt, int64_t nsteps, void* stream) {
    if (!s) return fail(GPE_ERR_INVALID_ARG, "null argument");
    if (!std::isfinite(dt) || nsteps < 0) return fail(GPE_ERR_INVALID_ARG, "bad dt or nsteps");
    if (s->n == 0 || nsteps == 0) return GPE_OK;
    { int rcf = check_flag(s, false, stream); if (rcf) return rcf; }
    const double h3 = cell_volume(s->grid->h.box);
    for (int64_t n = 0; n < nsteps; ++n) {
        int rc = stage(s, MODE_IMAG, s->t, dt, s->buf[0], nullptr, s->buf[1], nullptr, stream);
        if (rc) return rc;
        KL(launch_finalize(s->d_partials, s->n_blocks, s->d_sums, s->d_sums + NACC, s->n_target, h3, stream));
        s->launches += 1;
        std::swap(s->buf[0], s->buf[1]);
    }
    // flush the lazy scale so that every other call sees a normalised state
    return flush_scale(s, stream);
}

int gpe_imag_step(gpe_sim* s, double dt, void* stream) { return gpe_run_imag(s, dt, 1, stream); }

int gpe_run_imag_split(gpe_sim* s, double dt, int64_t nsteps, void* stream) {
    if (!s) return fail(GPE_ERR_INVALID_ARG, "null argument");
    if (!std::isfinite(dt) || nsteps < 0) return fail(GPE_ERR_INVALID_ARG, "bad dt or nsteps");
    if (s->n == 0 || nsteps == 0) return GPE_OK;
    { int rcf = check_flag(s, false, stream); if (rcf) return rcf; }
    const double h3 = cell_volume(s->grid->h.box);
    const double hdt = 0.5 * dt;
    const bool k1 = s->opt_k1 != 0;                         // GPE_OPT_FUSED_K1 = 0: three launches (PREP, KIN, SPLITB)
    for (int64_t n = 0; n < nsteps; ++n) {
        // A holds the un-normalised state of the previous iteration; its scale sits in d_sums[NACC]
        int rc;
        if (k1) {
            // the paper's two stencil kernels: K1 = Eq. 7 half step + lazy scale applied while loading, first
            // Euler half step; K2 = second Euler half step + Eq. 7 + partial sums.  4 values per point and iteration.
            rc = stage(s, MODE_KINP, s->t, hdt, s->buf[0], nullptr, s->buf[1], nullptr, stream);
            if (!rc) rc = stage(s, MODE_SPLITB, s->t, hdt, s->buf[1], nullptr, s->buf[0], nullptr, stream);
        } else {
            rc = stage(s, MODE_PREP, s->t, hdt, s->buf[0], nullptr, s->buf[1], nullptr, stream);
            if (!rc) rc = stage(s, MODE_KIN, s->t, hdt, s->buf[1], nullptr, s->buf[0], nullptr, stream);
            if (!rc) rc = stage(s, MODE_SPLITB, s->t, hdt, s->buf[0], nullptr, s->buf[1], nullptr, stream);
        }
        if (rc) return rc;
        KL(launch_finalize(s->d_partials, s->n_blocks, s->d_sums, s->d_sums + NACC, s->n_target, h3, stream));
        s->launches += 1;
        if (!k1) std::swap(s->buf[0], s->buf[1]);
    }
    return flush_scale(s, stream);
}

int gpe_imag_split_step(gpe_sim* s, double dt, void* stream) { return gpe_run_imag_split(s, dt, 1, stream); }

int gpe_norm(gpe_sim* s, double* out_host, void* stream) {
    if (!s || !out_host) return fail(GPE_ERR_INVALID_ARG, "null argument");
    const double h3 = cell_volume(s->grid->h.box);
    if (s->n == 0) { *out_host = 0.0; return GPE_OK; }
    KL(launch_norm_partials(pair_dtype(s->dtype), s->buf[0], pair_count(s->dtype, s->n), s->d_partials, stream));
    KL(launch_finalize(s->d_partials, norm_blocks(pair_count(s->dtype, s->n)), s->d_sums, nullptr, s->n_target, h3, stream));
    s->launches += 2;
    double sums[NACC];
    int rc = sums_to_host(s, sums, stream);
    if (!rc) rc = check_flag(s, true, stream);
    if (rc) return rc;
    const double v = h3 * sums[0];
    if (!std::isfinite(v)) return fail(GPE_ERR_STATE, "norm is not finite");
    *out_host = v;
    return GPE_OK;
}

int gpe_energy(gpe_sim* s, gpe_energy_out* o, void* stream) {
    if (!s || !o) return fail(GPE_ERR_INVALID_ARG, "null argument");
    const double h3 = cell_volume(s->grid->h.box);
    if (s->n == 0) return fail(GPE_ERR_STATE, "empty grid has no energy");
    int rc = stage(s, MODE_ENERGY, s->t, 0.0, s->buf[0], nullptr, nullptr, nullptr, stream);
    if (rc) return rc;
    KL(launch_finalize(s->d_partials, s->n_blocks, s->d_sums, nullptr, s->n_target, h3, stream));
    s->launches += 1;
    double sums[NACC];
    rc = sums_to_host(s, sums, stream);
    if (!rc) rc = check_flag(s, true, stream);
    if (rc) return rc;
    gpe_energy_out r;
    r.kin = h3 * sums[0];
    r.pot = h3 * sums[1];
    r.inter = h3 * 0.5 * s->g * sums[2];
    r.norm = h3 * sums[3];
    r.total = r.kin + r.pot + r.inter;
    r.mu = (r.kin + r.pot + 2.0 * r.inter) / r.norm;
    if (!std::isfinite(r.mu) || !(r.norm > 0.0)) return fail(GPE_ERR_STATE, "state has zero or non-finite norm");
    *o = r;
    return GPE_OK;
}

int gpe_sim_kernel_launches(const gpe_sim* s, int64_t* out) {
    if (!s || !out) return fail(GPE_ERR_INVALID_ARG, "null argument");
    *out = s->launches;
    return GPE_OK;
}

int gpe_sim_time_stages(gpe_sim* s, int on) {
    if (!s) return fail(GPE_ERR_INVALID_ARG, "null argument");
    s->timing = on != 0;
    for (int k = 0; k < 4; ++k) s->ev_used[k] = 0;
    return GPE_OK;
}

int gpe_sim_stage_time_ms(gpe_sim* s, double ms_out[4], int64_t count_out[4]) {
    if (!s || !ms_out || !count_out) return fail(GPE_ERR_INVALID_ARG, "null argument");
    for (int k = 0; k < 4; ++k) {
        double acc = 0.0;
        for (size_t u = 0; u + 1 < s->ev_used[k]; u += 2) {
            CU(cudaEventSynchronize(s->ev[k][u + 1]));
            float ms = 0.f;
            CU(cudaEventElapsedTime(&ms, s->ev[k][u], s->ev[k][u + 1]));
            acc += ms;
        }
        ms_out[k] = acc;
        count_out[k] = (int64_t)(s->ev_used[k] / 2);
        s->ev_used[k] = 0;
    }
    return GPE_OK;
}

int gpe_sim_set_compact_weights(gpe_sim* s, double centre, const double* face_xyz, const double* edge_xy_xz_yz, double corner) {
    if (!s || !face_xyz || !edge_xy_xz_yz) return fail(GPE_ERR_INVALID_ARG, "null argument");
    if (!s->hoc) return fail(GPE_ERR_STATE, "the sim was not created with the 19- or 27-point stencil");
    const double v[8] = {centre, face_xyz[0], face_xyz[1], face_xyz[2], edge_xy_xz_yz[0], edge_xy_xz_yz[1], edge_xy_xz_yz[2], corner};
    for (double x : v)
        if (!std::isfinite(x)) return fail(GPE_ERR_INVALID_ARG, "weights must be finite");
    for (int k = 0; k < 8; ++k) s->w27[k] = v[k];
    s->custom27 = true;
    return GPE_OK;
}

int gpe_sim_set_option(gpe_sim* s, int option, int value) {
    if (!s) return fail(GPE_ERR_INVALID_ARG, "null argument");
    if (value != 0 && value != 1) return fail(GPE_ERR_INVALID_ARG, "option values are 0 or 1");
    switch (option) {
        case GPE_OPT_FUSED_K1: s->opt_k1 = value; return GPE_OK;
        case GPE_OPT_RK4_GRAPH: s->opt_graph = value; return GPE_OK;
        case GPE_OPT_PDL:
            if (s->opt_pdl != value && s->rk4_exec) {   // the captured launches carry the old attribute
                CU(cudaDeviceSynchronize());
                cudaGraphExecDestroy(s->rk4_exec);
                s->rk4_exec = nullptr;
            }
            s->opt_pdl = value;
            return GPE_OK;
        default: return fail(GPE_ERR_INVALID_ARG, "unknown option");
    }
}

int gpe_sim_set_planes_per_block(gpe_sim* s, int kz) {
    if (!s) return fail(GPE_ERR_INVALID_ARG, "null argument");
    if (kz < 1 || kz > stage_max_planes()) return fail(GPE_ERR_INVALID_ARG, "planes per stream must be in 1..32");
    CU(cudaDeviceSynchronize());
    s->kz = kz;
    return build_work(s);
}

}  // extern "C"
