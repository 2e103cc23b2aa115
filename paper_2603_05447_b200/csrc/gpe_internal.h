// Internal declarations shared by the host layout builder (gpe_layout.cpp), the C-ABI glue
// (gpe_api.cu) and the kernels (gpe_kernels.cu).  Not part of the public boundary (include/gpe.h).
#pragma once

#include <cstdint>
#include <string>
#include <vector>

#include "gpe.h"

namespace gpe {

// ---------------------------------------------------------------------------------------------
// Host-side layout (prior art PAPER.md:81-85)
// ---------------------------------------------------------------------------------------------
struct GridHost {
    gpe_box box{};
    gpe_potential pot{};
    double v_cut = 0.0;
    int halo_width = 0;
    int tx = 8, ty = 8, zt = 32;
    int ntx = 0, nty = 0;
    int64_t n_active = 0;

    std::vector<int32_t> tile_xy;          // [n_tiles][2]
    std::vector<int32_t> tile_zlo, tile_zhi;
    std::vector<int64_t> tile_entry_base;  // [n_tiles]
    std::vector<int32_t> tile_nbr;         // [n_tiles][4]
    std::vector<uint64_t> slab_mask;       // [n_slabs]
    std::vector<int64_t> slab_base;        // [n_slabs]
    std::vector<int32_t> wi_tile, wi_z0, wi_nz;
    std::vector<int64_t> storage_to_canonical;  // [n_active]
    std::vector<int64_t> active_idx;            // [n_active]

    bool stored_ready = false;
    std::vector<int64_t> stored_idx;

    int64_t n_tiles() const { return (int64_t)tile_zlo.size(); }
    int64_t n_slabs() const { return (int64_t)slab_mask.size(); }
    int64_t n_work() const { return (int64_t)wi_tile.size(); }
};

// Builders: return GPE_OK or an error code and fill `err`.
int build_layout_from_potential(const gpe_box& box, const gpe_potential& pot, double v_cut, int halo_width,
                                GridHost* out, std::string* err);
int build_layout_from_indices(const gpe_box& box, const gpe_potential& pot, const int64_t* active, int64_t n,
                              int halo_width, GridHost* out, std::string* err);
void build_stored_indices(GridHost* g);

// Delta(t) of the linear ramp (R16); same formula as the oracle's, one rounding each.
double delta_of_t(const gpe_potential& pot, double t);

// ---------------------------------------------------------------------------------------------
// Device-side tables and kernel parameters
// ---------------------------------------------------------------------------------------------
struct Slab {                // one z-plane of one tile
    unsigned long long mask; // bit lx*8+ly set iff the point is in M
    long long base;          // storage position of the slab's first lane
};

// One stream (a warp's worth of work): nz consecutive planes of one tile (a piece of a work item).
// eoff[q] + zp = slab entry of plane zp in tile q (0 = own, 1..4 = -x,+x,-y,+y, 5..8 = the diagonal tiles
// (-x,-y), (-x,+y), (+x,-y), (+x,+y) whose corner points the 19-point stencil reads), valid for
// zlo[q] <= zp < zhi[q] (zlo = zhi = 0 when the neighbour tile is absent).
constexpr int NTILE = 9;
struct alignas(16) WorkRec {
    int32_t ix0, iy0;   // box index of the tile's (lx,ly) = (0,0) column
    int32_t z0, nz;
    long long eoff[NTILE];
    int32_t zlo[NTILE];
    int32_t zhi[NTILE];
    long long pos0;     // storage position of the first point of the piece
    int32_t npts;       // points in the piece (contiguous in storage from pos0)
    int32_t lead;       // overlap planes below z0 the stream reads: R, or 0 when the tile holds no point in them
    int32_t pad[2];
};
static_assert(sizeof(WorkRec) == 192, "WorkRec layout");

struct PotDev {
    int32_t kind;
    int32_t nx, ny, nz;
    double h, cx, cy, cz;   // h = spacing along x
    double hy, hz;          // spacing along y, z (= h on isotropic grids)
    double ax, ay, az;
    double delta;   // Delta at the stage time (host-computed, R16)
    double omega;
};

enum Mode : int {
    MODE_APPLY = 0,  // out1 = H c
    MODE_S1 = 1,     // out1 = c + ca * f(c)                        f(c) = -i H c
    MODE_S2 = 2,     // out1 = aux + ca * f(c); out2 = comb[0] aux + comb[1] c + comb[2] out1  (RK4: -1/3, 1/3, 2/3)
    MODE_S3 = 3,     // out1 = aux + ca * f(c)
    MODE_S4 = 4,     // out1 = aux + 1/3 c + ca * f(c)
    MODE_IMAG = 5,   // psi = scale * c; out1 = psi - ca * H psi; partial sum of |out1|^2
    MODE_ENERGY = 6, // partial sums of Re(conj(c) T c), V|c|^2, |c|^4, |c|^2
    // the paper's own imaginary-time iteration, ca = dt/2:
    MODE_PREP = 7,   // pointwise: psi = scale * c; out1 = psi exp(-V ca) (1 - g ca |psi|^2)       (Eq. 7, lazy scale)
    MODE_KIN = 8,    // out1 = c - ca T c                                                          (first Euler half step)
    MODE_SPLITB = 9, // u = c - ca T c; out1 = u exp(-V ca) (1 - g ca |u|^2); partial sum of |out1|^2
    // general stage of the memory-optimised Runge-Kutta form (PAPER.md:276-281 Eq. A6-A7; used for RKCK, A12-A13):
    MODE_LC = 10,    // out1 = sum_{j < n_aux} coef[j] auxn[j] + coefc c + ca * f(c)
    // the paper's kernel K1: MODE_PREP folded into MODE_KIN's load -- every value staged for the stencil
    // (own and halo) becomes a = s c exp(-V ca) (1 - g ca |s c|^2) in shared memory, then out1 = a - ca T a
    MODE_KINP = 11
};
constexpr int MAX_LC_AUX = 5;
constexpr int NACC = 4;           // accumulators per block in the partial-sum array
constexpr int STAGE_THREADS = 32;

struct StageParams {
    const Slab* slabs;
    const WorkRec* work;
    int32_t n_work;
    int32_t kz;            // max planes per stream (informational; the split is done on the host)
    PotDev pot;
    double g;
    double ca;             // stage coefficient (dt/2, dt, dt/6, or dt of the imaginary step)
    // host-precomputed constants (read from the parameter bank, no registers):
    // stencil weights times -1/2, per axis a = x, y, z with its own 1/d_a^2 (PAPER.md:337-343 Eq. B1-B2):
    // kw[a][s] = weight of the neighbours s steps along a (s = 1, 2; 19-point: the face weight at s = 1);
    // kw[0][0] = the centre weight (all axes together); ke[] = 19-point edge weights xy, xz, yz
    double kw[3][3];
    double ke[3];
    double kcn;            // corner weight of the 27-point compact stencil (0 for the 19-point one)
    float kwf[3][3];       // the same in fp32 (complex64 state)
    float kef[3];
    float kcnf;
    float padf[3];
    double xc, yc, zc;     // 0.5 (n-1) per axis: coordinate = (i - xc) h + cx
    double hax, hay, haz;  // 0.5 a_x, 0.5 a_y, 0.5 a_z
    double om2;            // Omega^2
    double delta_eff;      // Delta(t) for the dressed potential, 0 for the harmonic one
    const void* auxn[5];   // MODE_LC: earlier stage states y^(j) (storage order), read at the point itself only
    double coef[5];        // MODE_LC: a*_{ij} (or b*_j) of those states
    double coefc;          // MODE_LC: a*_{ii} (or b*_i) of the stage state c the stencil is applied to
    int32_t n_aux;         // MODE_LC: number of entries of auxn / coef in use
    int32_t pad_lc;
    double comb[3];        // MODE_S2: out2 = comb[0] aux + comb[1] c + comb[2] out1 (the b* terms known so far, Eq. A7)
    const void* in;        // array the stencil is applied to (storage order)
    const void* aux;       // y0 or p (storage order) or null
    void* out1;
    void* out2;
    const double* scale_in;  // MODE_IMAG: device scalar multiplying `in` on load (lazy renormalisation)
    double* partials;        // MODE_IMAG / MODE_ENERGY: [n_work][NACC] block partial sums
};

// Launchers (gpe_kernels.cu).  dtype: GPE_C64 / GPE_C128; radius 1 or 2.  Return cudaError_t as int.
// variant: 1 = 7-point, 2 = 13-point, 3 = 19-point higher-order compact (radius 1 + in-plane / z diagonals)
// pdl != 0: the launch carries the programmatic-stream-serialization attribute (the kernels call griddepcontrol)
int launch_stage(int dtype, int variant, int mode, const StageParams& p, void* stream, int pdl);
size_t stage_smem_bytes(int dtype, int variant);
int stage_max_planes();   // upper bound of WorkRec::nz the stage kernels accept
int launch_pack(int dtype, const void* canonical, void* storage, const int64_t* perm, int64_t n, void* stream);
int launch_unpack(int dtype, const void* storage, void* canonical, const int64_t* perm, int64_t n, void* stream);
// dst_canonical[i] = map[i] >= 0 ? src_canonical[map[i]] : 0   (re-gridding)
int launch_remap(int dtype, const void* src_canonical, void* dst_canonical, const int64_t* map, int64_t n_dst, void* stream);
// partials[b*NACC + 0] = sum over the block's contiguous chunk of |psi|^2; nblk = norm_blocks(n)
int norm_blocks(int64_t n);
int launch_norm_partials(int dtype, const void* storage, int64_t n, double* partials, void* stream);
// out[k] = sum_b partials[b*NACC + k] in a fixed order (k < NACC); if scale_out != null also writes
// scale_out[0] = sqrt(n_target / (h3 * out[0])), or 1 and the sticky flag scale_out[1] = 1 when out[0] is zero or
// not finite
int launch_finalize(const double* partials, int64_t nblk, double* out, double* scale_out,
                    double n_target, double h3, void* stream);
int launch_scale(int dtype, void* storage, int64_t n, const double* scale, void* stream);
int launch_set_scalar(double* dst, double v, void* stream);
int kernels_configure();  // sets max dynamic shared memory attributes once; returns cudaError_t

// Error text for entry points that live outside gpe_api.cu (gpe_noalloc.cu): store the calling thread's
// gpe_last_error() text and return `code` (api_fail) or GPE_ERR_CUDA (api_cuda_fail, text = what + the CUDA error string).
int api_fail(int code, const char* msg);
int api_cuda_fail(int cuda_error, const char* what);

}  // namespace gpe
