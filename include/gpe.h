/* gpe.h -- C ABI of libgpe_b200.so: the sparse-grid Gross-Pitaevskii hot path on one B200.
 *
 * What the library computes (citations: /root/reference/PAPER.md line, section / equation):
 *   H[psi;t] psi = -1/2 lap_h psi + V(r,t) psi + g |psi|^2 psi        PAPER.md:25-27 Eq. 1-2, :71 Eq. 8
 * on the region of interest M = {p in box : V_mask(r_p) < V_cut}          PAPER.md:50-52 Eq. 5
 * with the rows and columns of points outside M deleted (psi = 0 there)
 * fused into explicit RK4 stages in the memory-optimised form            PAPER.md:89-99, :276-281 Eq. A6-A7,
 *                                                                         :315-319 Eq. A10-A11
 * and into normalised imaginary-time steps with a particle-number
 * reduction and lazy renormalisation                                     PAPER.md:35, :60 Eq. 6, :87 (kernel K3)
 * DESIGN.md lists the readings taken where the paper is silent (R1..R18).
 *
 * Conventions
 *   - every function returns int: 0 = GPE_OK, negative = error; out-parameters are untouched on error;
 *     gpe_last_error() returns thread-local text for the last failing call of the calling thread.
 *   - "host" pointers are ordinary CPU memory owned by the caller; "dev" pointers are CUDA device memory
 *     owned by the caller (e.g. torch tensors' data_ptr()).  The library owns only its tables.
 *   - `stream` is a cudaStream_t passed as void* (0 = legacy default stream).  Device work is enqueued on
 *     it and is asynchronous, EXCEPT calls that return host scalars (gpe_norm, gpe_energy) and the *_host
 *     copies, which synchronise that stream before returning.
 *   - complex values are interleaved (re, im): complex128 = 2 doubles, complex64 = 2 floats.
 *   - global linear index L = (ix*ny + iy)*nz + iz (C order, z fastest); coordinates
 *     x_i = ((double)i - 0.5*(nx-1))*h + center[0] (same for y, z).
 *   - "canonical order" of a wavefunction = ascending L over M, length n_active.
 *   - nothing here falls back to the CPU: with no usable CUDA device the device calls return GPE_ERR_CUDA.
 *   - handles are not thread-safe; use one sim per host thread.
 */
#ifndef GPE_H_
#define GPE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GPE_OK 0
#define GPE_ERR_INVALID_ARG (-1)
#define GPE_ERR_OUT_OF_MEMORY (-2)
#define GPE_ERR_CUDA (-3)
#define GPE_ERR_UNSUPPORTED (-4)
#define GPE_ERR_STATE (-5)

/* potential kinds (BASELINE.json configs; dressed form after PAPER.md:139 Eq. 10) */
#define GPE_POT_HARMONIC 0 /* V = u,  u = 1/2 (ax x^2 + ay y^2 + az z^2)                    */
#define GPE_POT_DRESSED 1  /* V = sqrt((u - Delta(t))^2 + Omega^2) - Omega                  */
/* which Delta defines the mask (R13) */
#define GPE_MASK_AT_DELTA0 0
#define GPE_MASK_AT_DELTA1 1
#define GPE_MASK_UNION 2 /* union over the ramp: Delta = clamp(u, min(d0,d1), max(d0,d1))     */

#define GPE_C64 0  /* complex64 state; coordinates, V and all reductions still fp64           */
#define GPE_C128 1 /* complex128 state                                                        */
#define GPE_R64 2  /* real float64 state for ground states (imaginary time "does not require the
                      wavefunction to be complex"): half the bytes of complex128; the operator, the imaginary-time
                      calls, the reductions and re-gridding only -- the Runge-Kutta calls return UNSUPPORTED.
                      Canonical arrays hold n_active doubles. */

typedef struct gpe_grid gpe_grid; /* opaque: active set + layout tables (host, and device once a sim exists) */
typedef struct gpe_sim gpe_sim;   /* opaque: one wavefunction evolving on a grid                              */

typedef struct {
    int32_t nx, ny, nz; /* box size in points, each >= 1 */
    int32_t reserved;   /* must be 0 */
    double h;           /* grid spacing (along x when hy / hz are given), > 0 */
    double center[3];   /* coordinate of the box centre */
    double hy, hz;      /* grid spacing along y and z for anisotropic grids d_x != d_y != d_z (PAPER.md:333-343
                           App. B: every second difference carries its own 1/d_i^2, the 19-point cross terms
                           (d_i^2 + d_j^2)/12); <= 0 means "same as h".  Sums that stand for integrals use the
                           volume element h hy hz. */
} gpe_box;

typedef struct {
    int32_t kind;      /* GPE_POT_* */
    int32_t mask_mode; /* GPE_MASK_* (ignored for harmonic) */
    double ax, ay, az; /* quadratic-form coefficients */
    double delta0, delta1, t_ramp; /* Delta(t) = delta0 + (delta1-delta0)*clamp(t/t_ramp,0,1); t_ramp<=0: delta0 */
    double omega;
} gpe_potential;

/* Layout: 8x8 column tiles in (x,y), one 64-bit occupancy mask per z-plane ("slab") of a tile, points
 * stored COMPACTLY (no padding, no ghost lanes) in the order tile, z, bit = lx*ty + ly.
 * "Data layout".  Prior art: the paper's 8^3 blocks + 488-entry halo lists. */
typedef struct {
    int32_t tx, ty, zt, halo_width;
    int64_t n_active;  /* |M| */
    int64_t n_tiles;   /* present tiles */
    int64_t n_slabs;   /* sum over tiles of (zhi - zlo) */
    int64_t n_work;    /* work items */
} gpe_layout_info;

/* Caller-allocated host arrays to receive the canonical tables (any pointer may be NULL = skip).
 * Definitions: DESIGN.md "Layout tables"; lengths from gpe_layout_info. */
typedef struct {
    int32_t* tile_xy;              /* [n_tiles][2]  tile coordinates (i, j) = (ix/tx, iy/ty)           */
    int32_t* tile_zlo;             /* [n_tiles]     min iz over the tile's points                      */
    int32_t* tile_zhi;             /* [n_tiles]     max iz + 1                                         */
    int64_t* tile_entry_base;      /* [n_tiles]     index of the tile's first slab                     */
    int32_t* tile_nbr;             /* [n_tiles][4]  present-tile index of (i-1,j),(i+1,j),(i,j-1),(i,j+1) or -1 */
    uint64_t* slab_mask;           /* [n_slabs]     bit lx*ty+ly set iff the point is in M             */
    int64_t* slab_base;            /* [n_slabs]     storage position of the slab's first lane          */
    int32_t* wi_tile;              /* [n_work]      work items: tile,                                  */
    int32_t* wi_z0;                /* [n_work]        first plane,                                     */
    int32_t* wi_nz;                /* [n_work]        number of planes (<= zt)                         */
    int64_t* storage_to_canonical; /* [n_active]    canonical rank of the point in storage slot s     */
} gpe_layout_tables;

typedef struct {
    double kin;   /* h^3 sum Re(conj(psi) T psi),  T = -1/2 lap_h                                  */
    double pot;   /* h^3 sum V |psi|^2                                                              */
    double inter; /* h^3 (g/2) sum |psi|^4                                                          */
    double total; /* kin + pot + inter                                                              */
    double mu;    /* h^3 sum Re(conj(psi) H psi) / norm = (kin + pot + 2 inter) / norm  (Eq. 1)     */
    double norm;  /* h^3 sum |psi|^2  (Eq. 3)                                                       */
} gpe_energy_out;

/* ---- error text ------------------------------------------------------------------------------------ */
const char* gpe_last_error(void);

/* ---- a1: active-set layout builder (HOST ONLY: no CUDA call is made) ---------------------------------
 * PAPER.md:50-58 (ROI from the Thomas-Fermi density: V < cutoff), :81-85 (block post-selection, index
 * tables).  Evaluates the mask in the fixed floating-point order of DESIGN.md R2 (no FMA), strict '<',
 * and builds the tables above.  halo_width (0..8) only defines the ghost ring reported by
 * gpe_grid_stored_indices (R3); the ring is never stored on the device because every read
 * outside M is zero.  A sim needs halo_width >= stencil radius.  Errors: INVALID_ARG (null pointer,
 * n < 1, h <= 0, unknown kind/mode, box with more than 2^62 points), OUT_OF_MEMORY.  An empty mask is
 * valid (n_active = 0). */
int gpe_grid_create(const gpe_box* box, const gpe_potential* pot, double v_cut, int halo_width,
                    gpe_grid** out);

/* Same tables from an explicit active set: host array of n strictly ascending linear indices inside the
 * box (edge-case masks: random, single point, full box).  pot is still used for V(r,t). */
int gpe_grid_create_from_indices(const gpe_box* box, const gpe_potential* pot, const int64_t* active_host,
                                 int64_t n, int halo_width, gpe_grid** out);

/* Frees host tables and, if uploaded, device tables.  Sims created on the grid must be destroyed first.
 * NULL is a no-op. */
int gpe_grid_destroy(gpe_grid* g);

int gpe_grid_num_active(const gpe_grid* g, int64_t* out);
/* |S|, S = M u star-halo(M, halo_width) clipped to the box; computed on first use, O(|M| halo_width). */
int gpe_grid_num_stored(gpe_grid* g, int64_t* out);
int gpe_grid_layout_info(const gpe_grid* g, gpe_layout_info* out);
/* out_host: n_active int64, ascending L over M */
int gpe_grid_active_indices(const gpe_grid* g, int64_t* out_host);
/* out_host: gpe_grid_num_stored() int64, ascending L over S */
int gpe_grid_stored_indices(gpe_grid* g, int64_t* out_host);
int gpe_grid_layout_tables(const gpe_grid* g, const gpe_layout_tables* out_host);

/* ---- simulation object ------------------------------------------------------------------------------
 * Bytes of caller-owned device memory a sim needs: four state buffers in storage order (y0 / y2,y4 / y3 /
 * p of PAPER.md:276-281 Eq. A6-A7 specialised to RK4), one canonical staging buffer, reduction scratch. */
int gpe_sim_state_bytes(const gpe_grid* g, int dtype, size_t* out);

/* stencil: 7 (2nd order, PAPER.md:58, :337-339 Eq. B1), 13 (4th-order star, R5) or 19 (the paper's
 * higher-order compact Laplacian for dx = dy = dz = h, PAPER.md:341-343 Eq. B2: centre -4/h^2, faces 1/3h^2,
 * edges 1/6h^2; radius 1 plus the twelve edge neighbours, zero outside M like every other read), or 27 (3x3x3
 * compact stencil with caller-supplied weights, gpe_sim_set_compact_weights).
 * g: interaction strength multiplying |psi|^2; n_target: value of h^3 sum|psi|^2 that imaginary-time
 * steps renormalise to (Eq. 3).  dev_state: memory of the current device (cudaMalloc / a framework
 * allocator) or managed memory (cudaMallocManaged), 256-byte aligned, >= state_bytes, checked before anything is
 * allocated (INVALID_ARG);
 * must stay valid until gpe_sim_destroy; it is zero-initialised here (psi = 0, t = 0).  Uploads the
 * grid's tables to the current CUDA device on first use.  Errors: INVALID_ARG, UNSUPPORTED (tile shape
 * other than 8x8, halo_width < radius), CUDA (no device, not sm_100), OUT_OF_MEMORY. */
int gpe_sim_create(gpe_grid* g, int dtype, int stencil, double g_int, double n_target, void* dev_state,
                   size_t state_bytes, void* stream, gpe_sim** out);
int gpe_sim_destroy(gpe_sim* s);

/* a7: canonical <-> storage order.  dev_psi: n_active complex values of the sim's dtype on the device. */
int gpe_set_psi(gpe_sim* s, const void* dev_psi_canonical, void* stream);
int gpe_get_psi(gpe_sim* s, void* dev_psi_canonical, void* stream);
/* Same with HOST buffers: host->device copy + pack, unpack + device->host copy; synchronise `stream`. */
int gpe_set_psi_host(gpe_sim* s, const void* host_psi_canonical, void* stream);
int gpe_get_psi_host(gpe_sim* s, void* host_psi_canonical, void* stream);

int gpe_set_time(gpe_sim* s, double t);
int gpe_get_time(const gpe_sim* s, double* t);

/* a2+a3: dev_out = H[dev_in; t] dev_in, both canonical, n_active values, must not overlap.  Uses the
 * sim's g and stencil; does not touch the sim's own psi or clock.  (PAPER.md:27 Eq. 2, :58.) */
int gpe_apply_H(gpe_sim* s, double t, const void* dev_in_canonical, void* dev_out_canonical, void* stream);

/* a4: one / nsteps classic RK4 steps of i dpsi/dt = H psi (PAPER.md:71 Eq. 8, :91 Eq. 9) as four fused
 * stage kernels in the stage-state form (Eq. A6-A7, A10-A11).  V is evaluated at the stage times
 * t, t+dt/2, t+dt/2, t+dt.  Step n of a run starts at t_start + n*dt (a product, not a running sum); the
 * sim clock ends at t_start + nsteps*dt.  Asynchronous on `stream`.  Runs of 16 or more steps on grids below 4e6
 * points whose potential does not change during the run are replayed from a CUDA graph of 8 steps that the library
 * captures on a stream of its own (same kernels, parameters and order: bit-identical results;
 * gpe_sim_set_option(GPE_OPT_RK4_GRAPH, 0) turns it off, GPE_OPT_PDL = 0 turns off programmatic dependent launch of
 * the stage kernels).  If `stream` is itself being captured the library opens no capture of its own and the steps are
 * enqueued one by one. */
int gpe_step_rk4(gpe_sim* s, double dt, void* stream);
int gpe_run_rk4(gpe_sim* s, double dt, int64_t nsteps, void* stream);

/* The paper's cheaper integrator: Heun's third-order method "RKHE3" in the
 * stage-state form of Eq. A6-A7 with a* = [[1,0],[1,0]], b* = [1/4, 3/4, 0] (PAPER.md:286-290 Eq. A8-A9): three
 * fused stage kernels per step, y2 = y0 + dt/3 f(t, y0); y3 = y0 + 2dt/3 f(t + dt/3, y2) and p = y0/4 + 3 y2/4;
 * y_new = p + 3dt/4 f(t + 2dt/3, y3).  9 complex values per point and step (RK4: 12).  Clock as gpe_run_rk4. */
int gpe_step_rkhe3(gpe_sim* s, double dt, void* stream);
int gpe_run_rkhe3(gpe_sim* s, double dt, int64_t nsteps, void* stream);

/* The Cash-Karp method "RKCK", fifth-order solution, in the stage-state form of Eq. A6-A7 with the
 * modified tableau of PAPER.md:321-329 Eq. A12-A13 (two entries of the last row of a* are garbled in the
 * extracted text; 253/12288 and 1375/1536 follow from Eq. A4-A7 and are used): six fused stage kernels per
 * step, stage i reading the stencil operand y^(i) and, at the point itself, the earlier stage states
 * y^(1..i-1).  Needs six stage states: the four of the caller's state block plus two that the library
 * allocates on first use (n_active complex values each, freed by gpe_sim_destroy; OUT_OF_MEMORY if that
 * fails).  No step-size control (the embedded fourth-order solution is not formed).  Clock as gpe_run_rk4. */
int gpe_step_rkck(gpe_sim* s, double dt, void* stream);
int gpe_run_rkck(gpe_sim* s, double dt, int64_t nsteps, void* stream);

/* a5: psi' = psi - dt H[psi] psi, psi <- psi' sqrt(n_target / (h^3 sum|psi'|^2)) with V frozen at the sim
 * clock (PAPER.md:35, :60 Eq. 6, :87; forward-Euler reading DESIGN.md R7).  One fused kernel per step
 * (update + block partial sums) + a one-block finalise; the scale is applied lazily at the next load as
 * in the paper's kernel K1 and flushed at the end of the call, so the state seen by every
 * other call is normalised.
 * Degenerate states.  If the particle number becomes zero or non-finite during a run, no renormalisation is applied
 * (the values stay as they are, no NaN is manufactured) and a flag is raised on the device.  The runs are asynchronous,
 * so the flag is reported later, once, as GPE_ERR_STATE, by the first of these calls that follows the run: gpe_norm,
 * gpe_energy, gpe_get_psi_host (after their synchronisation; the out-parameters of gpe_norm / gpe_energy are not
 * written, the host array of gpe_get_psi_host is), or gpe_run_imag / gpe_run_imag_split / their single-step forms
 * (checked on entry without waiting: if the earlier run has finished and raised the flag, the new run is not enqueued).
 * The Runge-Kutta calls, gpe_apply_H and the device-side gpe_get_psi never report it.  Replacing the state -- gpe_set_psi,
 * gpe_set_psi_host, gpe_remap_psi into the sim -- discards a flag that has not been reported yet: it belonged to the
 * state that is gone (enqueue the replacement on the stream of the run, or ordered after it). */
int gpe_imag_step(gpe_sim* s, double dt, void* stream);
int gpe_run_imag(gpe_sim* s, double dt, int64_t nsteps, void* stream);

/* Re-gridding between ramp stages ("the grid post-selection procedure is repeated, and the
 * wavefunction is remapped between the old and new grids").  dst's state becomes src's
 * state on the points the two active sets share and 0 on the points that are new; values on points that are
 * dropped are lost (the caller checks gpe_norm(dst) and picks the cutoff, e.g. the paper's 5 max(mu_i, mu_i+1)).
 * Both sims must have the same precision and grids post-selected from the same bounding box (nx, ny, nz, h,
 * center), else INVALID_ARG.  dst's clock is set to src's.  The index match is one merge pass on the host over
 * the two ascending index lists; the table is copied to the device and the values move there (unpack, gather, pack),
 * all enqueued on `stream`: the call does not wait for them.  Each destination sim keeps ONE device table and one
 * staging area for remaps into it, so remaps into the same dst (and other calls that use dst's staging: the *_host
 * copies, gpe_apply_H) must be issued on one stream or otherwise ordered; src's staging area is used too.  `stream`
 * must not be in capture (UNSUPPORTED: the table comes from pageable host memory).  The first remap into a sim
 * allocates the table (OUT_OF_MEMORY if that fails). */
int gpe_remap_psi(gpe_sim* src, gpe_sim* dst, void* stream);

/* a5 (second mode): the paper's own ground-state iteration, in its order (PAPER.md:60-67,
 * :87 kernels K1-K3, footnote [44] at :236), V frozen at the sim clock:
 *   psi <- psi exp(-V dt/2) (1 - g |psi|^2 dt/2)        Eq. 7 for dt/2, interaction factor linearised (:67)
 *   psi <- psi - (dt/2) T psi, twice                     kinetic propagation for dt "in two steps using the
 *                                                        forward Euler method"
 *   psi <- psi exp(-V dt/2) (1 - g |psi|^2 dt/2)        Eq. 7 once more
 *   psi <- psi sqrt(n_target / (h^3 sum |psi|^2))        renormalisation
 * Two stencil launches per iteration, as the paper's K1 / K2 (:87): K1 applies Eq. 7 and the lazily applied scale of
 * the previous iteration to every value while it is staged for the stencil (own and halo) and takes the first Euler
 * half step; K2 takes the second Euler half step, applies Eq. 7 and writes block partial sums; then a one-block
 * finalise.  exp(-V dt/2) is evaluated analytically per value (no propagator array is read).  gpe_sim_set_option(GPE_OPT_FUSED_K1,
 * 0) runs the bit-identical three-launch form (pointwise Eq. 7, Euler half step, Euler half
 * step + Eq. 7).  The scale is flushed at the end of the call.
 * With a GPE_R64 sim the state is real (:67).  Same arguments and errors as gpe_run_imag. */
int gpe_imag_split_step(gpe_sim* s, double dt, void* stream);
int gpe_run_imag_split(gpe_sim* s, double dt, int64_t nsteps, void* stream);

/* a6: reductions over the sim's psi; fp64 accumulation, fixed summation order (bit-reproducible).
 * Synchronise `stream`.  Energy terms use V at the sim clock. */
int gpe_norm(gpe_sim* s, double* out_host, void* stream);
int gpe_energy(gpe_sim* s, gpe_energy_out* out_host, void* stream);

/* a6 without any allocation: *dev_out = cell_volume * sum_{k<n} |dev_psi[k]|^2  (Eq. 3; the sum of the
 * paper's kernel K3), fp64 accumulation in a fixed order (the same array gives the same bits every time),
 * asynchronous on `stream`.  The order of the values does not matter to the sum, so canonical order, a sim's storage
 * order or any other arrangement of the wavefunction will do.
 *
 * Why it exists.  gpe_norm needs a gpe_sim, and a sim costs four cudaMalloc calls and one cudaMallocHost.  Some
 * callers cannot have that happen: a process whose framework allocator (torch's caching allocator, typically) already
 * holds almost all device memory for 1e8-point state blocks, where a raw cudaMalloc made by a library fails although
 * the framework still has room; a norm check placed between time steps while other streams are busy, where cudaMalloc /
 * cudaFree would wait for the whole device on every call; code that has only an array of values (a checkpoint reader,
 * a diagnostic thread) and no grid or sim.  This call makes no cudaMalloc, cudaFree, cudaMallocHost or other allocating
 * call, now or later, and creates no stream or event.  The block partial sums go to a fixed array compiled into the
 * library: every GPU that loads the library's kernels holds GPE_NORM_NOALLOC_SCRATCH_BYTES for it until the process
 * exits, whether this function is called or not.
 *
 * Arguments.  dev_psi: n values on the current CUDA device (device or managed memory; may be NULL when n = 0), aligned
 * to their size: interleaved complex128 (GPE_C128), interleaved complex64 (GPE_C64) or real doubles (GPE_R64).
 * cell_volume: h hy hz of the grid (finite, > 0).  dev_out: one double on the same device, caller-owned, written by the
 * last kernel; read it after synchronising `stream` (or from later work on `stream`).  n = 0 writes 0.
 *
 * Limits and rules.
 *   - n <= GPE_NORM_NOALLOC_MAX_VALUES (2^29 = 536 870 912: one scratch slot per 8192 values); a larger n returns
 *     GPE_ERR_UNSUPPORTED and launches nothing.  For complex states of up to 19 398 656 values the summation order is
 *     the one gpe_norm uses on the same array; above that gpe_norm caps its block count, and for GPE_R64 it sums pairs,
 *     so there the two agree to rounding only.
 *   - The first call on each device looks up the scratch array's address on that device (which can also be the moment
 *     the CUDA runtime loads the library's kernels there).  Make that first call during start-up, with the device
 *     current, before any stream capture begins; later calls on that device only launch two kernels.
 *   - All calls on one device share the scratch.  It needs no clearing (a call overwrites every slot it later reads),
 *     but two calls whose kernels can overlap on the GPU -- different streams without an ordering between them, or
 *     different host threads -- corrupt each other's sums.  Calls queued on one stream are safe.
 *   - The device that owns dev_psi and dev_out must be current; otherwise INVALID_ARG.
 * Errors: INVALID_ARG (null or misaligned pointer, pointer not on the current device, n < 0, unknown dtype, bad
 * cell_volume), UNSUPPORTED (n over the limit, device ordinal above 63), CUDA. */
#define GPE_NORM_NOALLOC_SCRATCH_BYTES 524288
#define GPE_NORM_NOALLOC_MAX_VALUES 536870912LL
int gpe_norm_noalloc(const void* dev_psi, int64_t n, int dtype, double cell_volume, double* dev_out, void* stream);

/* Number of kernels this sim has launched so far (bench.py's gpu_launches). */
int gpe_sim_kernel_launches(const gpe_sim* s, int64_t* out);
/* Name/duration of the stage kernels: enables CUDA-event timing of every RK4 stage launch inside
 * gpe_run_rk4 on the launching stream (bench.py's roofline leg); on=0 disables.  gpe_sim_stage_time_ms
 * returns the accumulated milliseconds and launch count per stage index 0..3 and resets them. */
int gpe_sim_time_stages(gpe_sim* s, int on);
int gpe_sim_stage_time_ms(gpe_sim* s, double ms_out[4], int64_t count_out[4]);
/* The 27-point compact stencil (stencil = 27 at gpe_sim_create).  The paper's GPU results use a higher-order
 * compact stencil "of shape 3^3" but do not print its weights (they are in its ref.
 * [52]), so the caller supplies them: Laplacian weights in 1/length^2 of the centre, of the two face neighbours
 * per axis (x, y, z), of the four edge neighbours per plane (xy, xz, yz) and of the eight corners; T = -1/2 of
 * that stencil, zero outside M like every other read.  Until this is called a stencil-27 sim uses the weights of
 * Eq. B2 (corner 0), i.e. it equals stencil 19.  Also valid on a stencil-19 sim.  STATE for the star stencils. */
int gpe_sim_set_compact_weights(gpe_sim* s, double centre, const double* face_xyz, const double* edge_xy_xz_yz,
                                double corner);

/* Switches between forms of the same computation that give bit-identical results (tested); value 0 or 1, all default
 * to 1; a sim-level setting, read by every later call on the sim.  The library reads no environment variable.
 *   GPE_OPT_FUSED_K1   gpe_run_imag_split: 1 = the paper's K1 / K2 pair (two stencil launches per iteration),
 *                      0 = three launches (pointwise Eq. 7, Euler half step, Euler half step + Eq. 7).
 *   GPE_OPT_RK4_GRAPH  gpe_run_rk4: 1 = long runs on small grids in a static potential replay a captured CUDA graph,
 *                      0 = every step is enqueued launch by launch.
 *   GPE_OPT_PDL        1 = the stage kernels are launched with programmatic dependent launch (the next launch's
 *                      prologue overlaps the tail of the previous one), 0 = plain stream-ordered launches.  Changing it
 *                      drops the captured RK4 graph (waits for the device first).
 * Errors: INVALID_ARG (null sim, unknown option, value other than 0 / 1). */
#define GPE_OPT_FUSED_K1 0
#define GPE_OPT_RK4_GRAPH 1
#define GPE_OPT_PDL 2
int gpe_sim_set_option(gpe_sim* s, int option, int value);

/* Tuning knob: planes per thread block (1..32, default chosen per dtype/stencil).  INVALID_ARG otherwise. */
int gpe_sim_set_planes_per_block(gpe_sim* s, int kz);

#ifdef __cplusplus
}
#endif
#endif /* GPE_H_ */
