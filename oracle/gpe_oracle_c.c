/* CPU oracle, explicit-loop C version.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this.  It shares no code with the CUDA product.  complex128 throughout.
 *
 * Same definitions as oracle/gpe_oracle.py (which is pinned to the paper and the mathematics in
 * tests/test_oracle_pins.py); tests/test_oracle_c.py checks this file against that one.
 *   - reduced operator: PAPER.md:58 (rows/columns outside the ROI deleted, psi = 0 there)
 *   - H psi = T psi + V psi + g|psi|^2 psi: PAPER.md:27 Eq. 2, :71 Eq. 8
 *   - textbook RK4 with k1..k4 (Eq. 9); NOT the memory-optimised form
 *   - imaginary time: forward Euler + renormalisation (Eq. 6; R7)
 * The active set is a sorted list of linear indices; neighbours are found by binary search.
 * OpenMP over points is used so the timed CPU baseline uses all host cores; nothing is blocked,
 * fused or reordered beyond the definition.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

typedef struct {
    int32_t nx, ny, nz;
    int32_t kind;               /* 0 harmonic, 1 dressed */
    double h, cx, cy, cz;
    double ax, ay, az;
    double delta0, delta1, t_ramp, omega;
    double hy, hz;              /* step sizes along y, z (App. B Eq. B1); the wrapper passes h when isotropic */
} orc_problem;

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* threads of the parallel loops below (the timed baseline reports a one-thread figure beside the all-core one:
 * the paper's CPU numbers are single-thread); n <= 0 restores the default */
void orc_set_num_threads(int n) {
#ifdef _OPENMP
    omp_set_num_threads(n > 0 ? n : omp_get_num_procs());
#else
    (void)n;
#endif
}

static int64_t find_sorted(const int64_t* a, int64_t n, int64_t key) {
    int64_t lo = 0, hi = n;
    while (lo < hi) {
        int64_t mid = lo + (hi - lo) / 2;
        if (a[mid] < key) lo = mid + 1; else hi = mid;
    }
    return (lo < n && a[lo] == key) ? lo : -1;
}

/* nbr[k*6R + axis*2R + j], j = 0..2R-1 <-> s = -R..-1, 1..R ; -1 = absent (psi = 0) */
void orc_build_neighbours(const orc_problem* p, const int64_t* active, int64_t n, int R, int64_t* nbr) {
    const int64_t dims[3] = {p->nx, p->ny, p->nz};
    const int64_t strides[3] = {(int64_t)p->ny * p->nz, p->nz, 1};
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < n; ++k) {
        int64_t L = active[k];
        int64_t c[3] = {L / strides[0], (L / p->nz) % p->ny, L % p->nz};
        for (int axis = 0; axis < 3; ++axis) {
            int j = 0;
            for (int s = -R; s <= R; ++s) {
                if (s == 0) continue;
                int64_t q = c[axis] + s;
                int64_t r = -1;
                if (q >= 0 && q < dims[axis]) r = find_sorted(active, n, L + s * strides[axis]);
                nbr[k * 6 * R + axis * 2 * R + j] = r;
                ++j;
            }
        }
    }
}

static double delta_of_t(const orc_problem* p, double t) {
    if (p->t_ramp <= 0.0) return p->delta0;
    double s = t / p->t_ramp;
    if (s < 0.0) s = 0.0;
    if (s > 1.0) s = 1.0;
    return p->delta0 + (p->delta1 - p->delta0) * s;
}

static double potential(const orc_problem* p, int64_t L, double delta) {
    int64_t ix = L / ((int64_t)p->ny * p->nz), iy = (L / p->nz) % p->ny, iz = L % p->nz;
    double x = ((double)ix - 0.5 * (p->nx - 1)) * p->h + p->cx;
    double y = ((double)iy - 0.5 * (p->ny - 1)) * p->hy + p->cy;
    double z = ((double)iz - 0.5 * (p->nz - 1)) * p->hz + p->cz;
    double s = p->ax * (x * x) + p->ay * (y * y) + p->az * (z * z);
    double u = 0.5 * s;
    if (p->kind == 0) return u;
    double d = u - delta;
    return sqrt(d * d + p->omega * p->omega) - p->omega;
}

/* out = H[psi; t] psi */
void orc_apply_H(const orc_problem* p, const int64_t* active, const int64_t* nbr, int64_t n, int R,
                 double g, double t, const cplx* psi, cplx* out) {
    const double w7[2] = {-2.0, 1.0};
    const double w13[3] = {-5.0 / 2.0, 4.0 / 3.0, -1.0 / 12.0};
    const double* w = (R == 1) ? w7 : w13;
    const double delta = delta_of_t(p, t);
    const double inv[3] = {1.0 / (p->h * p->h), 1.0 / (p->hy * p->hy), 1.0 / (p->hz * p->hz)};   /* Eq. B1: 1/d_i^2 */
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < n; ++k) {
        cplx lap = 0.0;
        for (int axis = 0; axis < 3; ++axis) {
            cplx d2 = w[0] * psi[k];
            for (int s = 1; s <= R; ++s) {
                int64_t m = nbr[k * 6 * R + axis * 2 * R + (R - s)];       /* -s */
                int64_t q = nbr[k * 6 * R + axis * 2 * R + (R + s - 1)];   /* +s */
                cplx a = (m >= 0) ? psi[m] : 0.0;
                cplx b = (q >= 0) ? psi[q] : 0.0;
                d2 += w[s] * (a + b);
            }
            lap += inv[axis] * d2;
        }
        double v = potential(p, active[k], delta);
        double a2 = creal(psi[k]) * creal(psi[k]) + cimag(psi[k]) * cimag(psi[k]);
        out[k] = -0.5 * lap + (v + g * a2) * psi[k];
    }
}

/* textbook RK4, nsteps steps, step n starts at t0 + n dt; work holds 5 n complex values */
void orc_run_rk4(const orc_problem* p, const int64_t* active, const int64_t* nbr, int64_t n, int R,
                 double g, double t0, double dt, int64_t nsteps, cplx* psi, cplx* work) {
    cplx *k1 = work, *k2 = work + n, *k3 = work + 2 * n, *k4 = work + 3 * n, *y = work + 4 * n;
    for (int64_t s = 0; s < nsteps; ++s) {
        double t = t0 + (double)s * dt;
        orc_apply_H(p, active, nbr, n, R, g, t, psi, k1);
#pragma omp parallel for schedule(static)
        for (int64_t k = 0; k < n; ++k) { k1[k] = -I * k1[k]; y[k] = psi[k] + (0.5 * dt) * k1[k]; }
        orc_apply_H(p, active, nbr, n, R, g, t + 0.5 * dt, y, k2);
#pragma omp parallel for schedule(static)
        for (int64_t k = 0; k < n; ++k) { k2[k] = -I * k2[k]; y[k] = psi[k] + (0.5 * dt) * k2[k]; }
        orc_apply_H(p, active, nbr, n, R, g, t + 0.5 * dt, y, k3);
#pragma omp parallel for schedule(static)
        for (int64_t k = 0; k < n; ++k) { k3[k] = -I * k3[k]; y[k] = psi[k] + dt * k3[k]; }
        orc_apply_H(p, active, nbr, n, R, g, t + dt, y, k4);
#pragma omp parallel for schedule(static)
        for (int64_t k = 0; k < n; ++k) {
            k4[k] = -I * k4[k];
            psi[k] = psi[k] + (dt / 6.0) * (k1[k] + 2.0 * k2[k] + 2.0 * k3[k] + k4[k]);
        }
    }
}

static double norm_sum(int64_t n, const cplx* psi) {
    long double acc = 0.0L;
#pragma omp parallel for schedule(static) reduction(+ : acc)
    for (int64_t k = 0; k < n; ++k)
        acc += (long double)(creal(psi[k]) * creal(psi[k]) + cimag(psi[k]) * cimag(psi[k]));
    return (double)acc;
}

double orc_norm(const orc_problem* p, int64_t n, const cplx* psi) {
    return p->h * p->hy * p->hz * norm_sum(n, psi);
}

/* nsteps normalised forward-Euler imaginary-time steps, V frozen at time t; work holds n values */
void orc_run_imag(const orc_problem* p, const int64_t* active, const int64_t* nbr, int64_t n, int R,
                  double g, double t, double dt, int64_t nsteps, double n_target, cplx* psi, cplx* work) {
    for (int64_t s = 0; s < nsteps; ++s) {
        orc_apply_H(p, active, nbr, n, R, g, t, psi, work);
#pragma omp parallel for schedule(static)
        for (int64_t k = 0; k < n; ++k) work[k] = psi[k] - dt * work[k];
        double sc = sqrt(n_target / orc_norm(p, n, work));
#pragma omp parallel for schedule(static)
        for (int64_t k = 0; k < n; ++k) psi[k] = work[k] * sc;
    }
}

/* out[0..5] = kin, pot, inter, total, mu, norm ; work holds n values */
void orc_energy(const orc_problem* p, const int64_t* active, const int64_t* nbr, int64_t n, int R,
                double g, double t, const cplx* psi, cplx* work, double* out) {
    const double delta = delta_of_t(p, t);
    /* T psi = H psi with V = 0, g = 0 : compute through the same loop with a zeroed problem */
    orc_problem q = *p;
    q.kind = 0; q.ax = q.ay = q.az = 0.0;
    orc_apply_H(&q, active, nbr, n, R, 0.0, t, psi, work);
    long double kin = 0.0L, po = 0.0L, in4 = 0.0L, nn = 0.0L;
#pragma omp parallel for schedule(static) reduction(+ : kin, po, in4, nn)
    for (int64_t k = 0; k < n; ++k) {
        double a2 = creal(psi[k]) * creal(psi[k]) + cimag(psi[k]) * cimag(psi[k]);
        kin += (long double)creal(conj(psi[k]) * work[k]);
        po += (long double)(potential(p, active[k], delta) * a2);
        in4 += (long double)(a2 * a2);
        nn += (long double)a2;
    }
    double h3 = p->h * p->hy * p->hz;
    out[0] = h3 * (double)kin;
    out[1] = h3 * (double)po;
    out[2] = h3 * 0.5 * g * (double)in4;
    out[3] = out[0] + out[1] + out[2];
    out[5] = h3 * (double)nn;
    out[4] = (out[0] + out[1] + 2.0 * out[2]) / out[5];
}
