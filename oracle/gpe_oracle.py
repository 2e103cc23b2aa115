"""CPU oracle for the sparse-grid Gross-Pitaevskii hot path.  TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this.  It shares no code with the CUDA
product (``paper_2603_05447_b200/``); it never imports it.  complex128 / float64
throughout.  Every function cites the passage of /root/reference/PAPER.md it
follows (``PAPER.md:line``) or the reading in DESIGN.md ("R#") where the paper is
silent.

What the method computes (Eq. 1-3, 58, 71 Eq. 8): the finite-
difference operator  H psi = -1/2 lap_h psi + V psi + g |psi|^2 psi  restricted to
the region of interest (rows/columns outside it deleted, i.e. psi = 0 there),
fused into RK4 (real time) and normalised imaginary-time steps.  The sparse
layout, tiles and the memory-optimised Runge-Kutta form (App. A)
change where values live, not what is computed, so this oracle is the plain
definition: a sorted list of active points, neighbour look-up by linear index,
textbook k1..k4 RK4.

Pin status (tests/test_oracle_pins.py): coords/potential/mask, apply_T (7 and
13 pt), apply_H, rk4_step, norm/energy, layout tables: PINNED (P1-P12).
imag_step and energy()['mu'] for g > 0: PINNED (P20: a fixed point of the normalised Euler iteration satisfies
H[psi] psi = mu psi, Eq. 1, for any dt; P21: mu is the Rayleigh quotient of apply_H on a random state; P22:
Thomas-Fermi limit, Eq. 5, for large g).  Long nonlinear dynamics beyond the invariants (norm, energy, monotone
energy in imaginary time): "parity unpinned" (no closed form).
imag_split_step (the paper's own scheme): PINNED for g = 0 (P13: the
iteration matrix D K D built from Kronecker products, its top eigenvector and the
O(dt^2) splitting error of the ground-state energy), for the linearised interaction
factor, and for g > 0 to first order in dt (P23: it differs from the pinned Euler step by O(dt^2) only).
rkhe3_step / rkck_step (P15, P16), apply_T19 and anisotropic spacing (P17, P18), remap_psi (P14): PINNED.
apply_T27 / Compact27: the mechanism is PINNED (P19); for any particular published 27-point weight set
"parity unpinned" (PAPER.md does not print the weights of its 27-point stencil).
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

HARMONIC = 0
DRESSED = 1
MASK_AT_DELTA0 = 0
MASK_AT_DELTA1 = 1
MASK_UNION = 2

# Central-difference weights c_|s| of d^2/dx^2 * h^2 (R5):
# 7-point: 2nd order (App. B Eq. B1 at :337-339: [1,-2,1]/d^2).
# 13-point: standard 4th-order central weights (named by BASELINE.json; not in the paper).
STENCIL_WEIGHTS = {7: (-2.0, 1.0), 13: (-5.0 / 2.0, 4.0 / 3.0, -1.0 / 12.0)}


@dataclass
class Box:
    nx: int
    ny: int
    nz: int
    h: float
    center: tuple = (0.0, 0.0, 0.0)
    hy: float = 0.0          # step sizes along y and z; <= 0 means "same as h" (App. B:
    hz: float = 0.0          # anisotropic grids d_x != d_y != d_z)

    @property
    def spacing(self):
        return (self.h, self.hy if self.hy > 0 else self.h, self.hz if self.hz > 0 else self.h)

    @property
    def cell(self):
        """Volume element d_x d_y d_z of the sums that stand for integrals (Eq. 3)."""
        d = self.spacing
        return d[0] * d[1] * d[2]


@dataclass
class Potential:
    kind: int = HARMONIC
    ax: float = 1.0
    ay: float = 1.0
    az: float = 1.0
    delta0: float = 0.0
    delta1: float = 0.0
    t_ramp: float = 0.0
    omega: float = 0.0


# --------------------------------------------------------------------------
# coordinates, potential, mask
# --------------------------------------------------------------------------

def coords(n: int, h: float, c: float = 0.0) -> np.ndarray:
    """x_i = (i - (n-1)/2) h + c  ("centred at 0", R1)."""
    return (np.arange(n, dtype=np.float64) - 0.5 * (n - 1)) * h + c


def delta_of_t(pot: Potential, t: float) -> float:
    """Linear detuning ramp (BASELINE configs[2]; R16): static if t_ramp <= 0."""
    if pot.t_ramp <= 0.0:
        return pot.delta0
    s = min(max(t / pot.t_ramp, 0.0), 1.0)
    return pot.delta0 + (pot.delta1 - pot.delta0) * s


def quad_form(pot: Potential, x, y, z):
    """u = 1/2 (ax x^2 + ay y^2 + az z^2), fixed evaluation order (R2)."""
    s = pot.ax * (x * x) + pot.ay * (y * y) + pot.az * (z * z)
    return 0.5 * s


def potential_from_u(pot: Potential, u, delta):
    """V: harmonic V = u; dressed V = sqrt((u-delta)^2 + Omega^2) - Omega.

    Dressed form: BASELINE.json configs; physical origin PAPER.md:139 Eq. 10.
    """
    if pot.kind == HARMONIC:
        return u
    d = u - delta
    return np.sqrt(d * d + pot.omega * pot.omega) - pot.omega


def mask_potential_plane(box: Box, pot: Potential, mask_mode: int, ix: int) -> np.ndarray:
    """V_mask on the (ny, nz) plane ix (R13 for the UNION closed form)."""
    x = coords(box.nx, box.h, box.center[0])[ix]
    y = coords(box.ny, box.spacing[1], box.center[1])[:, None]
    z = coords(box.nz, box.spacing[2], box.center[2])[None, :]
    u = quad_form(pot, x, y, z)
    if pot.kind == HARMONIC:
        return u
    if mask_mode == MASK_AT_DELTA0:
        dl = pot.delta0
    elif mask_mode == MASK_AT_DELTA1:
        dl = pot.delta1
    else:
        lo, hi = min(pot.delta0, pot.delta1), max(pot.delta0, pot.delta1)
        dl = np.minimum(np.maximum(u, lo), hi)
    return potential_from_u(pot, u, dl)


def active_indices(box: Box, pot: Potential, v_cut: float, mask_mode: int = MASK_AT_DELTA0,
                   check_knife_edge: bool = False) -> np.ndarray:
    """M = {p : V_mask(r_p) < V_cut}, ascending linear index L = (ix*ny+iy)*nz+iz.

    PAPER.md:50-52 (Eq. 5): ROI = points where the Thomas-Fermi density
    max((mu - V)/g, 0) is nonzero, i.e. V < mu; mu is the cutoff V_cut.
    """
    out = []
    plane = box.ny * box.nz
    for ix in range(box.nx):
        v = mask_potential_plane(box, pot, mask_mode, ix)
        if check_knife_edge and math.isfinite(v_cut):
            assert np.min(np.abs(v - v_cut)) > 1e-9 * abs(v_cut), "point on the mask knife edge"
        idx = np.nonzero((v < v_cut).ravel())[0].astype(np.int64)
        out.append(idx + ix * plane)
    return np.concatenate(out) if out else np.zeros(0, np.int64)


def unravel(box: Box, lin: np.ndarray):
    iz = lin % box.nz
    iy = (lin // box.nz) % box.ny
    ix = lin // (box.nz * box.ny)
    return ix, iy, iz


def potential_at(box: Box, pot: Potential, lin: np.ndarray, t: float) -> np.ndarray:
    """V(r_p, t) on the given points (evaluated at the stage time, Eq. 9)."""
    ix, iy, iz = unravel(box, lin)
    x = coords(box.nx, box.h, box.center[0])[ix]
    y = coords(box.ny, box.spacing[1], box.center[1])[iy]
    z = coords(box.nz, box.spacing[2], box.center[2])[iz]
    u = quad_form(pot, x, y, z)
    return potential_from_u(pot, u, delta_of_t(pot, t))


# --------------------------------------------------------------------------
# the reduced operator
# --------------------------------------------------------------------------

class SparseGrid:
    """Sorted active set + neighbour table built by linear-index look-up.

    nbr[(axis, s)][k] = position in ``active`` of the point s steps along axis
    from active[k], or -1 if that point is outside the box or outside M (then it
    contributes psi = 0: PAPER.md:58, rows and columns outside the ROI deleted).
    """

    def __init__(self, box: Box, active: np.ndarray, radius: int):
        self.box = box
        self.active = np.asarray(active, dtype=np.int64)
        assert np.all(np.diff(self.active) > 0), "active indices must be strictly ascending"
        self.n = self.active.size
        self.radius = radius
        ix, iy, iz = unravel(box, self.active)
        dims = (box.nx, box.ny, box.nz)
        strides = (box.ny * box.nz, box.nz, 1)
        comp = (ix, iy, iz)
        self.nbr = {}
        for axis in range(3):
            for s in list(range(-radius, 0)) + list(range(1, radius + 1)):
                c = comp[axis] + s
                inside = (c >= 0) & (c < dims[axis])
                target = self.active + s * strides[axis]
                pos = np.searchsorted(self.active, target)
                pos_c = np.minimum(pos, max(self.n - 1, 0))
                hit = inside & (pos < self.n)
                if self.n:
                    hit &= self.active[pos_c] == target
                self.nbr[(axis, s)] = np.where(hit, pos_c, -1).astype(np.int64)


def neighbour_lookup(grid: SparseGrid, off) -> np.ndarray:
    """Position in ``active`` of the point at offset off = (dx, dy, dz) from every active point, -1 if that
    point is outside the box or outside M."""
    box = grid.box
    ix, iy, iz = unravel(box, grid.active)
    cx, cy, cz = ix + off[0], iy + off[1], iz + off[2]
    inside = (cx >= 0) & (cx < box.nx) & (cy >= 0) & (cy < box.ny) & (cz >= 0) & (cz < box.nz)
    target = (cx * box.ny + cy) * box.nz + cz
    pos = np.searchsorted(grid.active, target)
    pos_c = np.minimum(pos, max(grid.n - 1, 0))
    hit = inside & (pos < grid.n)
    if grid.n:
        hit &= grid.active[pos_c] == target
    return np.where(hit, pos_c, -1)


def apply_T19(grid: SparseGrid, psi: np.ndarray) -> np.ndarray:
    """T psi = -1/2 lap_19 psi with the 19-point higher-order compact Laplacian of PAPER.md:341-343 Eq. B2,
      lap_19 = lap_7 + 1/12 [ (dx^2+dy^2) dxx dyy + (dx^2+dz^2) dxx dzz + (dy^2+dz^2) dyy dzz ],  d_ii = [1,-2,1]/d_i^2,
    written out term by term as printed (products of second differences), psi = 0 outside M."""
    psi = np.asarray(psi, dtype=np.complex128)
    dsq = [d * d for d in grid.box.spacing]
    ext = np.concatenate([psi, np.zeros(1, np.complex128)])   # index -1 -> 0
    d2 = (1.0, -2.0, 1.0)

    def term(wx, wy, wz):
        """sum over offsets of wx[dx] wy[dy] wz[dz] psi(p + (dx,dy,dz)); w = False is the identity [0,1,0]."""
        out = np.zeros_like(psi)
        for dx in (-1, 0, 1):
            for dy in (-1, 0, 1):
                for dz in (-1, 0, 1):
                    c = 1.0
                    for axis, (wgt, d) in enumerate(((wx, dx), (wy, dy), (wz, dz))):
                        c *= (d2[d + 1] / dsq[axis]) if wgt else (1.0 if d == 0 else 0.0)
                    if c != 0.0:
                        out = out + c * ext[neighbour_lookup(grid, (dx, dy, dz))]
        return out

    lap7 = term(True, False, False) + term(False, True, False) + term(False, False, True)
    cross = ((dsq[0] + dsq[1]) * term(True, True, False) + (dsq[0] + dsq[2]) * term(True, False, True)
             + (dsq[1] + dsq[2]) * term(False, True, True))
    return -0.5 * (lap7 + (1.0 / 12.0) * cross)


@dataclass(frozen=True)
class Compact27:
    """A 3x3x3 compact Laplacian given by its weights (absolute, in 1/length^2): centre, the face weight per axis,
    the edge weight per pair (xy, xz, yz) and the corner weight.  The paper's GPU results use a 27-point
    higher-order compact stencil "of shape 3^3" whose weights it does not print (they
    are in its ref. [52]): PARITY UNPINNED for any particular published set; what is pinned is the mechanism,
    by its reductions to the 7- and 19-point stencils and by brute force (P19)."""
    centre: float
    face: tuple
    edge: tuple
    corner: float


def apply_T27(grid: SparseGrid, psi: np.ndarray, w: Compact27) -> np.ndarray:
    """T psi = -1/2 sum over the 27 offsets of weight(offset) psi(p + offset), psi = 0 outside M.
    weight: centre for (0,0,0); face[a] for +-e_a; edge[pair] for +-e_a +- e_b; corner for (+-1,+-1,+-1)."""
    psi = np.asarray(psi, dtype=np.complex128)
    ext = np.concatenate([psi, np.zeros(1, np.complex128)])
    lap = np.zeros_like(psi)
    pair = {(0, 1): 0, (0, 2): 1, (1, 2): 2}
    for dx in (-1, 0, 1):
        for dy in (-1, 0, 1):
            for dz in (-1, 0, 1):
                off = (dx, dy, dz)
                axes = tuple(a for a in range(3) if off[a] != 0)
                if len(axes) == 0:
                    c = w.centre
                elif len(axes) == 1:
                    c = w.face[axes[0]]
                elif len(axes) == 2:
                    c = w.edge[pair[axes]]
                else:
                    c = w.corner
                if c != 0.0:
                    lap = lap + c * ext[neighbour_lookup(grid, off)]
    return -0.5 * lap


def apply_T(grid: SparseGrid, psi: np.ndarray, stencil) -> np.ndarray:
    """T psi = -1/2 lap_h psi on M with psi = 0 outside M (weights R5).
    stencil may also be a Compact27 (caller-supplied 27-point weights, apply_T27).

    (lap_h psi)_p = (1/h^2) sum_axis sum_{s=-R..R} c_|s| psi(p + s e_axis).
    stencil = 19: the paper's higher-order compact Laplacian (apply_T19).
    """
    if isinstance(stencil, Compact27):
        return apply_T27(grid, psi, stencil)
    if stencil == 19:
        return apply_T19(grid, psi)
    w = STENCIL_WEIGHTS[stencil]
    R = len(w) - 1
    assert R <= grid.radius
    psi = np.asarray(psi, dtype=np.complex128)
    ext = np.concatenate([psi, np.zeros(1, np.complex128)])  # index -1 -> 0
    lap = np.zeros_like(psi)
    for axis in range(3):                                    # Eq. B1: each axis with its own step size d_i
        d = w[0] * psi
        for s in range(1, R + 1):
            d = d + w[s] * (ext[grid.nbr[(axis, -s)]] + ext[grid.nbr[(axis, s)]])
        lap = lap + d / (grid.box.spacing[axis] ** 2)
    return -0.5 * lap


def apply_H(grid: SparseGrid, pot: Potential, g: float, t: float, psi: np.ndarray,
            stencil: int) -> np.ndarray:
    """H[psi; t] psi = T psi + V(r, t) psi + g |psi|^2 psi  (PAPER.md:27 Eq. 2, :71 Eq. 8)."""
    v = potential_at(grid.box, pot, grid.active, t)
    return apply_T(grid, psi, stencil) + (v + g * (psi.real ** 2 + psi.imag ** 2)) * psi


def rk4_step(grid, pot, g, t, dt, psi, stencil):
    """Classic RK4 on d psi/dt = -i H psi (PAPER.md:71 Eq. 8, :91 Eq. 9, hbar = 1).

    Textbook k1..k4 form on purpose: the product uses the paper's memory-optimised
    form (PAPER.md:276-281 Eq. A6-A7, :315-319 Eq. A10-A11); this validates that algebra.
    """
    def f(tt, y):
        return -1j * apply_H(grid, pot, g, tt, y, stencil)
    k1 = f(t, psi)
    k2 = f(t + 0.5 * dt, psi + (0.5 * dt) * k1)
    k3 = f(t + 0.5 * dt, psi + (0.5 * dt) * k2)
    k4 = f(t + dt, psi + dt * k3)
    return psi + (dt / 6.0) * (k1 + 2.0 * k2 + 2.0 * k3 + k4)


def run_rk4(grid, pot, g, t0, dt, nsteps, psi, stencil):
    """nsteps RK4 steps; step n starts at t_n = t0 + n dt (a product, R16)."""
    for n in range(nsteps):
        psi = rk4_step(grid, pot, g, t0 + n * dt, dt, psi, stencil)
    return psi


def rkhe3_step(grid, pot, g, t, dt, psi, stencil):
    """Heun's third-order method ("RKHE3") on d psi/dt = -i H psi, textbook k form:
    c = (0, 1/3, 2/3), a21 = 1/3, a32 = 2/3, b = (1/4, 0, 3/4).  The product uses the paper's memory-optimised
    form (PAPER.md:286-290 Eq. A8-A9: a* = [[1,0],[1,0]], b* = [1/4, 3/4, 0])."""
    def f(tt, y):
        return -1j * apply_H(grid, pot, g, tt, y, stencil)
    k1 = f(t, psi)
    k2 = f(t + dt / 3.0, psi + (dt / 3.0) * k1)
    k3 = f(t + 2.0 * dt / 3.0, psi + (2.0 * dt / 3.0) * k2)
    return psi + dt * (0.25 * k1 + 0.75 * k3)


def run_rkhe3(grid, pot, g, t0, dt, nsteps, psi, stencil):
    for n in range(nsteps):
        psi = rkhe3_step(grid, pot, g, t0 + n * dt, dt, psi, stencil)
    return psi


# Cash-Karp tableau ("RKCK"; J. R. Cash and A. H. Karp 1990), fifth-order weights.
RKCK_C = (0.0, 1.0 / 5.0, 3.0 / 10.0, 3.0 / 5.0, 1.0, 7.0 / 8.0)
RKCK_A = ((),
          (1.0 / 5.0,),
          (3.0 / 40.0, 9.0 / 40.0),
          (3.0 / 10.0, -9.0 / 10.0, 6.0 / 5.0),
          (-11.0 / 54.0, 5.0 / 2.0, -70.0 / 27.0, 35.0 / 27.0),
          (1631.0 / 55296.0, 175.0 / 512.0, 575.0 / 13824.0, 44275.0 / 110592.0, 253.0 / 4096.0))
RKCK_B = (37.0 / 378.0, 0.0, 250.0 / 621.0, 125.0 / 594.0, 0.0, 512.0 / 1771.0)


def rkck_step(grid, pot, g, t, dt, psi, stencil):
    """One step of the Cash-Karp method (fifth-order solution) on d psi/dt = -i H psi, textbook k form
    (PAPER.md:248-252 Eq. A1: y^(i) = y0 + dt sum_{j<i} a_ij k_j).  The product uses the paper's memory-optimised
    form with a*, b* of PAPER.md:321-329 Eq. A12-A13."""
    def f(tt, y):
        return -1j * apply_H(grid, pot, g, tt, y, stencil)
    k = []
    for i in range(6):
        y = psi
        for j in range(i):
            y = y + (dt * RKCK_A[i][j]) * k[j]
        k.append(f(t + RKCK_C[i] * dt, y))
    out = psi
    for i in range(6):
        out = out + (dt * RKCK_B[i]) * k[i]
    return out


def run_rkck(grid, pot, g, t0, dt, nsteps, psi, stencil):
    for n in range(nsteps):
        psi = rkck_step(grid, pot, g, t0 + n * dt, dt, psi, stencil)
    return psi


def _sum(x) -> float:
    return float(np.sum(np.asarray(x, dtype=np.longdouble)))


def norm(grid: SparseGrid, psi) -> float:
    """h^3 sum |psi|^2  (Eq. 3)."""
    return grid.box.cell * _sum(psi.real ** 2 + psi.imag ** 2)


def imag_step(grid, pot, g, t, dt, psi, stencil, n_target=1.0):
    """psi' = psi - dt H[psi] psi, then psi <- psi' sqrt(N / (h^3 sum|psi'|^2)).

    PAPER.md:35 (imaginary time + renormalisation by Eq. 3), :60 Eq. 6; forward
    Euler reading of BASELINE's "normalised imaginary-time steps" (R7).
    V frozen at time t.
    """
    p = psi - dt * apply_H(grid, pot, g, t, psi, stencil)
    return p * math.sqrt(n_target / norm(grid, p))


def run_imag(grid, pot, g, t, dt, nsteps, psi, stencil, n_target=1.0):
    for _ in range(nsteps):
        psi = imag_step(grid, pot, g, t, dt, psi, stencil, n_target)
    return psi


def diag_propagator(grid, pot, g, t, dt, psi):
    """Eq. 7 for half a step with the interaction factor linearised as the paper does:
    psi -> psi * exp(-V dt/2) * (1 - g |psi|^2 dt/2)   ("the interaction propagator can be approximated as
    1 - g psi^2 dt / 2 hbar"; hbar = 1)."""
    v = potential_at(grid.box, pot, grid.active, t)
    return psi * np.exp(-0.5 * dt * v) * (1.0 - (0.5 * dt * g) * (psi.real ** 2 + psi.imag ** 2))


def imag_split_step(grid, pot, g, t, dt, psi, stencil, n_target=1.0):
    """One iteration of the paper's own ground-state scheme, in its order (PAPER.md:60-67, :87 kernels K1-K3):
    half a step of the diagonal operators (Eq. 7, linearised interaction), the kinetic propagation for a total
    time dt "in two steps using the forward Euler method" (two steps of dt/2 each, PAPER.md:67 and footnote
    [44] at :236), one more Eq. 7 half step, renormalisation to n_target.  V frozen at time t."""
    p = diag_propagator(grid, pot, g, t, dt, psi)
    p = p - (0.5 * dt) * apply_T(grid, p, stencil)
    p = p - (0.5 * dt) * apply_T(grid, p, stencil)
    p = diag_propagator(grid, pot, g, t, dt, p)
    return p * math.sqrt(n_target / norm(grid, p))


def run_imag_split(grid, pot, g, t, dt, nsteps, psi, stencil, n_target=1.0):
    for _ in range(nsteps):
        psi = imag_split_step(grid, pot, g, t, dt, psi, stencil, n_target)
    return psi


def remap_psi(active_old: np.ndarray, psi_old: np.ndarray, active_new: np.ndarray) -> np.ndarray:
    """Re-gridding between ramp stages ("the wavefunction is remapped between the old and new
    grids"): the value of a point that is in both active sets is kept, a point that is new starts at 0 (psi = 0
    outside the old region of interest), a point that is dropped is lost.  Explicit loop over a
    dictionary of the old points."""
    old = {int(L): k for k, L in enumerate(active_old)}
    out = np.zeros(len(active_new), dtype=np.complex128)
    for i, L in enumerate(active_new):
        k = old.get(int(L))
        if k is not None:
            out[i] = psi_old[k]
    return out


def energy(grid, pot, g, t, psi, stencil) -> dict:
    """Discrete GP functional with the same discrete Laplacian (R8).

    kin = h^3 sum Re(conj(psi) T psi); pot = h^3 sum V|psi|^2;
    inter = h^3 (g/2) sum |psi|^4; total = kin+pot+inter;
    mu = h^3 sum Re(conj(psi) H psi) / norm = (kin + pot + 2 inter)/norm (Eq. 1).
    """
    h3 = grid.box.cell
    tp = apply_T(grid, psi, stencil)
    v = potential_at(grid.box, pot, grid.active, t)
    a2 = psi.real ** 2 + psi.imag ** 2
    kin = h3 * _sum((np.conj(psi) * tp).real)
    po = h3 * _sum(v * a2)
    inter = h3 * 0.5 * g * _sum(a2 * a2)
    nrm = h3 * _sum(a2)
    return {"kin": kin, "pot": po, "inter": inter, "total": kin + po + inter,
            "mu": (kin + po + 2.0 * inter) / nrm, "norm": nrm}


# --------------------------------------------------------------------------
# dense second implementation (for pin P6 and small cross-checks)
# --------------------------------------------------------------------------

def dense_apply_T(box: Box, mask: np.ndarray, psi_dense: np.ndarray, stencil: int) -> np.ndarray:
    """Shifted-slice stencil on a dense (nx,ny,nz) array, zero outside mask and box."""
    w = STENCIL_WEIGHTS[stencil]
    R = len(w) - 1
    p = np.where(mask, psi_dense, 0.0).astype(np.complex128)
    lap = np.zeros_like(p)
    for axis in range(3):
        inv = 1.0 / box.spacing[axis] ** 2
        lap += (w[0] * inv) * p
        for s in range(1, R + 1):
            for sg in (-s, s):
                sh = np.zeros_like(p)
                src = [slice(None)] * 3
                dst = [slice(None)] * 3
                if sg > 0:
                    src[axis] = slice(sg, None)
                    dst[axis] = slice(None, -sg)
                else:
                    src[axis] = slice(None, sg)
                    dst[axis] = slice(-sg, None)
                sh[tuple(dst)] = p[tuple(src)]
                lap += (w[s] * inv) * sh
    return np.where(mask, -0.5 * lap, 0.0)


# --------------------------------------------------------------------------
# layout tables (independent Python builder)
# --------------------------------------------------------------------------

def stored_indices(box: Box, active: np.ndarray, halo_width: int) -> np.ndarray:
    """S = M u star-halo: points of the box within halo_width steps ALONG ONE AXIS
    of a point of M ("halo"; R3/R4: clipped to the box)."""
    ix, iy, iz = unravel(box, active)
    dims = (box.nx, box.ny, box.nz)
    strides = (box.ny * box.nz, box.nz, 1)
    comp = (ix, iy, iz)
    parts = [active]
    for axis in range(3):
        for s in range(1, halo_width + 1):
            for sg in (-s, s):
                c = comp[axis] + sg
                ok = (c >= 0) & (c < dims[axis])
                parts.append(active[ok] + sg * strides[axis])
    return np.unique(np.concatenate(parts))


def tile_layout(box: Box, active: np.ndarray, tx: int = 8, ty: int = 8, zt: int = 32) -> dict:
    """Column-tile / z-slab layout tables, built slowly and independently.

    Definitions:
      tile (i,j) = columns ix in [i*tx,(i+1)*tx), iy in [j*ty,(j+1)*ty); present iff it
        holds a point of M; listed by ascending i*nty+j (nty = ceil(ny/ty)).
      per tile: zlo = min iz, zhi = max iz + 1 over its points.
      slab (tile, z), zlo <= z < zhi: mask bit (lx*ty+ly) set iff the point is in M.
      storage order: tile ascending, z ascending, bit ascending; slab_base = storage
        position of the slab's first lane (also for empty slabs).
      tile_nbr: present-tile index of (i-1,j), (i+1,j), (i,j-1), (i,j+1), else -1.
      work items: per tile, maximal runs of consecutive non-empty slabs, a run of length
        l split into k = ceil(l/zt) pieces [z0+floor(i*l/k), z0+floor((i+1)*l/k)).
      storage_to_canonical[s] = rank in ascending-L order of the point at storage slot s.
    """
    assert tx * ty <= 64
    ix, iy, iz = unravel(box, active)
    nty = -(-box.ny // ty)
    tid = (ix // tx) * nty + (iy // ty)
    bit = (ix % tx) * ty + (iy % ty)
    # storage order = sort by (tile, z, bit)
    order = np.lexsort((bit, iz, tid))
    tid_s, iz_s, bit_s = tid[order], iz[order], bit[order]
    present = np.unique(tid_s)
    n_tiles = present.size
    tile_of = {int(t): k for k, t in enumerate(present)}
    tile_xy = np.stack([present // nty, present % nty], axis=1).astype(np.int32)
    tile_zlo = np.zeros(n_tiles, np.int32)
    tile_zhi = np.zeros(n_tiles, np.int32)
    tile_entry_base = np.zeros(n_tiles, np.int64)
    masks, bases = [], []
    wi_tile, wi_z0, wi_nz = [], [], []
    starts = np.searchsorted(tid_s, present, side="left")
    ends = np.searchsorted(tid_s, present, side="right")
    e = 0
    for k in range(n_tiles):
        a, b = int(starts[k]), int(ends[k])
        zs, bs = iz_s[a:b], bit_s[a:b]
        zlo, zhi = int(zs.min()), int(zs.max()) + 1
        tile_zlo[k], tile_zhi[k], tile_entry_base[k] = zlo, zhi, e
        m = np.zeros(zhi - zlo, np.uint64)
        np.bitwise_or.at(m, zs - zlo, np.uint64(1) << bs.astype(np.uint64))
        cnt = np.bincount(zs - zlo, minlength=zhi - zlo)
        base = a + np.concatenate([[0], np.cumsum(cnt)[:-1]])
        masks.append(m)
        bases.append(base.astype(np.int64))
        e += zhi - zlo
        # work items
        z = zlo
        while z < zhi:
            if cnt[z - zlo] == 0:
                z += 1
                continue
            z1 = z
            while z1 < zhi and cnt[z1 - zlo] > 0:
                z1 += 1
            l = z1 - z
            kk = -(-l // zt)
            for i in range(kk):
                s0 = z + (i * l) // kk
                s1 = z + ((i + 1) * l) // kk
                wi_tile.append(k)
                wi_z0.append(s0)
                wi_nz.append(s1 - s0)
            z = z1
    nbr = np.full((n_tiles, 4), -1, np.int32)
    ntx = -(-box.nx // tx)
    for k in range(n_tiles):
        i, j = int(tile_xy[k, 0]), int(tile_xy[k, 1])
        for q, (di, dj) in enumerate(((-1, 0), (1, 0), (0, -1), (0, 1))):
            ii, jj = i + di, j + dj
            if 0 <= ii < ntx and 0 <= jj < nty:
                nbr[k, q] = tile_of.get(ii * nty + jj, -1)
    return {
        "tx": tx, "ty": ty, "zt": zt, "n_tiles": n_tiles,
        "tile_xy": tile_xy, "tile_zlo": tile_zlo, "tile_zhi": tile_zhi,
        "tile_entry_base": tile_entry_base, "tile_nbr": nbr,
        "slab_mask": np.concatenate(masks) if masks else np.zeros(0, np.uint64),
        "slab_base": np.concatenate(bases) if bases else np.zeros(0, np.int64),
        "wi_tile": np.asarray(wi_tile, np.int32), "wi_z0": np.asarray(wi_z0, np.int32),
        "wi_nz": np.asarray(wi_nz, np.int32),
        "storage_to_canonical": order.astype(np.int64),
    }
