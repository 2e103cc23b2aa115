"""Seeded synthetic inputs for the sparse-grid Gross-Pitaevskii hot path.

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the
CUDA product (``paper_2603_05447_b200/``).  It holds workload descriptions
(plain numbers taken from BASELINE.json's ``configs``) and seeded initial-state
recipes.  It holds none of the method's arithmetic: no mask rule, no stencil,
no potential used by the operator, no stepper, no reduction.  The initial-state
recipes are *inputs*; they use their own closed-form envelopes (a Gaussian, a
parabolic shell profile) evaluated at the coordinates of a caller-supplied list
of active linear indices.

Stand-in statement: the paper measures on RF-dressed
atom-chip potentials of the Cold Atom Laboratory (ref. [46]) that
are not available here.  The analytic harmonic / dressed-shell workloads below,
from BASELINE.json, stand in for them; they have the paper's thin-shell geometry
(PAPER.md:13, 44, 56).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace

import numpy as np

HARMONIC = 0
DRESSED = 1

MASK_AT_DELTA0 = 0
MASK_AT_DELTA1 = 1
MASK_UNION = 2


@dataclass(frozen=True)
class Workload:
    """One synthetic workload: box, potential parameters, cutoff, solver knobs."""

    name: str
    nx: int
    ny: int
    nz: int
    h: float
    kind: int                 # HARMONIC or DRESSED
    ax: float = 1.0
    ay: float = 1.0
    az: float = 1.0
    delta0: float = 0.0
    delta1: float = 0.0
    t_ramp: float = 0.0       # <= 0: static potential at delta0
    omega: float = 0.0
    mask_mode: int = MASK_AT_DELTA0
    v_cut: float = math.inf
    halo_width: int = 2
    stencil: int = 7          # 7 or 13
    g: float = 0.0
    dt: float = 1e-3
    nsteps: int = 1
    dtype: str = "complex128"
    seed: int = 0
    psi0: str = "shell"       # gaussian | constant | shell | blob
    center: tuple = (0.0, 0.0, 0.0)
    note: str = ""
    hy: float = 0.0           # step sizes along y, z; <= 0: same as h (anisotropic grids, App. B)
    hz: float = 0.0

    @property
    def spacing(self):
        return (self.h, self.hy if self.hy > 0 else self.h, self.hz if self.hz > 0 else self.h)

    def with_(self, **kw) -> "Workload":
        return replace(self, **kw)


# --------------------------------------------------------------------------
# BASELINE.json configs (readings: SURVEY.md section 8c)
# --------------------------------------------------------------------------

def config1() -> Workload:
    return Workload(
        name="cfg1_harmonic_48", nx=48, ny=48, nz=48, h=0.25, kind=HARMONIC,
        v_cut=20.0, halo_width=2, stencil=7, g=100.0, dt=1e-3, nsteps=100,
        seed=1, psi0="gaussian",
        note="BASELINE configs[0]: isotropic harmonic trap, RK4")


def config2() -> Workload:
    return Workload(
        name="cfg2_bubble_256", nx=256, ny=256, nz=256, h=0.4, kind=DRESSED,
        delta0=800.0, delta1=800.0, omega=20.0, v_cut=60.0, halo_width=2,
        stencil=13, g=2000.0, dt=5e-4, nsteps=2000, seed=2, psi0="constant",
        note="BASELINE configs[1]: dressed bubble, imaginary time")


def config3(union: bool = True) -> Workload:
    return Workload(
        name="cfg3a_ramp_union_512" if union else "cfg3b_ramp_final_512",
        nx=512, ny=512, nz=512, h=0.2, kind=DRESSED, delta0=0.0, delta1=800.0,
        t_ramp=2e4 * 2e-4, omega=20.0, v_cut=60.0,
        mask_mode=MASK_UNION if union else MASK_AT_DELTA1, halo_width=2,
        stencil=7, g=2000.0, dt=2e-4, nsteps=20000, seed=3,
        psi0="blob" if union else "shell",
        note="BASELINE configs[2]: hollowing-out ramp, V evaluated per stage")


def config4(dtype: str = "complex128") -> Workload:
    return Workload(
        name="cfg4_ellipsoid_1024_" + ("c128" if dtype == "complex128" else "c64"),
        nx=1024, ny=1024, nz=1024, h=0.12, kind=DRESSED, ax=1.0, ay=2.25,
        az=4.0, delta0=2000.0, delta1=2000.0, omega=30.0, v_cut=80.0,
        halo_width=2, stencil=13, g=5000.0, dt=1e-4, nsteps=200, seed=4,
        psi0="shell", dtype=dtype,
        note="BASELINE configs[3]: anisotropic ellipsoidal bubble (largest shell)")


def config5_shell(n_target: float, thickness_pts: int = 24, stencil: int = 13,
                  dtype: str = "complex128", index: int = 0) -> Workload:
    """Bandwidth-sweep shell (SURVEY.md section 8d, config 5 recipe)."""
    h = 0.4
    t = thickness_pts * h
    r_pts = math.sqrt(n_target / (4.0 * math.pi * thickness_pts))
    r0 = r_pts * h
    delta = 0.5 * r0 * r0
    w = r0 * t / 2.0
    v_cut = min(60.0, w / 2.0)
    omega = (w * w - v_cut * v_cut) / (2.0 * v_cut)
    n = 64
    while n < 2048 and n / 2 < r_pts + thickness_pts / 2 + 2:
        n *= 2
    return Workload(
        name=f"cfg5_shell_{n_target:.0e}_T{thickness_pts}_{stencil}pt_"
             + ("c128" if dtype == "complex128" else "c64"),
        nx=n, ny=n, nz=n, h=h, kind=DRESSED, delta0=delta, delta1=delta,
        omega=omega, v_cut=v_cut, halo_width=2, stencil=stencil, g=2000.0,
        dt=1e-3, nsteps=50, seed=5000 + index, psi0="shell", dtype=dtype,
        note="BASELINE configs[4]: bandwidth sweep shell")


def config5_dense(n: int = 512, stencil: int = 13, dtype: str = "complex128") -> Workload:
    return Workload(
        name=f"cfg5_dense_{n}_{stencil}pt_" + ("c128" if dtype == "complex128" else "c64"),
        nx=n, ny=n, nz=n, h=0.05, kind=HARMONIC, v_cut=math.inf, halo_width=2,
        stencil=stencil, g=2000.0, dt=1e-4, nsteps=50, seed=5999, psi0="gaussian",
        dtype=dtype, note="BASELINE configs[4]: fully active dense box")


def small_shell(n: int = 40, stencil: int = 13, dtype: str = "complex128",
                seed: int = 11, aniso: bool = True) -> Workload:
    """A shell small enough for the oracle to finish in seconds.

    Same dressed form as configs 2-4, radius ~13 grid points, thickness ~8;
    spans several 8x8 column tiles and has ragged tails.
    """
    return Workload(
        name=f"small_shell_{n}_{stencil}pt", nx=n, ny=n + 3, nz=n + 5, h=0.5,
        kind=DRESSED, ax=1.0, ay=1.3 if aniso else 1.0, az=0.8 if aniso else 1.0,
        delta0=20.0, delta1=20.0, omega=6.0, v_cut=12.0, halo_width=2,
        stencil=stencil, g=300.0, dt=1e-3, nsteps=20, seed=seed, psi0="shell",
        dtype=dtype, note="test-size dressed shell")


# --------------------------------------------------------------------------
# Counter-based uniform numbers: value depends on (seed, L) only, not on layout
# --------------------------------------------------------------------------

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def uniform01(seed: int, lin: np.ndarray, stream: int = 0) -> np.ndarray:
    """splitmix64-style mix of (seed, stream, L) -> float64 in [0, 1).

    Top 53 bits times 2**-53.  Pure integer arithmetic, vectorised.
    """
    with np.errstate(over="ignore"):
        z = lin.astype(np.uint64)
        z = z + np.uint64((0x9E3779B97F4A7C15 * (2 * seed + 1) + 0xD1B54A32D192ED03 * stream)
                          & 0xFFFFFFFFFFFFFFFF)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
        z = (z + np.uint64(0x9E3779B97F4A7C15)) & _M64
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def _coords_of(w: Workload, lin: np.ndarray):
    iz = lin % w.nz
    iy = (lin // w.nz) % w.ny
    ix = lin // (w.nz * w.ny)
    x = (ix.astype(np.float64) - 0.5 * (w.nx - 1)) * w.h + w.center[0]
    y = (iy.astype(np.float64) - 0.5 * (w.ny - 1)) * w.spacing[1] + w.center[1]
    z = (iz.astype(np.float64) - 0.5 * (w.nz - 1)) * w.spacing[2] + w.center[2]
    return x, y, z


def make_psi0(w: Workload, active_idx: np.ndarray, n_target: float = 1.0) -> np.ndarray:
    """Seeded complex128 initial state on the given active points (canonical order).

    Recipes:
      gaussian : exp(-r^2/2) * exp(i*phi),  phi = 1e-3*(2u-1)
      constant : 1 on every active point
      shell    : sqrt(max(1-((q-delta1)/W)^2, 0)) + 0.05, q = (ax x^2+ay y^2+az z^2)/2,
                 W = 0.7*sqrt((v_cut+omega)^2-omega^2), times exp(i*phi_smooth + i*phi)
      blob     : sqrt(max(1 - q/30, 0)) + 0.02 (compact cloud at the centre), same phases
    Normalised so that h^3 * sum |psi|^2 = n_target.
    """
    lin = np.asarray(active_idx, dtype=np.int64)
    x, y, z = _coords_of(w, lin)
    u = uniform01(w.seed, lin)
    phi = 1e-3 * (2.0 * u - 1.0)
    if w.psi0 == "gaussian":
        amp = np.exp(-0.5 * (x * x + y * y + z * z))
    elif w.psi0 == "constant":
        amp = np.ones(lin.shape, dtype=np.float64)
        phi = np.zeros_like(phi)
    elif w.psi0 in ("shell", "blob"):
        q = 0.5 * (w.ax * x * x + w.ay * y * y + w.az * z * z)
        if w.psi0 == "shell":
            W = 0.7 * math.sqrt(max((w.v_cut + w.omega) ** 2 - w.omega ** 2, 1e-30))
            amp = np.sqrt(np.maximum(1.0 - ((q - w.delta1) / W) ** 2, 0.0)) + 0.05
        else:
            amp = np.sqrt(np.maximum(1.0 - q / 30.0, 0.0)) + 0.02
        # smooth seeded phase field: 16 plane waves
        rng = np.random.Generator(np.random.PCG64(w.seed))
        box = max(w.nx, w.ny, w.nz) * w.h
        kmin, kmax = 2.0 * math.pi / box, 2.0 * math.pi / (8.0 * w.h)
        ph = np.zeros_like(amp)
        for _ in range(16):
            kmag = kmin + (kmax - kmin) * rng.random()
            d = rng.normal(size=3)
            d /= np.linalg.norm(d)
            th = 2.0 * math.pi * rng.random()
            ph += np.cos(kmag * (d[0] * x + d[1] * y + d[2] * z) + th)
        phi = phi + 0.05 * ph / 4.0
    else:
        raise ValueError(w.psi0)
    psi = amp * np.exp(1j * phi)
    nrm = w.spacing[0] * w.spacing[1] * w.spacing[2] * float(np.sum(np.abs(psi) ** 2))
    psi *= math.sqrt(n_target / nrm)
    return psi.astype(np.complex128)


def random_psi(seed: int, n: int) -> np.ndarray:
    """Seeded complex128 vector with O(1) entries (for operator-level parity cases)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    return (rng.normal(size=n) + 1j * rng.normal(size=n)).astype(np.complex128)


def random_mask_lin(seed: int, nx: int, ny: int, nz: int, p: float) -> np.ndarray:
    """Seeded random subset of a box as ascending linear indices (edge-case masks)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    m = rng.random(nx * ny * nz) < p
    return np.nonzero(m)[0].astype(np.int64)
