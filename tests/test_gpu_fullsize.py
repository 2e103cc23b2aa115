"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (library-default planes
per stream), on SAMPLED outputs the oracle can compute one by one.

The CUDA path advances the whole grid.  The oracle (oracle/gpe_oracle_c.c, explicit loops, textbook k1..k4) is run
on the active points of a sample box B enlarged by the dependency margin m = 4 R K of K RK4 steps (4 operator
applications of star radius R per step): every point of B has its whole dependency cone inside B + m, so its
value after K steps does not depend on what the oracle assumes outside B + m (it assumes psi = 0 there).  The
comparison is made on the points of B only, in the DESIGN.md R10 norm max|a-b| / max|b| over those points.
Boxes sit where the layout is hardest: on the clipped tip of the shell at the box face (configs 1 and 4 touch
it), at a pole (short z runs, full slabs), on the equator (long z runs, partial slabs) and at a seeded random
active point.

Tolerances (north_star): 1e-12 per operator application in complex128, 1e-5 in complex64; K = 2 steps are 8
applications, so 1e-11 and 1e-4 are asked after the steps.  Config 2 (1.2e6 points) runs whole: 2000 normalised
imaginary-time steps against the C oracle at the 1000-step bound 1e-9."""
import numpy as np
import pytest

import gpe_inputs as I
from helpers import RADIUS, oracle_objs, rel_max
from oracle import c_oracle as CO

pytestmark = pytest.mark.gpu

K_STEPS = 2
HALF = 10          # sample box half-width in grid points (B is 21^3 cells)


@pytest.fixture(scope="module")
def P():
    import paper_2603_05447_b200 as P
    return P


def _ijk(w, lin):
    iz = lin % w.nz
    iy = (lin // w.nz) % w.ny
    ix = lin // (w.nz * w.ny)
    return ix, iy, iz


def _sample_centres(w, act, seed):
    """Active points at the extremes of the shell and one seeded random one."""
    ix, iy, iz = _ijk(w, act)
    picks = [int(np.argmax(ix)), int(np.argmin(ix)), int(np.argmax(iz)), int(np.argmax(iy)),
             int(np.random.Generator(np.random.PCG64(seed)).integers(0, act.size))]
    # equator: a point with iz closest to the mid-plane and the largest ix among those
    mid = np.nonzero(np.abs(iz - w.nz // 2) <= 1)[0]
    picks.append(int(mid[np.argmax(iy[mid])]))
    return [(int(ix[p]), int(iy[p]), int(iz[p])) for p in picks], (ix, iy, iz)


def _in_box(ijk, c, half):
    ix, iy, iz = ijk
    return ((np.abs(ix - c[0]) <= half) & (np.abs(iy - c[1]) <= half) & (np.abs(iz - c[2]) <= half))


class _NumpyOracle:
    """Same calls as c_oracle.COracle on the NumPy oracle (the C restatement has no 19-point stencil)."""

    def __init__(self, box, pot, active, stencil):
        from oracle import gpe_oracle as O
        self.O, self.pot, self.stencil = O, pot, stencil
        self.grid = O.SparseGrid(box, active, RADIUS[stencil])

    def apply_H(self, g, t, psi):
        return self.O.apply_H(self.grid, self.pot, g, t, psi, self.stencil)

    def run_rk4(self, g, t0, dt, nsteps, psi):
        return self.O.run_rk4(self.grid, self.pot, g, t0, dt, nsteps, psi, self.stencil)


_cache = {}


def _setup(P, w):
    """Grid, full psi0 and the sample geometry of a workload (cached per mask: c64 / c128 share it)."""
    key = (w.nx, w.ny, w.nz, w.h, w.kind, w.delta0, w.delta1, w.omega, w.v_cut, w.mask_mode, w.psi0, w.seed)
    if key not in _cache:
        _cache.clear()                                    # one full-size state at a time on the host
        grid = P.Grid.from_workload(w)
        act = grid.active_indices()
        psi0 = I.make_psi0(w, act)
        centres, ijk = _sample_centres(w, act, w.seed + 17)
        _cache[key] = (grid, act, psi0, centres, ijk)
    return _cache[key]


def _check_rk4_samples(P, w, t0, tol_apply, tol_steps):
    grid, act, psi0, centres, ijk = _setup(P, w)
    R = RADIUS[w.stencil]
    box, pot, _ = oracle_objs(w, active=act[:1])
    sim = P.Sim(grid, w.dtype, w.stencil, w.g)
    psi_in = psi0.astype(sim.npdtype)
    import torch
    d_in = torch.from_numpy(psi_in).to("cuda:0")
    h_gpu = sim.apply_H(t0, d_in).cpu().numpy()
    del d_in
    sim.set_psi_host(psi_in)
    sim.time = t0
    sim.run_rk4(w.dt, K_STEPS)
    got = sim.get_psi_host()
    assert np.all(np.isfinite(got.view(np.float32 if w.dtype == "complex64" else np.float64)))
    margin = 4 * R * K_STEPS
    checked = 0
    for c in centres:
        sub = np.nonzero(_in_box(ijk, c, HALF + margin))[0]
        inner = _in_box(tuple(a[sub] for a in ijk), c, HALF)
        co = _NumpyOracle(box, pot, act[sub], w.stencil) if w.stencil == 19 else CO.COracle(box, pot, act[sub], w.stencil)
        p_sub = psi_in[sub].astype(np.complex128)         # complex64: the oracle gets the fp32-rounded input
        # one operator application: exact for the points whose star lies inside the sub-box
        inner1 = _in_box(tuple(a[sub] for a in ijk), c, HALF + margin - R)
        ref_h = co.apply_H(w.g, t0, p_sub)
        assert rel_max(h_gpu[sub][inner1], ref_h[inner1]) < tol_apply, (w.name, c, "apply_H")
        ref = co.run_rk4(w.g, t0, w.dt, K_STEPS, p_sub)
        err = rel_max(got[sub][inner], ref[inner])
        assert err < tol_steps, (w.name, c, err)
        checked += int(inner.sum())
    assert checked > 1000
    # property that holds at any size: RK4 conserves the norm up to its local error, O(dt^5) per step (P8; for
    # the ramped potential of config 3 the constant also carries dV/dt, measured 3e-9 after two steps)
    assert abs(sim.norm() - 1.0) < (1e-7 if w.dtype == "complex128" else 1e-4)


@pytest.mark.parametrize("dtype", ["complex128", "complex64"])
def test_config4_sampled(P, dtype):
    """BASELINE configs[3]: 1024^3 ellipsoidal bubble, 13-point stencil, both precisions (shell tips clipped
    by the box face)."""
    w = I.config4(dtype)
    tol = (1e-12, 1e-11) if dtype == "complex128" else (1e-5, 1e-4)
    _check_rk4_samples(P, w, 0.0, *tol)


@pytest.mark.parametrize("union", [True, False])
def test_config3_sampled(P, union):
    """BASELINE configs[2]: 512^3 hollowing-out ramp, 7-point stencil, Delta(t) evaluated per stage; started in
    the middle of the ramp (t0 = 1) so that every stage sees a different potential."""
    _check_rk4_samples(P, I.config3(union), 1.0, 1e-12, 1e-11)


def test_config4_19pt_sampled(P):
    """The 1024^3 ellipsoidal bubble with the paper's 19-point higher-order compact stencil."""
    _check_rk4_samples(P, I.config4("complex128").with_(stencil=19), 0.0, 1e-12, 1e-11)


def test_config5_sweep_point_sampled(P):
    """BASELINE configs[4]: the 1e7-point shell of the bandwidth sweep (13-point, complex128)."""
    _check_rk4_samples(P, I.config5_shell(1e7, 24, 13, "complex128", 4), 0.0, 1e-12, 1e-11)


def test_config5_sweep_point_7pt_c64_sampled(P):
    _check_rk4_samples(P, I.config5_shell(3e6, 24, 7, "complex64", 3), 0.0, 1e-5, 1e-4)


@pytest.mark.parametrize("target,thickness,stencil,dtype,index", [
    (3e7, 24, 13, "complex128", 5), (3e7, 24, 7, "complex64", 5), (1e8, 24, 13, "complex128", 6),
    (1e7, 8, 13, "complex128", 4)], ids=["3e7_13pt_c128", "3e7_7pt_c64", "1e8_13pt_c128", "thin_T8_1e7_13pt_c128"])
def test_config5_large_and_thin_sweep_shells_sampled(P, target, thickness, stencil, dtype, index):
    """BASELINE configs[4] above 1e7 points (boxes 1024^3 and 2048^3: what `bench.py --sweep` times there) and the thin
    T = 8 shell of SURVEY.md 8d: the same sampled-box comparison as config 4.  The 3e8-point shell is not run here: its
    host-side input (indices, coordinates and the seeded state of 3e8 points in NumPy) needs about 25 GB and minutes."""
    tol = (1e-12, 1e-11) if dtype == "complex128" else (1e-5, 1e-4)
    w = I.config5_shell(target, thickness, stencil, dtype, index)
    _check_rk4_samples(P, w, 0.0, *tol)       # the two 3e7 cases share one grid and state through _setup's cache


def test_config5_dense_512_box_sampled(P):
    """The fully active 512^3 box that `bench.py --sweep` times (1.34e8 points, every slab full)."""
    _check_rk4_samples(P, I.config5_dense(512, 13, "complex128"), 0.0, 1e-12, 1e-11)
    _cache.clear()


def test_config5_dense_box_sampled(P):
    """BASELINE configs[4]: the fully active dense box (every slab full, box faces on all sides); 256^3 keeps
    the host-side input generation short, the 512^3 box is what bench.py times."""
    _check_rk4_samples(P, I.config5_dense(256, 13, "complex128"), 0.0, 1e-12, 1e-11)


def test_config2_full_imaginary_time(P):
    """BASELINE configs[1]: 256^3 dressed bubble, 13-point stencil, g = 2000, uniform-on-shell psi0, 2000
    normalised imaginary-time steps dt = 5e-4 -- the whole grid against the C oracle, state, norm, energy, mu."""
    w = I.config2()
    box, pot, act = oracle_objs(w)
    grid = P.Grid.from_workload(w)
    assert np.array_equal(grid.active_indices(), act)
    sim = P.Sim(grid, "complex128", w.stencil, w.g)
    co = CO.COracle(box, pot, act, w.stencil)
    psi = I.make_psi0(w, act)
    sim.set_psi_host(psi)
    ref = psi
    e_prev = None
    for nsteps in (100, 900, 1000):
        sim.run_imag(w.dt, nsteps)
        ref = co.run_imag(w.g, 0.0, w.dt, nsteps, ref)
        assert rel_max(sim.get_psi_host(), ref) < 1e-9
        e, eo = sim.energy(), co.energy(w.g, 0.0, ref)
        for k in ("kin", "pot", "inter", "total", "mu"):
            assert abs(e[k] - eo[k]) <= 1e-10 * max(1.0, abs(eo[k])), (k, e[k], eo[k])
        assert abs(sim.norm() - 1.0) < 1e-12
        if e_prev is not None:
            assert e["total"] < e_prev                    # imaginary time lowers the energy (invariant)
        e_prev = e["total"]


def test_config2_split_scheme_iterations(P):
    """BASELINE configs[1] with the paper's own iteration: 10 iterations on the whole grid
    against the NumPy oracle (imag_split_step)."""
    from oracle import gpe_oracle as O
    w = I.config2()
    box, pot, act = oracle_objs(w)
    grid = P.Grid.from_workload(w)
    sim = P.Sim(grid, "complex128", w.stencil, w.g)
    og = O.SparseGrid(box, act, RADIUS[w.stencil])
    psi = I.make_psi0(w, act)
    sim.set_psi_host(psi)
    sim.run_imag_split(w.dt, 10)
    ref = O.run_imag_split(og, pot, w.g, 0.0, w.dt, 10, psi, w.stencil)
    assert rel_max(sim.get_psi_host(), ref) < 1e-11
    assert abs(sim.norm() - 1.0) < 1e-12


def _full_length(P, w, t0, nsteps, tol):
    """Whole grid, `nsteps` RK4 steps from t0, GPU against the C oracle (textbook k1..k4, explicit loops, all host
    cores) element by element; the active set the GPU runs on is first compared with the oracle's own."""
    box, pot, act = oracle_objs(w)
    grid, gact, psi0, _, _ = _setup(P, w)
    assert np.array_equal(gact, act)
    sim = P.Sim(grid, w.dtype, w.stencil, w.g)
    psi_in = psi0.astype(sim.npdtype)
    sim.set_psi_host(psi_in)
    sim.time = t0
    sim.run_rk4(w.dt, nsteps)
    got = sim.get_psi_host()
    nrm = sim.norm()
    co = CO.COracle(box, pot, act, w.stencil)
    ref = co.run_rk4(w.g, t0, w.dt, nsteps, psi_in.astype(np.complex128))   # complex64: the fp32-rounded input
    err = rel_max(got, ref)
    assert err < tol, (w.name, w.dtype, nsteps, err)
    assert abs(nrm - co.norm(ref)) < (1e-10 if w.dtype == "complex128" else 1e-4)
    return sim, psi_in, got


@pytest.mark.slow
def test_config4_full_length_complex128(P):
    """BASELINE configs[3] as specified: 200 real-time RK4 steps dt = 1e-4 on the whole 1024^3 bubble, every one of
    the 31 523 416 values against the oracle (2.5e10 stage updates: about a minute on the box's host cores).  Bound:
    the north_star's 1e-9 (asked after 1000 steps).  Also what must hold at any size: the static potential
    conserves norm and energy up to RK4's O(dt^4) error (P8), and a second run from the same input is bit-identical."""
    w = I.config4("complex128")
    assert w.nsteps == 200
    sim, psi_in, got = _full_length(P, w, 0.0, w.nsteps, 1e-9)
    assert abs(sim.time - 200 * w.dt) < 1e-15
    e1 = sim.energy()
    sim.set_psi_host(psi_in)
    sim.time = 0.0
    e0 = sim.energy()
    assert abs(sim.norm() - 1.0) < 1e-12
    assert abs(e1["total"] - e0["total"]) < 1e-7 * abs(e0["total"])
    sim.run_rk4(w.dt, w.nsteps)
    assert np.array_equal(sim.get_psi_host(), got)


@pytest.mark.slow
def test_config4_full_length_complex64(P):
    """The same 200 steps in complex64 against the complex128 oracle fed the fp32-rounded input (north_star: 1e-3)."""
    _full_length(P, I.config4("complex64"), 0.0, 200, 1e-3)


@pytest.mark.slow
@pytest.mark.parametrize("union", [True, False])
def test_config3_first_50_steps_full_size(P, union):
    """BASELINE configs[2] at full size (512^3, 7-point, Delta(t) evaluated per stage): 50 RK4 steps on the whole
    grid starting inside the ramp (t0 = 1), union mask (3.85e7 points) and final-shell mask (9.7e6)."""
    _full_length(P, I.config3(union), 1.0, 50, 1e-9)


def test_config3_whole_ramp_on_a_replica(P):
    """BASELINE configs[2], the whole hollowing-out ramp Delta: 0 -> 800 (t_ramp = 4) against the oracle on a
    128^3, h = 0.8 replica of the 512^3 box (same physical box and potential, union mask; the oracle cannot follow
    3e12 stage updates at full size): 2000 RK4 steps dt = 2e-3, V evaluated at every stage time."""
    w = I.config3(True).with_(nx=128, ny=128, nz=128, h=0.8, dt=2e-3, name="cfg3a_replica_128")
    box, pot, act = oracle_objs(w)
    grid = P.Grid.from_workload(w)
    assert np.array_equal(grid.active_indices(), act) and act.size > 4e5
    sim = P.Sim(grid, "complex128", w.stencil, w.g)
    co = CO.COracle(box, pot, act, w.stencil)
    psi = I.make_psi0(w, act)
    sim.set_psi_host(psi)
    sim.run_rk4(w.dt, 2000)
    assert abs(sim.time - w.t_ramp) < 1e-12
    ref = co.run_rk4(w.g, 0.0, w.dt, 2000, psi)
    assert rel_max(sim.get_psi_host(), ref) < 2e-9
    assert abs(sim.norm() - co.norm(ref)) < 1e-10
