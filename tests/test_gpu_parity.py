"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  Tolerances are BASELINE.json's north_star: max relative error (R10:
max|a-b| / max|b|) 1e-12 per operator application and 1e-9 after 1000 steps in complex128; 1e-5 and 1e-3
in complex64 (the complex64 result is compared against the complex128 oracle fed the fp32-rounded input)."""
import numpy as np
import pytest

import gpe_inputs as I
from helpers import RADIUS, oracle_objs, rel_max
from oracle import c_oracle as CO
from oracle import gpe_oracle as O

pytestmark = pytest.mark.gpu

TOL_APPLY = {"complex128": 1e-12, "complex64": 1e-5}
TOL_STEPS = {"complex128": 1e-9, "complex64": 1e-3}


@pytest.fixture(scope="module")
def P():
    import paper_2603_05447_b200 as P
    return P


def _torch():
    import torch
    return torch


def _dev(x, dtype):
    torch = _torch()
    return torch.from_numpy(np.ascontiguousarray(x)).to("cuda:0").to(getattr(torch, dtype))


def _make(P, w, active=None, dtype=None):
    box, pot, act = oracle_objs(w, active)
    grid = P.Grid.from_workload(w, active=active)
    assert np.array_equal(grid.active_indices(), act)
    sim = P.Sim(grid, dtype or w.dtype, w.stencil, w.g)
    return box, pot, act, grid, sim


@pytest.mark.parametrize("dtype", ["complex128", "complex64"])
@pytest.mark.parametrize("stencil", [7, 13])
@pytest.mark.parametrize("kz", [16, 5, 32])
def test_apply_H_small_shell(P, stencil, dtype, kz):
    w = I.small_shell(40, stencil, dtype).with_(delta0=14.0, delta1=22.0, t_ramp=0.5)
    box, pot, act, grid, sim = _make(P, w)
    sim.set_planes_per_block(kz)
    og = O.SparseGrid(box, act, RADIUS[stencil])
    psi = I.random_psi(7, act.size).astype(sim.npdtype)
    for t in (0.0, 0.3, 2.0):
        got = sim.apply_H(t, _dev(psi, dtype)).cpu().numpy()
        ref = O.apply_H(og, pot, w.g, t, psi.astype(np.complex128), stencil)
        assert rel_max(got, ref) < TOL_APPLY[dtype]


@pytest.mark.parametrize("dims,p,seed", [((9, 7, 11), 0.4, 3), ((17, 16, 40), 0.15, 4), ((8, 8, 70), 0.9, 5),
                                         ((6, 6, 6), 1.1, 6), ((19, 21, 37), 0.6, 8)])
@pytest.mark.parametrize("stencil", [7, 13])
def test_apply_H_random_masks(P, dims, p, seed, stencil):
    """Random masks (holes everywhere, box faces touched) and the full 6^3 box."""
    nx, ny, nz = dims
    w = I.Workload(name="rnd", nx=nx, ny=ny, nz=nz, h=0.3, kind=I.DRESSED, ax=1.0, ay=0.7, az=1.2, delta0=2.0,
                   delta1=2.0, omega=1.5, stencil=stencil, g=3.0)
    act = I.random_mask_lin(seed, nx, ny, nz, p)
    box, pot, act, grid, sim = _make(P, w, active=act)
    og = O.SparseGrid(box, act, RADIUS[stencil])
    psi = I.random_psi(seed + 100, act.size)
    got = sim.apply_H(0.1, _dev(psi, "complex128")).cpu().numpy()
    assert rel_max(got, O.apply_H(og, pot, w.g, 0.1, psi, stencil)) < 1e-12


def test_single_point_and_empty(P):
    w = I.Workload(name="one", nx=5, ny=4, nz=3, h=0.5, kind=I.HARMONIC, stencil=13, g=2.0)
    box, pot, act, grid, sim = _make(P, w, active=np.array([17], np.int64))
    og = O.SparseGrid(box, act, 2)
    psi = np.array([0.3 - 0.8j])
    got = sim.apply_H(0.0, _dev(psi, "complex128")).cpu().numpy()
    assert rel_max(got, O.apply_H(og, pot, w.g, 0.0, psi, 13)) < 1e-12
    sim.set_psi_host(psi)
    sim.run_rk4(1e-3, 3)
    assert rel_max(sim.get_psi_host(), O.run_rk4(og, pot, w.g, 0.0, 1e-3, 3, psi, 13)) < 1e-12
    # empty grid: every call is a no-op
    grid0 = P.Grid.from_workload(w.with_(v_cut=-1.0))
    sim0 = P.Sim(grid0, "complex128", 13, 1.0)
    sim0.run_rk4(1e-3, 2)
    sim0.run_imag(1e-3, 2)
    assert sim0.norm() == 0.0 and sim0.get_psi_host().size == 0


def test_set_get_roundtrip_and_norm(P):
    w = I.small_shell(40, 13)
    box, pot, act, grid, sim = _make(P, w)
    psi = I.make_psi0(w, act)
    sim.set_psi_host(psi)
    assert np.array_equal(sim.get_psi_host(), psi)
    d = _dev(psi, "complex128")
    sim.set_psi(d)
    assert np.array_equal(sim.get_psi().cpu().numpy(), psi)
    og = O.SparseGrid(box, act, 2)
    assert abs(sim.norm() - O.norm(og, psi)) < 1e-13
    assert sim.norm() == sim.norm()  # fixed summation order: bit-reproducible


@pytest.mark.parametrize("dtype", ["complex128", "complex64"])
@pytest.mark.parametrize("stencil", [7, 13])
def test_rk4_small_shell_with_ramp(P, stencil, dtype):
    """RK4 stage-state form (PAPER.md Eq. A6-A7, A10-A11) against the textbook k1..k4 oracle with a
    time-ramped potential (stage times t, t+dt/2, t+dt/2, t+dt)."""
    w = I.small_shell(40, stencil, dtype).with_(delta0=14.0, delta1=22.0, t_ramp=0.02)
    box, pot, act, grid, sim = _make(P, w)
    og = O.SparseGrid(box, act, RADIUS[stencil])
    psi = I.make_psi0(w, act).astype(sim.npdtype)
    sim.set_psi_host(psi)
    sim.time = 0.005
    sim.run_rk4(w.dt, 4)
    sim.step_rk4(w.dt)
    assert abs(sim.time - (0.005 + 5 * w.dt)) < 1e-15
    ref = O.run_rk4(og, pot, w.g, 0.005, w.dt, 5, psi.astype(np.complex128), stencil)
    assert rel_max(sim.get_psi_host(), ref) < (1e-12 if dtype == "complex128" else 1e-5)


@pytest.mark.parametrize("stencil", [7, 13])
def test_imag_and_energy_small_shell(P, stencil):
    w = I.small_shell(40, stencil)
    box, pot, act, grid, sim = _make(P, w)
    og = O.SparseGrid(box, act, RADIUS[stencil])
    psi = I.make_psi0(w, act)
    sim.set_psi_host(psi)
    e = sim.energy()
    ref = O.energy(og, pot, w.g, 0.0, psi, stencil)
    for k in ref:
        assert abs(e[k] - ref[k]) <= 1e-12 * max(1.0, abs(ref[k])), k
    sim.run_imag(1e-3, 9)
    sim.imag_step(1e-3)
    ref = O.run_imag(og, pot, w.g, 0.0, 1e-3, 10, psi, stencil)
    assert rel_max(sim.get_psi_host(), ref) < 1e-12
    assert abs(sim.norm() - 1.0) < 1e-12
    e2 = sim.energy()
    assert e2["total"] < e["total"]  # imaginary time lowers the energy


def test_config1_100_and_1000_steps(P):
    """BASELINE configs[0]: 48^3 harmonic trap, 7-pt, g=100, complex128; 100 steps and the 1e-9 bound
    after 1000 steps (C oracle: explicit loops, textbook RK4)."""
    w = I.config1()
    box, pot, act, grid, sim = _make(P, w)
    co = CO.COracle(box, pot, act, w.stencil)
    psi = I.make_psi0(w, act)
    sim.set_psi_host(psi)
    sim.run_rk4(w.dt, 100)
    ref = co.run_rk4(w.g, 0.0, w.dt, 100, psi)
    assert rel_max(sim.get_psi_host(), ref) < 1e-11
    sim.run_rk4(w.dt, 900)
    ref = co.run_rk4(w.g, 100 * w.dt, w.dt, 900, ref)
    assert rel_max(sim.get_psi_host(), ref) < 1e-9
    assert abs(sim.norm() - co.norm(ref)) < 1e-11


def test_config1_complex64_1000_steps(P):
    w = I.config1().with_(dtype="complex64")
    box, pot, act, grid, sim = _make(P, w)
    co = CO.COracle(box, pot, act, w.stencil)
    psi = I.make_psi0(w, act).astype(np.complex64)
    sim.set_psi_host(psi)
    sim.run_rk4(w.dt, 1000)
    ref = co.run_rk4(w.g, 0.0, w.dt, 1000, psi.astype(np.complex128))
    assert rel_max(sim.get_psi_host(), ref) < 1e-3


@pytest.mark.parametrize("dtype", ["complex128", "complex64"])
@pytest.mark.parametrize("stencil", [7, 13])
def test_imag_split_small_shell(P, stencil, dtype):
    """The paper's own ground-state iteration (Eq. 7 half steps with the linearised interaction
    factor, two forward-Euler kinetic half steps, renormalisation) against the oracle's imag_split_step."""
    w = I.small_shell(40, stencil, dtype).with_(g=400.0)
    box, pot, act, grid, sim = _make(P, w)
    og = O.SparseGrid(box, act, RADIUS[stencil])
    psi = I.make_psi0(w, act).astype(sim.npdtype)
    sim.set_psi_host(psi)
    sim.run_imag_split(2e-3, 7)
    sim.imag_split_step(2e-3)
    ref = O.run_imag_split(og, pot, w.g, 0.0, 2e-3, 8, psi.astype(np.complex128), stencil)
    assert rel_max(sim.get_psi_host(), ref) < (1e-12 if dtype == "complex128" else 1e-5)
    assert abs(sim.norm() - 1.0) < (1e-12 if dtype == "complex128" else 1e-5)
    if dtype == "complex128":
        # both schemes lower the energy from the same start, and the Euler scheme follows within O(dt)
        e0 = O.energy(og, pot, w.g, 0.0, psi.astype(np.complex128), stencil)["total"]
        assert sim.energy()["total"] < e0


@pytest.mark.parametrize("dtype", ["complex128", "complex64", "float64"])
@pytest.mark.parametrize("stencil", [7, 13, 19, 27])
def test_imag_split_k1_equals_three_launches(P, stencil, dtype):
    """The paper's K1 (Eq. 7 half step and lazy scale applied to every value while it is staged, own
    and halo, then the first Euler half step) gives bit for bit what the separate pointwise launch followed by the
    kinetic launch gives (gpe_sim_set_option GPE_OPT_FUSED_K1 = 0): the same arithmetic at the same point, whichever
    tile stages the value.  Stencil 27 runs with caller-supplied weights and a non-zero corner weight, so the eight
    corner reads of the diagonal tiles go through the folded load too."""
    w = I.small_shell(40, stencil, "complex128" if dtype == "float64" else dtype).with_(g=400.0)
    grid = P.Grid.from_workload(w)
    act = grid.active_indices()
    psi = I.make_psi0(w, act)
    psi = np.abs(psi).astype(np.float64) if dtype == "float64" else psi.astype(np.complex64 if dtype == "complex64" else np.complex128)
    out = []
    for k1 in (1, 0):
        sim = P.Sim(grid, dtype, stencil, w.g)
        sim.set_option(P.OPT_FUSED_K1, k1)
        if stencil == 27:
            h2 = w.h ** 2
            sim.set_compact_weights(-64.0 / 15.0 / h2, [7.0 / 15.0 / h2] * 3, [0.1 / h2] * 3, 1.0 / 30.0 / h2)
        sim.set_psi_host(psi)
        n0 = sim.kernel_launches
        sim.run_imag_split(2e-3, 6)
        out.append((sim.get_psi_host().copy(), sim.kernel_launches - n0))
        sim.close()
    assert np.array_equal(out[0][0], out[1][0])
    assert np.all(np.isfinite(out[0][0].view(np.float64 if dtype != "complex64" else np.float32)))
    assert out[1][1] - out[0][1] == 6          # one stencil launch less per iteration


@pytest.mark.parametrize("dims,p,seed", [((9, 7, 11), 0.4, 3), ((17, 16, 40), 0.15, 4), ((8, 8, 70), 0.9, 5),
                                         ((6, 6, 6), 1.1, 6), ((19, 21, 37), 0.6, 8), ((1, 20, 33), 0.8, 9), ((24, 1, 1), 0.7, 10)])
@pytest.mark.parametrize("stencil", [7, 13, 19])
@pytest.mark.parametrize("kz", [32, 3, 1])
def test_imag_split_k1_random_masks(P, dims, p, seed, stencil, kz):
    """K1 on random masks (holes everywhere, box faces touched, streams of 1-3 planes, boxes one point thick): the
    iteration against the oracle, and bit for bit against the three-launch form."""
    nx, ny, nz = dims
    w = I.Workload(name="rnd", nx=nx, ny=ny, nz=nz, h=0.3, kind=I.DRESSED, ax=1.0, ay=0.7, az=1.2, delta0=2.0,
                   delta1=2.0, omega=1.5, stencil=stencil, g=3.0)
    act = I.random_mask_lin(seed, nx, ny, nz, p)
    box, pot, act = oracle_objs(w, act)
    grid = P.Grid.from_workload(w, active=act)
    og = O.SparseGrid(box, act, RADIUS[stencil])
    psi = I.random_psi(seed + 100, act.size)
    out = []
    for k1 in (1, 0):
        sim = P.Sim(grid, "complex128", stencil, w.g)
        sim.set_option(P.OPT_FUSED_K1, k1)
        sim.set_planes_per_block(kz)
        sim.set_psi_host(psi)
        sim.run_imag_split(5e-3, 4)
        out.append(sim.get_psi_host().copy())
        sim.close()
    assert np.array_equal(out[0], out[1])
    assert rel_max(out[0], O.run_imag_split(og, pot, w.g, 0.0, 5e-3, 4, psi, stencil)) < 1e-12


@pytest.mark.parametrize("dtype", ["complex128", "complex64"])
def test_regrid_remap(P, dtype):
    """Re-gridding between ramp stages: the state is carried from the shell at Delta = 14 to the
    post-selection at Delta = 22 (a larger, partly overlapping shell) and evolved on; against the oracle."""
    wa = I.small_shell(40, 13, dtype).with_(delta0=14.0, delta1=14.0)
    wb = wa.with_(delta0=22.0, delta1=22.0)
    box, pot_a, act_a, grid_a, sim_a = _make(P, wa)
    _, pot_b, act_b, grid_b, sim_b = _make(P, wb)
    assert 0 < np.intersect1d(act_a, act_b).size < min(act_a.size, act_b.size)
    psi = I.make_psi0(wa, act_a).astype(sim_a.npdtype)
    sim_a.set_psi_host(psi)
    sim_a.time = 0.25
    sim_b.remap_from(sim_a)
    want = O.remap_psi(act_a, psi.astype(np.complex128), act_b)
    assert np.array_equal(sim_b.get_psi_host(), want.astype(sim_b.npdtype))     # a copy: bit-exact
    assert sim_b.time == 0.25
    sim_b.run_rk4(wb.dt, 2)
    og = O.SparseGrid(box, act_b, 2)
    ref = O.run_rk4(og, pot_b, wb.g, 0.25, wb.dt, 2, want, 13)
    assert rel_max(sim_b.get_psi_host(), ref) < (1e-12 if dtype == "complex128" else 1e-5)
    # different precision or box: refused
    other = P.Sim(grid_b, "complex64" if dtype == "complex128" else "complex128", 13, wb.g)
    with pytest.raises(P.GpeError):
        other.remap_from(sim_a)


@pytest.mark.parametrize("dtype", ["complex128", "complex64"])
@pytest.mark.parametrize("stencil", [7, 13])
def test_rkhe3_small_shell_with_ramp(P, stencil, dtype):
    """Heun's third-order method in the paper's stage-state form (PAPER.md Eq. A6-A9) against the textbook
    k1..k3 oracle, time-ramped potential (stage times t, t + dt/3, t + 2dt/3)."""
    w = I.small_shell(40, stencil, dtype).with_(delta0=14.0, delta1=22.0, t_ramp=0.02)
    box, pot, act, grid, sim = _make(P, w)
    og = O.SparseGrid(box, act, RADIUS[stencil])
    psi = I.make_psi0(w, act).astype(sim.npdtype)
    sim.set_psi_host(psi)
    sim.time = 0.005
    sim.run_rkhe3(w.dt, 4)
    sim.step_rkhe3(w.dt)
    assert abs(sim.time - (0.005 + 5 * w.dt)) < 1e-15
    ref = O.run_rkhe3(og, pot, w.g, 0.005, w.dt, 5, psi.astype(np.complex128), stencil)
    assert rel_max(sim.get_psi_host(), ref) < (1e-12 if dtype == "complex128" else 1e-5)


@pytest.mark.parametrize("dtype", ["complex128", "complex64"])
@pytest.mark.parametrize("stencil", [7, 13])
def test_rkck_small_shell_with_ramp(P, stencil, dtype):
    """Cash-Karp in the paper's stage-state form (PAPER.md Eq. A6-A7, A12-A13) against the textbook k1..k6
    oracle, time-ramped potential (stage times t + c_i dt)."""
    w = I.small_shell(40, stencil, dtype).with_(delta0=14.0, delta1=22.0, t_ramp=0.02)
    box, pot, act, grid, sim = _make(P, w)
    og = O.SparseGrid(box, act, RADIUS[stencil])
    psi = I.make_psi0(w, act).astype(sim.npdtype)
    sim.set_psi_host(psi)
    sim.time = 0.005
    sim.run_rkck(w.dt, 2)
    sim.step_rkck(w.dt)
    ref = O.run_rkck(og, pot, w.g, 0.005, w.dt, 3, psi.astype(np.complex128), stencil)
    assert rel_max(sim.get_psi_host(), ref) < (1e-12 if dtype == "complex128" else 2e-5)
    # the other integrators still run on the same sim afterwards (buffers A-D are shared)
    sim.run_rk4(w.dt, 1)
    ref = O.run_rk4(og, pot, w.g, 0.005 + 3 * w.dt, w.dt, 1, ref, stencil)
    assert rel_max(sim.get_psi_host(), ref) < (1e-12 if dtype == "complex128" else 2e-5)


@pytest.mark.parametrize("dtype", ["complex128", "complex64"])
def test_19pt_hoc_stencil(P, dtype):
    """The paper's 19-point higher-order compact Laplacian (PAPER.md:341-343 Eq. B2, isotropic spacing): operator,
    RK4 with a ramped potential, imaginary time and the energy sums against the oracle; shells with ragged
    tails (diagonal tiles present and absent) and random masks touching the box faces."""
    tol = 1e-12 if dtype == "complex128" else 1e-5
    w = I.small_shell(40, 19, dtype).with_(delta0=14.0, delta1=22.0, t_ramp=0.02)
    box, pot, act, grid, sim = _make(P, w)
    og = O.SparseGrid(box, act, 1)
    psi = I.random_psi(7, act.size).astype(sim.npdtype)
    for kz in (5, 32):
        sim.set_planes_per_block(kz)
        got = sim.apply_H(0.3, _dev(psi, dtype)).cpu().numpy()
        assert rel_max(got, O.apply_H(og, pot, w.g, 0.3, psi.astype(np.complex128), 19)) < tol
    psi = I.make_psi0(w, act).astype(sim.npdtype)
    sim.set_psi_host(psi)
    sim.time = 0.005
    sim.run_rk4(w.dt, 3)
    ref = O.run_rk4(og, pot, w.g, 0.005, w.dt, 3, psi.astype(np.complex128), 19)
    assert rel_max(sim.get_psi_host(), ref) < tol
    if dtype == "complex128":
        e, eo = sim.energy(), O.energy(og, pot, w.g, sim.time, ref, 19)
        for k in eo:
            assert abs(e[k] - eo[k]) <= 1e-11 * max(1.0, abs(eo[k])), k
        sim.set_psi_host(psi)
        sim.run_imag(1e-3, 4)
        assert rel_max(sim.get_psi_host(), O.run_imag(og, pot, w.g, sim.time, 1e-3, 4, psi, 19)) < tol
        sim.set_psi_host(psi)
        sim.run_imag_split(1e-3, 3)
        assert rel_max(sim.get_psi_host(), O.run_imag_split(og, pot, w.g, sim.time, 1e-3, 3, psi, 19)) < tol


@pytest.mark.parametrize("dims,p,seed", [((9, 7, 11), 0.4, 3), ((17, 16, 40), 0.15, 4), ((6, 6, 6), 1.1, 6), ((19, 21, 37), 0.6, 8)])
def test_19pt_random_masks(P, dims, p, seed):
    nx, ny, nz = dims
    w = I.Workload(name="rnd", nx=nx, ny=ny, nz=nz, h=0.3, kind=I.DRESSED, ax=1.0, ay=0.7, az=1.2, delta0=2.0,
                   delta1=2.0, omega=1.5, stencil=19, g=3.0)
    act = I.random_mask_lin(seed, nx, ny, nz, p)
    box, pot, act, grid, sim = _make(P, w, active=act)
    og = O.SparseGrid(box, act, 1)
    psi = I.random_psi(seed + 100, act.size)
    got = sim.apply_H(0.1, _dev(psi, "complex128")).cpu().numpy()
    assert rel_max(got, O.apply_H(og, pot, w.g, 0.1, psi, 19)) < 1e-12


@pytest.mark.parametrize("dtype,stencil", [("complex128", 13), ("complex64", 13), ("complex128", 19)])
def test_small_shell_1000_steps(P, dtype, stencil):
    """The north_star's long-run bound on a shell (ragged tiles, ramped potential): max relative error 1e-9 after
    1000 RK4 steps in complex128, 1e-3 in complex64 (19-point: 200 steps)."""
    w = I.small_shell(40, stencil, dtype).with_(delta0=14.0, delta1=16.0, t_ramp=0.5)
    box, pot, act, grid, sim = _make(P, w)
    psi = I.make_psi0(w, act).astype(sim.npdtype)
    sim.set_psi_host(psi)
    nsteps = 200 if stencil == 19 else 1000          # the NumPy oracle (no C restatement of the 19-point stencil)
    sim.run_rk4(w.dt, nsteps)
    if stencil == 19:
        og = O.SparseGrid(box, act, 1)
        ref = O.run_rk4(og, pot, w.g, 0.0, w.dt, nsteps, psi.astype(np.complex128), 19)
    else:
        ref = CO.COracle(box, pot, act, stencil).run_rk4(w.g, 0.0, w.dt, 1000, psi.astype(np.complex128))
    assert rel_max(sim.get_psi_host(), ref) < TOL_STEPS[dtype]


@pytest.mark.parametrize("dtype", ["complex128", "complex64"])
@pytest.mark.parametrize("stencil", [7, 13, 19])
def test_anisotropic_spacing(P, stencil, dtype):
    """Anisotropic grids d_x != d_y != d_z (App. B, Eq. B1-B2): the mask, the operator with
    per-axis weights (19-point: pair weights (d_i^2 + d_j^2)/12), RK4, the volume element of the reductions."""
    tol = 1e-12 if dtype == "complex128" else 1e-5
    w = I.small_shell(40, stencil, dtype).with_(hy=0.8 * 0.5, hz=1.3 * 0.5, delta0=14.0, delta1=20.0, t_ramp=0.02)
    w = w.with_(h=0.5)
    box, pot, act, grid, sim = _make(P, w)
    assert act.size > 3000
    og = O.SparseGrid(box, act, RADIUS[stencil])
    psi = I.random_psi(9, act.size).astype(sim.npdtype)
    got = sim.apply_H(0.004, _dev(psi, dtype)).cpu().numpy()
    assert rel_max(got, O.apply_H(og, pot, w.g, 0.004, psi.astype(np.complex128), stencil)) < tol
    psi = I.make_psi0(w, act).astype(sim.npdtype)
    sim.set_psi_host(psi)
    assert abs(sim.norm() - 1.0) < (1e-12 if dtype == "complex128" else 1e-6)     # h hy hz sum |psi|^2
    sim.run_rk4(w.dt, 3)
    ref = O.run_rk4(og, pot, w.g, 0.0, w.dt, 3, psi.astype(np.complex128), stencil)
    assert rel_max(sim.get_psi_host(), ref) < tol
    if dtype == "complex128":
        e, eo = sim.energy(), O.energy(og, pot, w.g, sim.time, ref, stencil)
        for k in eo:
            assert abs(e[k] - eo[k]) <= 1e-11 * max(1.0, abs(eo[k])), k


@pytest.mark.parametrize("stencil", [7, 13, 19])
def test_real_valued_ground_state_mode(P, stencil):
    """Real float64 state (imaginary time "does not require the wavefunction to be complex"): the
    operator, both imaginary-time schemes, norm, energy and re-gridding on half the bytes; the oracle runs the
    same real initial state as complex128 and must stay real exactly."""
    w = I.small_shell(40, stencil)
    box, pot, act, grid, _ = _make(P, w)
    sim = P.Sim(grid, "float64", stencil, w.g)
    og = O.SparseGrid(box, act, RADIUS[stencil])
    psi = np.abs(I.make_psi0(w, act)) * (1.0 + 0.1 * np.cos(np.arange(act.size)))
    psi = psi / np.sqrt(O.norm(og, psi.astype(np.complex128)))
    import torch
    got = sim.apply_H(0.0, torch.from_numpy(psi).to("cuda:0")).cpu().numpy()
    ref = O.apply_H(og, pot, w.g, 0.0, psi.astype(np.complex128), stencil)
    assert np.all(ref.imag == 0) and rel_max(got, ref.real) < 1e-12
    sim.set_psi_host(psi)
    assert np.array_equal(sim.get_psi_host(), psi)
    assert abs(sim.norm() - 1.0) < 1e-13
    sim.run_imag(1e-3, 7)
    ref = O.run_imag(og, pot, w.g, 0.0, 1e-3, 7, psi.astype(np.complex128), stencil)
    assert np.all(ref.imag == 0) and rel_max(sim.get_psi_host(), ref.real) < 1e-12
    e, eo = sim.energy(), O.energy(og, pot, w.g, 0.0, ref, stencil)
    for k in eo:
        assert abs(e[k] - eo[k]) <= 1e-12 * max(1.0, abs(eo[k])), k
    sim.run_imag_split(1e-3, 5)
    ref = O.run_imag_split(og, pot, w.g, 0.0, 1e-3, 5, ref, stencil)
    assert rel_max(sim.get_psi_host(), ref.real) < 1e-12
    assert abs(sim.norm() - 1.0) < 1e-12
    # real time needs the imaginary part
    with pytest.raises(P.GpeError):
        sim.run_rk4(1e-3, 1)
    # re-gridding, and an odd number of points (the pair-wise reductions see a zero tail)
    wb = w.with_(delta0=22.0, delta1=22.0)
    _, _, act_b, grid_b, _ = _make(P, wb)
    sim_b = P.Sim(grid_b, "float64", stencil, w.g)
    sim_b.remap_from(sim)
    assert np.array_equal(sim_b.get_psi_host(), O.remap_psi(act, sim.get_psi_host(), act_b).real)
    odd = act[: (act.size // 2) * 2 - 1]
    _, _, _, grid_o, _ = _make(P, w, active=odd)
    sim_o = P.Sim(grid_o, "float64", stencil, w.g)
    sim_o.set_psi_host(psi[: odd.size])
    assert abs(sim_o.norm() - O.norm(O.SparseGrid(box, odd, RADIUS[stencil]), psi[: odd.size].astype(np.complex128))) < 1e-13


@pytest.mark.parametrize("dtype", ["complex128", "complex64"])
def test_27pt_compact_stencil_with_supplied_weights(P, dtype):
    """stencil = 27: the 3x3x3 compact stencil with caller-supplied weights (the paper does not print those of its
    27-point stencil; parity unpinned for any published set, mechanism pinned by P19): all four
    neighbour classes non-zero, anisotropic, against the oracle's apply_T27; default weights = the 19-point ones."""
    tol = 1e-12 if dtype == "complex128" else 1e-5
    w = I.small_shell(40, 13, dtype).with_(hy=0.45, hz=0.6, delta0=14.0, delta1=20.0, t_ramp=0.02)
    box, pot, act = oracle_objs(w)
    grid = P.Grid.from_workload(w)
    sim = P.Sim(grid, dtype, 27, w.g)
    og = O.SparseGrid(box, act, 1)
    psi = I.random_psi(5, act.size).astype(sim.npdtype)
    got = sim.apply_H(0.0, _dev(psi, dtype)).cpu().numpy()
    assert rel_max(got, O.apply_H(og, pot, w.g, 0.0, psi.astype(np.complex128), 19)) < tol
    cw = O.Compact27(-9.3, (1.9, 2.6, 1.2), (0.31, 0.22, 0.27), 0.05)
    sim.set_compact_weights(cw.centre, cw.face, cw.edge, cw.corner)
    got = sim.apply_H(0.0, _dev(psi, dtype)).cpu().numpy()
    assert rel_max(got, O.apply_H(og, pot, w.g, 0.0, psi.astype(np.complex128), cw)) < tol
    psi = I.make_psi0(w, act).astype(sim.npdtype)
    sim.set_psi_host(psi)
    sim.run_rk4(w.dt, 3)
    assert rel_max(sim.get_psi_host(), O.run_rk4(og, pot, w.g, 0.0, w.dt, 3, psi.astype(np.complex128), cw)) < tol
    star = P.Sim(grid, dtype, 13, w.g)
    with pytest.raises(P.GpeError):
        star.set_compact_weights(cw.centre, cw.face, cw.edge, cw.corner)


@pytest.mark.parametrize("stencil", [7, 13, 19])
@pytest.mark.parametrize("kz", [1, 2, 3])
def test_shortest_streams(P, stencil, kz):
    """Streams of 1, 2 and 3 planes (shorter than the prefetch depth): operator and two RK4 steps."""
    w = I.small_shell(24, stencil).with_(delta0=5.0, delta1=8.0, t_ramp=0.02)
    box, pot, act, grid, sim = _make(P, w)
    sim.set_planes_per_block(kz)
    og = O.SparseGrid(box, act, RADIUS[stencil])
    psi = I.make_psi0(w, act)
    got = sim.apply_H(0.01, _dev(psi, "complex128")).cpu().numpy()
    assert rel_max(got, O.apply_H(og, pot, w.g, 0.01, psi, stencil)) < 1e-12
    sim.set_psi_host(psi)
    sim.run_rk4(w.dt, 2)
    assert rel_max(sim.get_psi_host(), O.run_rk4(og, pot, w.g, 0.0, w.dt, 2, psi, stencil)) < 1e-12


@pytest.mark.parametrize("stencil", [7, 13, 19])
@pytest.mark.parametrize("dims", [(5, 3, 1), (1, 1, 9), (8, 8, 1), (1, 17, 2), (16, 1, 3)])
def test_degenerate_boxes(P, dims, stencil):
    """Boxes one point thick along one or two axes, fully active: every neighbour lookup hits a box face."""
    nx, ny, nz = dims
    w = I.Workload(name="thin", nx=nx, ny=ny, nz=nz, h=0.4, kind=I.HARMONIC, ax=1.0, ay=2.0, az=0.5, stencil=stencil, g=2.0)
    act = np.arange(nx * ny * nz, dtype=np.int64)
    box, pot, act, grid, sim = _make(P, w, active=act)
    og = O.SparseGrid(box, act, RADIUS[stencil])
    psi = I.random_psi(3, act.size)
    got = sim.apply_H(0.0, _dev(psi, "complex128")).cpu().numpy()
    assert rel_max(got, O.apply_H(og, pot, w.g, 0.0, psi, stencil)) < 1e-12
    sim.set_psi_host(psi)
    sim.run_rk4(1e-3, 2)
    assert rel_max(sim.get_psi_host(), O.run_rk4(og, pot, w.g, 0.0, 1e-3, 2, psi, stencil)) < 1e-12


def test_zero_state_has_no_renormalisation(P):
    """A state with zero particle number cannot be renormalised: no NaN is produced (the scale stays 1) and
    GPE_ERR_STATE is reported by the first synchronising call after the run (the runs themselves stay asynchronous);
    the sim stays usable."""
    w = I.small_shell(24, 13)
    box, pot, act, grid, sim = _make(P, w)
    zero = np.zeros(act.size, np.complex128)
    for run in (sim.run_imag, sim.run_imag_split):
        sim.set_psi_host(zero)
        run(1e-3, 3)
        with pytest.raises(P.GpeError) as e:
            sim.norm()
        assert e.value.code == -5
        assert np.all(sim.get_psi_host() == 0)             # scale 1 was applied: no NaN; the flag was reported once
    psi = I.make_psi0(w, act)
    sim.set_psi_host(psi)
    sim.run_imag(1e-3, 2)
    og = O.SparseGrid(box, act, 2)
    assert rel_max(sim.get_psi_host(), O.run_imag(og, pot, w.g, 0.0, 1e-3, 2, psi, 13)) < 1e-12


def test_replacing_the_state_discards_an_unreported_degenerate_flag(P):
    """include/gpe.h, gpe_imag_step: the deferred GPE_ERR_STATE belongs to the state that raised it.  A zero state runs
    through both imaginary-time forms with no reporting call in between; then the state is replaced (host copy, device
    copy, re-gridding from another sim) and the next run, norm and read-back succeed and match the oracle."""
    w = I.small_shell(24, 13)
    box, pot, act, grid, sim = _make(P, w)
    og = O.SparseGrid(box, act, 2)
    zero = np.zeros(act.size, np.complex128)
    psi = I.make_psi0(w, act)
    ref = O.run_imag(og, pot, w.g, 0.0, 1e-3, 2, psi, 13)
    src = P.Sim(grid, "complex128", 13, w.g)
    src.set_psi_host(psi)
    for replace in (lambda: sim.set_psi_host(psi), lambda: sim.set_psi(_dev(psi, "complex128")), lambda: sim.remap_from(src)):
        sim.set_psi_host(zero)
        sim.run_imag(1e-3, 3)
        _torch().cuda.synchronize()                        # the flag is up and its copy has landed, nobody has asked yet
        replace()
        sim.run_imag(1e-3, 2)                              # would return GPE_ERR_STATE if the stale flag were still pending
        assert abs(sim.norm() - 1.0) < 1e-12
        assert rel_max(sim.get_psi_host(), ref) < 1e-12
    # and a flag raised by the new state is still reported
    sim.set_psi_host(zero)
    sim.run_imag_split(1e-3, 2)
    with pytest.raises(P.GpeError) as e:
        sim.norm()
    assert e.value.code == -5


def test_staged_ramp_with_regridding(P):
    """The ramp as the paper runs it: stage after stage of a linearly interpolated potential;
    at the end of each stage the grid post-selection is repeated with the threshold 5 max(mu_i, mu_i+1) and the
    wavefunction is remapped from the old grid to the new one.  Here: the 128^3, h = 0.8 replica of BASELINE
    configs[2] (Omega = 20, g = 2000, 7-point), Delta: 0 -> 80 in 8 stages of 100 RK4 steps (dt = 2e-3, stage
    length 0.2; the full 0 -> 800 in this time is far from adiabatic and leaves RK4's stability range); mu_i is the chemical potential of the evolving state at the stage boundary (gpe_energy).  The
    oracle does the same with energy()['mu'], active_indices and remap_psi: every grid must be identical and the
    final state agree at the 1000-step bound."""
    n_stage, steps, dt = 8, 100, 2e-3
    T = steps * dt
    base = I.config3(True).with_(nx=128, ny=128, nz=128, h=0.8, dt=dt, delta1=80.0, name="cfg3_staged_128")
    dd = (base.delta1 - base.delta0) / n_stage

    def stage_workload(s, v_cut):
        return base.with_(delta0=base.delta0 + s * dd, delta1=base.delta0 + (s + 1) * dd, t_ramp=T, v_cut=v_cut,
                          mask_mode=I.MASK_UNION)

    # stage 0 on BASELINE's own cut; reference state on the oracle side
    w = stage_workload(0, base.v_cut)
    box, pot, act, grid, sim = _make(P, w)
    psi = I.make_psi0(w, act)
    sim.set_psi_host(psi)
    ref = psi.copy()
    co = CO.COracle(box, pot, act, w.stencil)
    mu_gpu, mu_ref = sim.energy()["mu"], co.energy(w.g, 0.0, ref)["mu"]
    sizes = [act.size]
    keep = []                                               # sims of earlier stages stay alive until the end
    for s in range(n_stage):
        sim.time = 0.0
        sim.run_rk4(dt, steps)
        ref = co.run_rk4(w.g, 0.0, dt, steps, ref)
        assert rel_max(sim.get_psi_host(), ref) < 1e-9, s
        e_gpu, e_ref = sim.energy(), co.energy(w.g, T, ref)        # mu at the stage boundary, V at Delta_{s+1}
        assert abs(e_gpu["mu"] - e_ref["mu"]) < 1e-10 * abs(e_ref["mu"])
        if s == n_stage - 1:
            break
        cut_gpu, cut_ref = 5.0 * max(mu_gpu, e_gpu["mu"]), 5.0 * max(mu_ref, e_ref["mu"])
        mu_gpu, mu_ref = e_gpu["mu"], e_ref["mu"]
        # re-select: library on its own threshold, oracle on its own
        w_new = stage_workload(s + 1, cut_gpu)
        grid_new = P.Grid.from_workload(w_new)
        box_n, pot_n, act_n = oracle_objs(stage_workload(s + 1, cut_ref))
        assert np.array_equal(grid_new.active_indices(), act_n), s
        sim_new = P.Sim(grid_new, w_new.dtype, w_new.stencil, w_new.g)
        sim_new.remap_from(sim)
        ref = O.remap_psi(act, ref, act_n)
        assert np.array_equal(sim_new.get_psi_host() != 0, ref != 0)
        keep.append((sim, grid))
        sim, grid, w, act, pot = sim_new, grid_new, w_new, act_n, pot_n
        co = CO.COracle(box_n, pot_n, act_n, w.stencil)
        sizes.append(act_n.size)
    assert len(set(sizes)) > 1                              # the mask really followed the cloud
    assert abs(sim.norm() - co.norm(ref)) < 1e-10


@pytest.mark.parametrize("dtype", ["complex128", "complex64"])
def test_graph_replay_is_bit_identical(P, dtype):
    """Runs of 16 or more steps on small grids in a static potential replay a captured CUDA graph of 8 steps
    (gpe_run_rk4): same kernels, same parameters, same order, so the state is bit-identical to the one reached step
    by step; a ramped potential (parameters change every stage) takes the step-by-step path and agrees with it too."""
    w = I.config1().with_(dtype=dtype)
    box, pot, act, grid, sim = _make(P, w)
    psi = I.make_psi0(w, act).astype(sim.npdtype)
    sim.set_psi_host(psi)
    sim.run_rk4(w.dt, 43)                                   # 5 graph replays + 3 single steps
    got = sim.get_psi_host().copy()
    assert abs(sim.time - 43 * w.dt) < 1e-15
    sim.set_psi_host(psi)
    sim.time = 0.0
    for _ in range(43):
        sim.run_rk4(w.dt, 1)
    assert np.array_equal(sim.get_psi_host(), got)
    co = CO.COracle(box, pot, act, w.stencil)
    assert rel_max(got, co.run_rk4(w.g, 0.0, w.dt, 43, psi.astype(np.complex128))) < (1e-11 if dtype == "complex128" else 1e-4)
    # second run on the same sim reuses the graph; a changed dt rebuilds it
    sim.run_rk4(w.dt, 16)
    sim.run_rk4(0.5 * w.dt, 16)
    ref = co.run_rk4(w.g, 43 * w.dt, w.dt, 16, got.astype(np.complex128))
    ref = co.run_rk4(w.g, 59 * w.dt, 0.5 * w.dt, 16, ref)
    assert rel_max(sim.get_psi_host(), ref) < (1e-11 if dtype == "complex128" else 1e-4)
    # ramped dressed potential: no graph, still right
    wr = I.small_shell(24, 13, dtype).with_(delta0=14.0, delta1=22.0, t_ramp=0.05)
    box, pot, act, grid, sim = _make(P, wr)
    psi = I.make_psi0(wr, act).astype(sim.npdtype)
    sim.set_psi_host(psi)
    sim.run_rk4(wr.dt, 20)
    og = O.SparseGrid(box, act, 2)
    assert rel_max(sim.get_psi_host(), O.run_rk4(og, pot, wr.g, 0.0, wr.dt, 20, psi.astype(np.complex128), 13)) < (1e-11 if dtype == "complex128" else 1e-4)



@pytest.mark.parametrize("stencil", [13, 19])
def test_graph_replay_dressed_static_at_nonzero_t0_and_after_knob_changes(P, stencil):
    """gpe_run_rk4's graph path on the dressed potential: (a) Delta constant (delta0 == delta1) with the run starting
    at t0 != 0; (b) a ramp that has already ended at t0 (Delta(t) = delta1 from there on); (c) re-entry after
    gpe_sim_set_planes_per_block and, for the compact stencil, after gpe_sim_set_compact_weights -- each bit-identical
    to the same run taken one step per call (runs of one step never use the graph)."""
    def both_ways(sim, psi, t0, dt, n):
        sim.set_psi_host(psi)
        sim.time = t0
        sim.run_rk4(dt, n)
        got = sim.get_psi_host().copy()
        assert abs(sim.time - (t0 + n * dt)) < 1e-15
        sim.set_psi_host(psi)
        for k in range(n):
            sim.time = t0 + k * dt                          # step k of a run starts at t0 + k dt (a product, gpe.h)
            sim.run_rk4(dt, 1)
        assert np.array_equal(sim.get_psi_host(), got)
        return got

    w = I.small_shell(24, stencil)
    box, pot, act, grid, sim = _make(P, w)
    psi = I.make_psi0(w, act)
    a = both_ways(sim, psi, 0.37, w.dt, 19)                 # 2 replays + 3 single steps
    og = O.SparseGrid(box, act, 2)
    assert rel_max(a, O.run_rk4(og, pot, w.g, 0.37, w.dt, 19, psi, stencil)) < 1e-11
    sim.set_planes_per_block(5)                             # new work records: the graph is rebuilt, same numbers
    assert np.array_equal(both_ways(sim, psi, 0.37, w.dt, 19), a)
    if stencil == 19:
        sim.set_compact_weights(-4.2 / w.h ** 2, [0.4 / w.h ** 2] * 3, [0.15 / w.h ** 2] * 3, 0.0)
        b = both_ways(sim, psi, 0.37, w.dt, 16)
        assert not np.array_equal(b, a)
    # (b) the ramp 14 -> 22 ends at t = 0.05; from t0 = 0.06 on the potential is static at delta1
    wr = w.with_(delta0=14.0, delta1=22.0, t_ramp=0.05)
    box, pot, act, grid, sim = _make(P, wr)
    psi = I.make_psi0(wr, act)
    got = both_ways(sim, psi, 0.06, wr.dt, 17)
    og = O.SparseGrid(box, act, 2)
    assert rel_max(got, O.run_rk4(og, pot, wr.g, 0.06, wr.dt, 17, psi, stencil)) < 1e-11
    # the same sim inside the ramp (no graph), then after it again (the kept graph is still the right one)
    both_ways(sim, psi, 0.0, wr.dt, 17)
    assert np.array_equal(both_ways(sim, psi, 0.06, wr.dt, 17), got)


def test_sim_options_switch_between_bit_identical_forms(P):
    """gpe_sim_set_option (include/gpe.h): the graph replay and programmatic dependent launch change how the launches
    are issued, not what they compute; bad arguments are refused."""
    w = I.config1()
    box, pot, act, grid, sim = _make(P, w)
    psi = I.make_psi0(w, act)
    res = []
    for graph, pdl in ((1, 1), (0, 1), (1, 0), (0, 0), (1, 1)):
        sim.set_option(P.OPT_RK4_GRAPH, graph)
        sim.set_option(P.OPT_PDL, pdl)
        sim.set_psi_host(psi)
        sim.time = 0.0
        n0 = sim.kernel_launches
        sim.run_rk4(w.dt, 24)
        res.append(sim.get_psi_host().copy())
        assert sim.kernel_launches - n0 == 24 * 4 + 1       # + the unpack of the read-back: replayed launches are counted too
    for r in res[1:]:
        assert np.array_equal(r, res[0])
    for opt, val in ((7, 1), (-1, 0), (P.OPT_PDL, 2), (P.OPT_FUSED_K1, -1)):
        with pytest.raises(P.GpeError) as e:
            sim.set_option(opt, val)
        assert e.value.code == -1
