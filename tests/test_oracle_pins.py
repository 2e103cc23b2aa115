"""Pins for the CPU oracle: it is checked against what the paper and the mathematics fix,
never against itself.  P# labels follow DESIGN.md "Oracle pins".  All CPU, no GPU.
"""
import json
import math
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import gpe_oracle as O
import gpe_inputs as I

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def full_box_grid(nx, ny, nz, h, radius=2):
    box = O.Box(nx, ny, nz, h)
    return box, O.SparseGrid(box, np.arange(nx * ny * nz, dtype=np.int64), radius)


def sine_mode(nx, ny, nz, m):
    ax = [np.sin(math.pi * m[d] * (np.arange(n) + 1) / (n + 1)) for d, n in enumerate((nx, ny, nz))]
    return (ax[0][:, None, None] * ax[1][None, :, None] * ax[2][None, None, :]).astype(np.complex128)


# ---- P1: exact discrete eigenvalues of sine modes, 7-point, Dirichlet box --------------
@pytest.mark.parametrize("m", [(1, 1, 1), (2, 3, 1), (5, 1, 4)])
def test_P1_sine_modes_7pt(m):
    nx, ny, nz, h = 7, 9, 8, 0.3
    box, grid = full_box_grid(nx, ny, nz, h)
    psi = sine_mode(nx, ny, nz, m).ravel() * (1 + 0.5j)
    lam = sum(-(4.0 / h ** 2) * math.sin(0.5 * math.pi * m[d] / (n + 1)) ** 2
              for d, n in enumerate((nx, ny, nz)))
    t = O.apply_T(grid, psi, 7)
    assert np.max(np.abs(t - (-0.5 * lam) * psi)) < 1e-12 * abs(lam)


# ---- P2: 13-point symbol in the interior, and the exact outer-layer defect -------------
def test_P2_sine_modes_13pt_symbol_and_defect():
    nx, ny, nz, h = 9, 8, 10, 0.37
    m = (2, 1, 3)
    box, grid = full_box_grid(nx, ny, nz, h)
    psi3 = sine_mode(nx, ny, nz, m)
    th = [math.pi * m[d] / (n + 1) for d, n in enumerate((nx, ny, nz))]
    sym = [-(1.0 / h ** 2) * (2.5 - (8.0 / 3.0) * math.cos(t) + (1.0 / 6.0) * math.cos(2 * t)) for t in th]
    lap = -2.0 * O.apply_T(grid, psi3.ravel(), 13).reshape(nx, ny, nz)
    expect = sum(sym) * psi3
    inner = (slice(1, -1),) * 3
    assert np.max(np.abs(lap[inner] - expect[inner])) < 1e-11 * abs(sum(sym))
    # outermost layer: zero extension drops the analytic image psi(-2) = -sin(theta) (and the
    # mirror one at n+1); the stencil weight there is -1/12, so lap_zero_ext = lap_nat + psi_nat/12h^2.
    sx = np.sin(th[0] * (np.arange(-2, nx + 2) + 1))      # analytic extension along x
    fy = np.sin(th[1] * (np.arange(ny) + 1))
    fz = np.sin(th[2] * (np.arange(nz) + 1))
    for i, ghost in ((0, sx[0]), (nx - 1, sx[-1])):      # sx[0] = psi(-2), sx[-1] = psi(nx+1)
        want = expect[i, 1:-1, 1:-1] + (1.0 / (12 * h * h)) * ghost * fy[1:-1, None] * fz[None, 1:-1]
        assert np.max(np.abs(lap[i, 1:-1, 1:-1] - want)) < 1e-11 * abs(sum(sym))
    assert abs(sx[0] + math.sin(th[0])) < 1e-15


# ---- 1-D reference operators built independently (dense matrices + library eigh) -------
def lap1d(n, h, stencil):
    w = {7: [-2.0, 1.0], 13: [-2.5, 4.0 / 3.0, -1.0 / 12.0]}[stencil]
    d = np.zeros((n, n))
    for i in range(n):
        for s in range(-(len(w) - 1), len(w)):
            if 0 <= i + s < n:
                d[i, i + s] = w[abs(s)] / h ** 2
    return d


def ho_ground_state_1d(n, h, stencil):
    x = (np.arange(n) - 0.5 * (n - 1)) * h
    hm = -0.5 * lap1d(n, h, stencil) + np.diag(0.5 * x * x)
    e, v = np.linalg.eigh(hm)
    return e[0], v[:, 0]


# ---- P3 / P4: harmonic-trap ground-state energy 3/2 at g = 0, at the stencil's order ---
@pytest.mark.parametrize("stencil,closed", [(7, lambda h: 1.5 - 3 * h ** 2 / 32),
                                            (13, lambda h: 1.5 - h ** 4 / 32)])
def test_P3_P4_harmonic_ground_state(stencil, closed):
    n, h = 48, 0.25
    e1, v1 = ho_ground_state_1d(n, h, stencil)
    box, grid = full_box_grid(n, n, n, h)
    psi = (v1[:, None, None] * v1[None, :, None] * v1[None, None, :]).ravel().astype(np.complex128)
    psi /= math.sqrt(h ** 3 * np.sum(np.abs(psi) ** 2))
    pot = O.Potential(kind=O.HARMONIC)
    en = O.energy(grid, pot, 0.0, 0.0, psi, stencil)
    hp = O.apply_H(grid, pot, 0.0, 0.0, psi, stencil)
    assert abs(en["norm"] - 1.0) < 1e-13
    assert np.max(np.abs(hp - 3 * e1 * psi)) < 1e-11 * np.max(np.abs(psi))
    assert abs(en["total"] - 3 * e1) < 1e-12 and abs(en["mu"] - 3 * e1) < 1e-12
    # closed forms: 3/2 - 3h^2/32 + O(h^4) (2nd order), 3/2 - h^4/32 + O(h^6) (4th order)
    tol = 3e-5 if stencil == 7 else 4e-6   # O(h^4) resp. O(h^6) remainder; the h^2 / h^4 terms are 5.9e-3 / 1.2e-4
    assert abs(en["total"] - closed(h)) < tol
    assert abs(en["total"] - 1.5) > 10 * tol if stencil == 7 else True


def test_P3_order_of_convergence():
    # the 1-D references converge at order 2 / 4; the 3-D oracle was tied to them above
    for stencil, order in ((7, 2), (13, 4)):
        e = [ho_ground_state_1d(int(round(12 / h)), h, stencil)[0] for h in (0.5, 0.25)]
        ratio = (e[0] - 0.5) / (e[1] - 0.5)
        assert abs(math.log2(ratio) - order) < 0.15


def test_P3_imaginary_time_converges_to_ground_state():
    n, h = 20, 0.6
    box, grid = full_box_grid(n, n, n, h)
    pot = O.Potential(kind=O.HARMONIC)
    e1, v1 = ho_ground_state_1d(n, h, 7)
    rng = np.random.default_rng(0)
    x = O.coords(n, h)
    g0 = np.exp(-0.35 * x * x)
    psi = (g0[:, None, None] * g0[None, :, None] * g0[None, None, :]).ravel() * (1 + 0.1 * rng.normal(size=n ** 3))
    psi = psi.astype(np.complex128)
    psi /= math.sqrt(O.norm(grid, psi))
    last = O.energy(grid, pot, 0.0, 0.0, psi, 7)["total"]
    for _ in range(20):      # dt * lambda_max ~ 0.65: stable forward Euler
        psi = O.run_imag(grid, pot, 0.0, 0.0, 0.01, 25, psi, 7)
        assert abs(O.norm(grid, psi) - 1.0) < 1e-13
        e = O.energy(grid, pot, 0.0, 0.0, psi, 7)["total"]
        assert e <= last + 1e-13      # monotone for small dt
        last = e
    assert abs(last - 3 * e1) < 2e-4
    assert last > 3 * e1 - 1e-12


# ---- P5: brute-force operator matrices from Kronecker products, rows/cols deleted ------
@pytest.mark.parametrize("stencil", [7, 13])
@pytest.mark.parametrize("dims", [(6, 6, 6), (5, 6, 7)])
def test_P5_kronecker_submatrix(stencil, dims):
    nx, ny, nz = dims
    h = 0.7
    eye = np.eye
    lap = (np.kron(np.kron(lap1d(nx, h, stencil), eye(ny)), eye(nz))
           + np.kron(np.kron(eye(nx), lap1d(ny, h, stencil)), eye(nz))
           + np.kron(np.kron(eye(nx), eye(ny)), lap1d(nz, h, stencil)))
    for seed, p in ((1, 0.5), (2, 0.85), (3, 0.15)):
        act = I.random_mask_lin(seed, nx, ny, nz, p)
        tmat = -0.5 * lap[np.ix_(act, act)]           # remove rows and columns
        grid = O.SparseGrid(O.Box(nx, ny, nz, h), act, 2)
        for k in range(0, act.size, max(1, act.size // 7)):
            e = np.zeros(act.size, np.complex128)
            e[k] = 1.0
            assert np.max(np.abs(O.apply_T(grid, e, stencil) - tmat[:, k])) < 1e-13
        psi = I.random_psi(seed, act.size)
        assert np.max(np.abs(O.apply_T(grid, psi, stencil) - tmat @ psi)) < 1e-12 * np.max(np.abs(tmat)) * 8


# ---- P6: sparse operator == dense shifted-slice stencil -------------------------------
@pytest.mark.parametrize("stencil", [7, 13])
def test_P6_sparse_equals_dense(stencil):
    nx, ny, nz, h = 9, 7, 11, 0.4
    box = O.Box(nx, ny, nz, h)
    for p in (1.0, 0.6):
        act = np.arange(nx * ny * nz, dtype=np.int64) if p == 1.0 else I.random_mask_lin(7, nx, ny, nz, p)
        grid = O.SparseGrid(box, act, 2)
        psi = I.random_psi(5, act.size)
        dense = np.zeros(nx * ny * nz, np.complex128)
        dense[act] = psi
        mask = np.zeros(nx * ny * nz, bool)
        mask[act] = True
        td = O.dense_apply_T(box, mask.reshape(nx, ny, nz), dense.reshape(nx, ny, nz), stencil).ravel()[act]
        assert np.max(np.abs(O.apply_T(grid, psi, stencil) - td)) < 1e-12 * np.max(np.abs(td))


# ---- P7: sign of i -- psi(t) = exp(-i E t) psi(0)  (Eq. 2) -----------------
def test_P7_phase_rotation_sign():
    n, h = 16, 0.7
    box, grid = full_box_grid(n, n, n, h)
    e1, v1 = ho_ground_state_1d(n, h, 7)
    psi0 = (v1[:, None, None] * v1[None, :, None] * v1[None, None, :]).ravel().astype(np.complex128)
    pot = O.Potential(kind=O.HARMONIC)
    dt, ns = 2e-3, 50
    psi = O.run_rk4(grid, pot, 0.0, 0.0, dt, ns, psi0, 7)
    ph = np.angle(np.vdot(psi0, psi))
    assert abs(ph - (-3 * e1 * dt * ns)) < 1e-9


# ---- P8: RK4 tableau -- exact amplification factor of an eigenmode, and order 4 --------
def test_P8_amplification_factor_and_order():
    nx, ny, nz, h = 6, 5, 7, 0.5
    box, grid = full_box_grid(nx, ny, nz, h)
    m = (2, 1, 3)
    psi = sine_mode(nx, ny, nz, m).ravel()
    lam = -0.5 * sum(-(4.0 / h ** 2) * math.sin(0.5 * math.pi * m[d] / (n + 1)) ** 2
                     for d, n in enumerate((nx, ny, nz)))
    pot = O.Potential(kind=O.HARMONIC, ax=0.0, ay=0.0, az=0.0)
    dt = 0.02
    z = lam * dt
    out = O.rk4_step(grid, pot, 0.0, 0.0, dt, psi, 7)
    rz = 1 - 1j * z - z * z / 2 + 1j * z ** 3 / 6 + z ** 4 / 24
    assert np.max(np.abs(out - rz * psi)) < 1e-13
    assert abs(abs(rz) ** 2 - (1 - z ** 6 / 72 + z ** 8 / 576)) < 1e-14
    # order: linear problem on a random mask, exact propagator from library eigh
    act = I.random_mask_lin(4, 6, 6, 6, 0.7)
    g2 = O.SparseGrid(O.Box(6, 6, 6, 0.5), act, 2)
    lap = (np.kron(np.kron(lap1d(6, 0.5, 13), np.eye(6)), np.eye(6))
           + np.kron(np.kron(np.eye(6), lap1d(6, 0.5, 13)), np.eye(6))
           + np.kron(np.kron(np.eye(6), np.eye(6)), lap1d(6, 0.5, 13)))
    pot2 = O.Potential(kind=O.HARMONIC, ax=1.0, ay=2.0, az=0.5)
    hmat = -0.5 * lap[np.ix_(act, act)] + np.diag(O.potential_at(g2.box, pot2, act, 0.0))
    ev, U = np.linalg.eigh(hmat)
    p0 = I.random_psi(9, act.size)
    T = 0.2
    exact = U @ (np.exp(-1j * ev * T) * (U.conj().T @ p0))
    errs = []
    for ns in (40, 80):
        p = O.run_rk4(g2, pot2, 0.0, 0.0, T / ns, ns, p0, 13)
        errs.append(np.max(np.abs(p - exact)))
    assert 13.0 < errs[0] / errs[1] < 19.0


def test_P8_norm_and_energy_conservation_nonlinear():
    w = I.small_shell(24, 7)
    box = O.Box(w.nx, w.ny, w.nz, w.h)
    pot = O.Potential(w.kind, w.ax, w.ay, w.az, w.delta0, w.delta1, w.t_ramp, w.omega)
    act = O.active_indices(box, pot, w.v_cut)
    grid = O.SparseGrid(box, act, 2)
    psi = I.make_psi0(w, act)
    e0 = O.energy(grid, pot, w.g, 0.0, psi, 7)
    drift = []
    for dt in (2e-3, 1e-3):
        p = O.run_rk4(grid, pot, w.g, 0.0, dt, int(round(0.02 / dt)), psi, 7)
        e1 = O.energy(grid, pot, w.g, 0.0, p, 7)
        drift.append((abs(e1["norm"] - 1.0), abs(e1["total"] - e0["total"])))
    assert drift[1][0] < 1e-9 and drift[1][1] < 1e-7 * abs(e0["total"])
    assert drift[0][0] / max(drift[1][0], 1e-300) > 8      # norm drift ~ dt^5 per unit time
    assert drift[0][1] / max(drift[1][1], 1e-300) > 8      # energy drift ~ dt^4 or better


# ---- P9: the memory-optimised RK form ---------------------
def modified_tableau(a, b):
    """a*, b* from a standard explicit Butcher tableau via PAPER.md Eq. A4-A7 (dt = 1)."""
    n = len(b)
    M = [[Fraction(0)] * n for _ in range(n)]
    for i in range(n):
        M[i][0] = Fraction(1)
        for j in range(i):
            M[i][j + 1] = Fraction(a[i][j])
    # invert lower-triangular M:  K = Minv Y   with K = (y0, k1..k_{n-1}), Y = (y1..yn)
    Minv = [[Fraction(0)] * n for _ in range(n)]
    for c in range(n):
        for r in range(n):
            rhs = Fraction(1 if r == c else 0) - sum(M[r][k] * Minv[k][c] for k in range(r))
            Minv[r][c] = rhs / M[r][r]
    astar = []
    for i in range(1, n):            # y^(i+1) = y0 + sum_{j<i} a_{i+1,j} k_j + a_{i+1,i} k_i
        row = [Fraction(0)] * i
        coef = [Fraction(1)] + [Fraction(a[i][j]) for j in range(i - 1)]
        for j, cj in enumerate(coef):
            for c in range(i):
                row[c] += cj * Minv[j][c]
        astar.append(row)
    coef = [Fraction(1)] + [Fraction(b[j]) for j in range(n - 1)]
    bstar = [Fraction(0)] * n
    for j, cj in enumerate(coef):
        for c in range(n):
            bstar[c] += cj * Minv[j][c]
    return astar, bstar


def test_P9_modified_tableau_matches_paper():
    gold = json.load(open(os.path.join(GOLD, "paper_values.json")))
    F = Fraction
    a4 = [[], [F(1, 2)], [0, F(1, 2)], [0, 0, 1]]
    b4 = [F(1, 6), F(1, 3), F(1, 3), F(1, 6)]
    astar, bstar = modified_tableau(a4, b4)
    assert bstar == [F(s) for s in gold["rk4_b_star"]["value"]]
    for i, row in enumerate(gold["rk4_a_star"]["value"]):
        assert astar[i] == [F(v) for v in row[: i + 1]]
    a3 = [[], [F(1, 3)], [0, F(2, 3)]]
    b3 = [F(1, 4), 0, F(3, 4)]
    astar3, bstar3 = modified_tableau(a3, b3)
    assert bstar3 == [F(s) for s in gold["rkhe3_b_star"]["value"]]
    for i, row in enumerate(gold["rkhe3_a_star"]["value"]):
        assert astar3[i] == [F(v) for v in row[: i + 1]]


def test_P9_stage_form_equals_textbook_rk4():
    """The S1-S4 stage form the CUDA path uses == textbook RK4, via the oracle's H."""
    w = I.small_shell(20, 13)
    box = O.Box(w.nx, w.ny, w.nz, w.h)
    pot = O.Potential(w.kind, w.ax, w.ay, w.az, 5.0, 20.0, 0.01, w.omega)
    act = O.active_indices(box, pot, w.v_cut, O.MASK_UNION)
    grid = O.SparseGrid(box, act, 2)
    y0 = I.make_psi0(w, act)
    t, dt, g = 0.003, 1e-3, w.g
    f = lambda tt, y: -1j * O.apply_H(grid, pot, g, tt, y, 13)
    y2 = y0 + 0.5 * dt * f(t, y0)
    y3 = y0 + 0.5 * dt * f(t + 0.5 * dt, y2)
    p = -y0 / 3 + y2 / 3 + 2 * y3 / 3
    y4 = y0 + dt * f(t + 0.5 * dt, y3)
    ynew = p + y4 / 3 + (dt / 6) * f(t + dt, y4)
    ref = O.rk4_step(grid, pot, g, t, dt, y0, 13)
    assert np.max(np.abs(ynew - ref)) < 1e-14 * np.max(np.abs(ref))


# ---- P10: Hermiticity of the reduced operator (principal sub-matrix) ------
@pytest.mark.parametrize("stencil", [7, 13])
def test_P10_hermitian(stencil):
    act = I.random_mask_lin(12, 8, 9, 7, 0.55)
    grid = O.SparseGrid(O.Box(8, 9, 7, 0.3), act, 2)
    a, b = I.random_psi(1, act.size), I.random_psi(2, act.size)
    lhs = np.vdot(a, O.apply_T(grid, b, stencil))
    rhs = np.vdot(O.apply_T(grid, a, stencil), b)
    assert abs(lhs - rhs) < 1e-11 * abs(lhs)


# ---- P11: stage times c = 0, 1/2, 1/2, 1 -- one-point mask = scalar ODE ----------------
def test_P11_one_point_mask_scalar_ode():
    from scipy.integrate import quad
    box = O.Box(5, 5, 5, 0.5)
    pot = O.Potential(kind=O.DRESSED, ax=1.0, ay=1.0, az=1.0, delta0=0.0, delta1=6.0, t_ramp=0.5, omega=1.5)
    lin = np.array([(1 * 5 + 3) * 5 + 4], dtype=np.int64)
    grid = O.SparseGrid(box, lin, 2)
    g, stencil = 3.0, 13
    x, y, z = (O.coords(5, 0.5)[i] for i in (1, 3, 4))
    u = 0.5 * (x * x + y * y + z * z)
    vt = lambda t: math.sqrt((u - (0.0 + 6.0 * min(max(t / 0.5, 0.0), 1.0))) ** 2 + 1.5 ** 2) - 1.5
    c = -0.5 * 3 * (-2.5) / 0.5 ** 2               # diagonal of T for the 13-point stencil
    psi0 = np.array([0.8 - 0.3j])
    T, ns = 0.4, 400        # z = dt*(c+V+g|psi|^2) ~ 0.02: RK4 phase error z^5/120 per step ~ 1e-8 total
    psi = O.run_rk4(grid, pot, g, 0.05, T / ns, ns, psi0, stencil)
    integral = quad(vt, 0.05, 0.05 + T, epsabs=1e-13, epsrel=1e-13)[0]
    exact = psi0 * np.exp(-1j * (integral + (g * abs(psi0[0]) ** 2 + c) * T))
    assert abs(psi[0] - exact[0]) < 5e-8            # O(dt^4); wrong stage times give O(dt) ~ 1e-2
    wrong = psi0 * np.exp(-1j * (vt(0.05) * T + (g * abs(psi0[0]) ** 2 + c) * T))
    assert abs(wrong[0] - exact[0]) > 1e-2


# ---- P12: layout -- counts, halo, tile tables ------------------------------------------
def _wl_objects(w):
    box = O.Box(w.nx, w.ny, w.nz, w.h, w.center)
    pot = O.Potential(w.kind, w.ax, w.ay, w.az, w.delta0, w.delta1, w.t_ramp, w.omega)
    return box, pot


def test_P12_counts_fixture_config1_config2():
    gold = json.load(open(os.path.join(GOLD, "paper_values.json")))
    assert gold["block_tile_points"]["value"] - gold["block_interior_points"]["value"] == gold["block_halo_points"]["value"] == 10 ** 3 - 8 ** 3
    counts = json.load(open(os.path.join(GOLD, "counts.json")))
    for w in (I.config1(), I.config2()):
        box, pot = _wl_objects(w)
        act = O.active_indices(box, pot, w.v_cut, w.mask_mode, check_knife_edge=True)
        st = O.stored_indices(box, act, w.halo_width)
        assert act.size == counts[w.name]["n_active"]
        assert st.size == counts[w.name]["n_stored"]
    # the survey's independent count script gave the same numbers
    sv = {"cfg1_harmonic_48": (67080, 9888), "cfg2_bubble_256": (1215760, 418000), "cfg3a_ramp_union_512": (38495288, 922496),
          "cfg3b_ramp_final_512": (9730864, 1671856), "cfg4_ellipsoid_1024_c128": (31523416, 5942744)}   # SURVEY.md:237-241
    for name, (na, halo) in sv.items():
        assert (counts[name]["n_active"], counts[name]["n_stored"]) == (na, na + halo), name


def test_P12_mask_is_ball_for_harmonic():
    w = I.config1()
    box, pot = _wl_objects(w)
    act = O.active_indices(box, pot, w.v_cut)
    ix, iy, iz = O.unravel(box, act)
    c = O.coords(48, 0.25)
    r2 = c[ix] ** 2 + c[iy] ** 2 + c[iz] ** 2
    assert np.all(r2 < 40.0)
    allr2 = (c[:, None, None] ** 2 + c[None, :, None] ** 2 + c[None, None, :] ** 2).ravel()
    assert act.size == int(np.sum(allr2 < 40.0 - 1e-9)) == int(np.sum(allr2 < 40.0 + 1e-9))
    assert abs(c[0] + 5.875) < 1e-15 and abs(c[23] + 0.125) < 1e-15     # symmetric, no point at 0


def test_P12_union_mask_is_union_over_ramp():
    w = I.small_shell(24, 7)
    box, _ = _wl_objects(w)
    pot = O.Potential(O.DRESSED, 1.0, 1.2, 0.9, 0.0, 20.0, 1.0, 6.0)
    uni = set(O.active_indices(box, pot, w.v_cut, O.MASK_UNION).tolist())
    acc = set()
    for d in np.linspace(0.0, 20.0, 401):
        p = O.Potential(O.DRESSED, 1.0, 1.2, 0.9, d, d, 0.0, 6.0)
        acc |= set(O.active_indices(box, p, w.v_cut, O.MASK_AT_DELTA0).tolist())
    assert acc <= uni and len(uni - acc) <= 0.002 * len(uni)


def test_P12_halo_resolves_every_neighbour():
    w = I.small_shell(24, 13)
    box, pot = _wl_objects(w)
    act = O.active_indices(box, pot, w.v_cut)
    st = set(O.stored_indices(box, act, 2).tolist())
    ix, iy, iz = O.unravel(box, act)
    for (dx, dy, dz) in [(s * a, s * b, s * c) for s in (-2, -1, 1, 2) for (a, b, c) in ((1, 0, 0), (0, 1, 0), (0, 0, 1))]:
        jx, jy, jz = ix + dx, iy + dy, iz + dz
        inside = (0 <= jx) & (jx < box.nx) & (0 <= jy) & (jy < box.ny) & (0 <= jz) & (jz < box.nz)
        lin = (jx * box.ny + jy) * box.nz + jz
        assert all(int(l) in st for l in lin[inside])
    assert set(act.tolist()) <= st


@pytest.mark.parametrize("zt", [32, 5])
def test_P12_tile_layout_invariants(zt):
    w = I.small_shell(24, 13)
    box, pot = _wl_objects(w)
    act = O.active_indices(box, pot, w.v_cut)
    L = O.tile_layout(box, act, 8, 8, zt)
    perm = L["storage_to_canonical"]
    assert np.array_equal(np.sort(perm), np.arange(act.size))
    # decode every slab lane back to a linear index and compare with the permuted active list
    lin = []
    for k in range(L["n_tiles"]):
        i, j = L["tile_xy"][k]
        for z in range(L["tile_zlo"][k], L["tile_zhi"][k]):
            e = L["tile_entry_base"][k] + z - L["tile_zlo"][k]
            m = int(L["slab_mask"][e])
            assert L["slab_base"][e] == len(lin)
            for b in range(64):
                if m >> b & 1:
                    lin.append(((i * 8 + b // 8) * box.ny + (j * 8 + b % 8)) * box.nz + z)
    assert np.array_equal(np.asarray(lin), act[perm])
    # work items cover each non-empty slab exactly once, never exceed zt, never hold an empty slab
    seen = set()
    for t, z0, nz in zip(L["wi_tile"], L["wi_z0"], L["wi_nz"]):
        assert 1 <= nz <= zt
        for z in range(z0, z0 + nz):
            e = L["tile_entry_base"][t] + z - L["tile_zlo"][t]
            assert L["slab_mask"][e] != 0 and (t, z) not in seen
            seen.add((int(t), int(z)))
    assert len(seen) == int(np.count_nonzero(L["slab_mask"]))
    # neighbour table is symmetric
    for k in range(L["n_tiles"]):
        for q, qq in ((0, 1), (1, 0), (2, 3), (3, 2)):
            n = L["tile_nbr"][k, q]
            if n >= 0:
                assert L["tile_nbr"][n, qq] == k


def test_uniform01_is_layout_independent_and_uniform():
    lin = np.arange(200000, dtype=np.int64)
    u = I.uniform01(3, lin)
    assert 0.0 <= u.min() and u.max() < 1.0 and abs(u.mean() - 0.5) < 5e-3
    p = np.random.default_rng(0).permutation(lin.size)
    assert np.array_equal(I.uniform01(3, lin[p]), u[p])
    assert not np.array_equal(I.uniform01(4, lin), u)


# ---- P13: the paper's own imaginary-time scheme: D K K D, renormalise -----------------
def _kron_T(nx, ny, nz, h, stencil, act):
    eye = np.eye
    lap = (np.kron(np.kron(lap1d(nx, h, stencil), eye(ny)), eye(nz))
           + np.kron(np.kron(eye(nx), lap1d(ny, h, stencil)), eye(nz))
           + np.kron(np.kron(eye(nx), eye(ny)), lap1d(nz, h, stencil)))
    return -0.5 * lap[np.ix_(act, act)]


@pytest.mark.parametrize("stencil", [7, 13])
def test_P13_split_step_is_DKKD_matrix_at_g0(stencil):
    """g = 0: one iteration is the matrix M = D (1 - dt/2 T)^2 D, D = diag exp(-V dt/2), applied and
    normalised; T from Kronecker products with rows / columns deleted, V from the coordinates."""
    nx, ny, nz, h, dt = 6, 5, 7, 0.6, 0.02
    act = I.random_mask_lin(11, nx, ny, nz, 0.7)
    box = O.Box(nx, ny, nz, h)
    grid = O.SparseGrid(box, act, 2)
    pot = O.Potential(kind=O.HARMONIC, ax=1.0, ay=2.0, az=0.5)
    ix, iy, iz = act // (ny * nz), (act // nz) % ny, act % nz
    x, y, z = (ix - 0.5 * (nx - 1)) * h, (iy - 0.5 * (ny - 1)) * h, (iz - 0.5 * (nz - 1)) * h
    d = np.exp(-0.5 * dt * 0.5 * (1.0 * x * x + 2.0 * y * y + 0.5 * z * z))
    k = np.eye(act.size) - 0.5 * dt * _kron_T(nx, ny, nz, h, stencil, act)
    m = np.diag(d) @ k @ k @ np.diag(d)
    assert np.max(np.abs(m - m.T)) < 1e-14                      # symmetric: a power iteration
    psi = I.random_psi(12, act.size)
    want = m @ psi
    want = want / math.sqrt(h ** 3 * np.sum(np.abs(want) ** 2))
    got = O.imag_split_step(grid, pot, 0.0, 0.0, dt, psi, stencil)
    assert np.max(np.abs(got - want)) < 1e-13 * np.max(np.abs(want)) * 10
    # fixed point = top eigenvector of M
    ev, evec = np.linalg.eigh(m)
    top = evec[:, -1] * np.sign(evec[np.argmax(np.abs(evec[:, -1])), -1])
    top = top / math.sqrt(h ** 3 * np.sum(top ** 2))
    psi = np.abs(psi.real).astype(np.complex128) + 0.1
    psi = O.run_imag_split(grid, pot, 0.0, 0.0, dt, 4000, psi, stencil)
    assert np.max(np.abs(psi - top)) < 1e-9 * np.max(np.abs(top))


def test_P13_split_scheme_ground_state_energy_error_is_second_order_in_dt():
    """Symmetric splitting: the energy of the fixed point differs from the discrete ground-state energy by
    O(dt^2) (the first-order term cancels between the two half steps); halving dt divides the error by 4."""
    n, h = 10, 0.7
    box, grid = full_box_grid(n, n, n, h)
    act = np.arange(n ** 3)
    pot = O.Potential(kind=O.HARMONIC)
    e1, _ = ho_ground_state_1d(n, h, 7)
    x = O.coords(n, h)
    v = 0.5 * (x[:, None, None] ** 2 + x[None, :, None] ** 2 + x[None, None, :] ** 2).ravel()
    tm = _kron_T(n, n, n, h, 7, act)
    errs = []
    for dt in (0.08, 0.04):
        d = np.exp(-0.5 * dt * v)
        k = np.eye(n ** 3) - 0.5 * dt * tm
        m = (d[:, None] * (k @ k)) * d[None, :]
        ev, evec = np.linalg.eigh(m)
        top = np.abs(evec[:, -1]).astype(np.complex128)
        top /= math.sqrt(O.norm(grid, top))
        # the oracle's iteration has that fixed point ...
        assert np.max(np.abs(O.imag_split_step(grid, pot, 0.0, 0.0, dt, top, 7) - top)) < 1e-12
        # ... whose energy is off by O(dt^2)
        errs.append(O.energy(grid, pot, 0.0, 0.0, top, 7)["total"] - 3 * e1)
    assert errs[0] > errs[1] > 0
    assert 3.5 < errs[0] / errs[1] < 4.5


def test_P13_linearised_interaction_factor():
    """exp(-g|psi|^2 dt/2) approximated as 1 - g|psi|^2 dt/2: the oracle's factor differs from the
    exponential one by x^2/2 - x^3/6 + ... with x = g |psi|^2 dt / 2, point by point."""
    w = I.small_shell(24, 7)
    box = O.Box(w.nx, w.ny, w.nz, w.h, w.center)
    pot = O.Potential(w.kind, w.ax, w.ay, w.az, w.delta0, w.delta1, w.t_ramp, w.omega)
    act = O.active_indices(box, pot, w.v_cut, w.mask_mode)
    grid = O.SparseGrid(box, act, 1)
    psi = I.make_psi0(w, act)
    g, dt = 3.0e4, 0.01
    x = g * np.abs(psi) ** 2 * dt / 2
    assert 0.01 < x.max() < 0.5
    exact = psi * np.exp(-0.5 * dt * O.potential_at(box, pot, act, 0.0)) * np.exp(-x)
    lin = O.diag_propagator(grid, pot, g, 0.0, dt, psi)
    ratio = lin / exact                                        # = (1 - x) e^{x} = 1 - x^2/2 - x^3/3 - ...
    assert np.max(np.abs(ratio - (1 - x) * np.exp(x))) < 1e-14
    assert np.all(ratio.real <= 1.0) and np.max(np.abs(1 - ratio.real - x ** 2 / 2)) < x.max() ** 3


# ---- P14: re-gridding -----------------------------------------------------------------------
def test_P14_remap_is_restriction_and_zero_extension():
    """What the remap is fixed by: on a dense array it is "scatter the old values into the box, read the new
    points" (zero where nothing was scattered); shared points keep their value, round trips lose exactly the
    points that were dropped, and the norm splits into kept + dropped."""
    nx, ny, nz = 7, 6, 9
    a = I.random_mask_lin(21, nx, ny, nz, 0.5)
    b = I.random_mask_lin(22, nx, ny, nz, 0.6)
    psi = I.random_psi(23, a.size)
    dense = np.zeros(nx * ny * nz, np.complex128)
    dense[a] = psi
    got = O.remap_psi(a, psi, b)
    assert np.array_equal(got, dense[b])
    back = O.remap_psi(b, got, a)
    shared = np.isin(a, b)
    assert np.array_equal(back[shared], psi[shared]) and np.all(back[~shared] == 0)
    assert abs(np.sum(np.abs(got) ** 2) + np.sum(np.abs(psi[~shared]) ** 2) - np.sum(np.abs(psi) ** 2)) < 1e-12
    assert O.remap_psi(a, psi, np.zeros(0, np.int64)).size == 0
    assert np.all(O.remap_psi(np.zeros(0, np.int64), np.zeros(0, np.complex128), b) == 0)


# ---- P15: Heun's third-order method (RKHE3, A8-A9) ------------------------------------------------
def test_P15_rkhe3_amplification_factor_and_stage_form():
    """g = 0, static V: on an eigenvector of H one step multiplies by R(z) = 1 + z + z^2/2 + z^3/6, z = -i E dt
    (any third-order three-stage method); and the paper's stage-state form (Eq. A6-A9) gives the same step."""
    n, h = 12, 0.6
    box, grid = full_box_grid(n, n, n, h)
    pot = O.Potential(kind=O.HARMONIC)
    e1, v1 = ho_ground_state_1d(n, h, 7)
    psi = (v1[:, None, None] * v1[None, :, None] * v1[None, None, :]).ravel().astype(np.complex128)
    dt = 0.05
    z = -1j * 3 * e1 * dt
    got = O.rkhe3_step(grid, pot, 0.0, 0.0, dt, psi, 7)
    assert np.max(np.abs(got - (1 + z + z * z / 2 + z ** 3 / 6) * psi)) < 1e-13
    # stage-state form with a ramped potential and g > 0 (stage times t, t + dt/3, t + 2dt/3)
    w = I.small_shell(20, 13)
    box = O.Box(w.nx, w.ny, w.nz, w.h)
    pot = O.Potential(w.kind, w.ax, w.ay, w.az, 5.0, 20.0, 0.01, w.omega)
    act = O.active_indices(box, pot, w.v_cut, O.MASK_UNION)
    grid = O.SparseGrid(box, act, 2)
    y0 = I.make_psi0(w, act)
    t, dt, g = 0.003, 1e-3, w.g
    f = lambda tt, y: -1j * O.apply_H(grid, pot, g, tt, y, 13)
    y2 = y0 + dt / 3 * f(t, y0)                               # a* row 1: [1]
    y3 = y0 + 2 * dt / 3 * f(t + dt / 3, y2)                  # a* row 2: [1, 0]
    ynew = y0 / 4 + 3 * y2 / 4 + 3 * dt / 4 * f(t + 2 * dt / 3, y3)   # b* = [1/4, 3/4, 0], b_3 = 3/4
    ref = O.rkhe3_step(grid, pot, g, t, dt, y0, 13)
    assert np.max(np.abs(ynew - ref)) < 1e-14 * np.max(np.abs(ref))


def test_P15_rkhe3_is_third_order():
    w = I.small_shell(20, 7)
    box = O.Box(w.nx, w.ny, w.nz, w.h)
    pot = O.Potential(w.kind, w.ax, w.ay, w.az, w.delta0, w.delta1, w.t_ramp, w.omega)
    act = O.active_indices(box, pot, w.v_cut, w.mask_mode)
    grid = O.SparseGrid(box, act, 1)
    y0 = I.make_psi0(w, act)
    T = 0.02
    ref = O.run_rk4(grid, pot, w.g, 0.0, T / 64, 64, y0, 7)
    errs = [np.max(np.abs(O.run_rkhe3(grid, pot, w.g, 0.0, T / n, n, y0, 7) - ref)) for n in (4, 8, 16)]
    assert 6.5 < errs[0] / errs[1] < 9.5 and 6.5 < errs[1] / errs[2] < 9.5


# ---- P16: Cash-Karp (RKCK, Eq. A12-A13) -------------------------------------------------------
CK_A = [[], [Fraction(1, 5)], [Fraction(3, 40), Fraction(9, 40)], [Fraction(3, 10), Fraction(-9, 10), Fraction(6, 5)],
        [Fraction(-11, 54), Fraction(5, 2), Fraction(-70, 27), Fraction(35, 27)],
        [Fraction(1631, 55296), Fraction(175, 512), Fraction(575, 13824), Fraction(44275, 110592), Fraction(253, 4096)]]
CK_B = [Fraction(37, 378), 0, Fraction(250, 621), Fraction(125, 594), 0, Fraction(512, 1771)]


def test_P16_rkck_modified_tableau_matches_paper():
    """Eq. A4-A7 applied to the Cash-Karp tableau reproduce the paper's a*, b* (Eq. A12-A13) entry by entry; the
    two entries the extracted text garbles differ from the printed ones in one digit each and every row of a*
    sums to 1 (consistency: y^(i+1) = y0 when all k vanish)."""
    gold = json.load(open(os.path.join(GOLD, "paper_values.json")))
    astar, bstar = modified_tableau(CK_A, CK_B)
    assert bstar == [Fraction(s) for s in gold["rkck_b_star"]["value"]]
    for i, row in enumerate(gold["rkck_a_star"]["value"]):
        assert astar[i] == [Fraction(v) for v in row]
        assert sum(astar[i]) == 1
    assert sum(bstar) == 1
    g = gold["rkck_a_star"]["printed_garbled"]
    assert Fraction(g["row5_col1"]) != astar[4][0] and Fraction(g["row5_col3"]) != astar[4][2]
    # the oracle's float tableau is that tableau
    for i in range(6):
        assert [float(x) for x in CK_A[i]] == list(O.RKCK_A[i])
        assert float(CK_B[i]) == O.RKCK_B[i]
        assert float(sum(CK_A[i], Fraction(0))) == pytest.approx(O.RKCK_C[i], abs=1e-16)


def test_P16_rkck_is_fifth_order_and_stage_form_matches():
    w = I.small_shell(20, 7)
    box = O.Box(w.nx, w.ny, w.nz, w.h)
    pot = O.Potential(w.kind, w.ax, w.ay, w.az, 5.0, 20.0, 0.05, w.omega)
    act = O.active_indices(box, pot, w.v_cut, O.MASK_UNION)
    grid = O.SparseGrid(box, act, 1)
    y0 = I.make_psi0(w, act)
    g = w.g
    # linear test equation: amplification factor = degree-5 Taylor polynomial + z^6 b6 a65 a54 a43 a32 a21 (= z^6/800)
    pot0 = O.Potential(kind=O.HARMONIC)
    n, h = 12, 0.6
    boxf, gridf = full_box_grid(n, n, n, h)
    e1, v1 = ho_ground_state_1d(n, h, 7)
    psi = (v1[:, None, None] * v1[None, :, None] * v1[None, None, :]).ravel().astype(np.complex128)
    dt = 0.2
    z = -1j * 3 * e1 * dt
    taylor5 = sum(z ** k / math.factorial(k) for k in range(6))
    got = O.rkck_step(gridf, pot0, 0.0, 0.0, dt, psi, 7)
    fac = np.vdot(psi, got) / np.vdot(psi, psi)
    c6 = CK_B[5] * CK_A[5][4] * CK_A[4][3] * CK_A[3][2] * CK_A[2][1] * CK_A[1][0]
    assert c6 == Fraction(1, 800)
    assert abs(fac - taylor5 - z ** 6 * float(c6)) < 1e-13
    # order 5 on the nonlinear, ramped problem
    T = 0.04
    ref = O.run_rkck(grid, pot, g, 0.0, T / 64, 64, y0, 7)
    errs = [np.max(np.abs(O.run_rkck(grid, pot, g, 0.0, T / k, k, y0, 7) - ref)) for k in (2, 4)]
    assert 20 < errs[0] / errs[1] < 45
    # the stage-state form with the paper's a*, b* gives the textbook step
    astar, bstar = modified_tableau(CK_A, CK_B)
    t, dt = 0.003, 2e-3
    f = lambda tt, y: -1j * O.apply_H(grid, pot, g, tt, y, 7)
    ys = [y0]
    for i in range(1, 6):
        nxt = sum(float(astar[i - 1][j]) * ys[j] for j in range(i)) + dt * float(CK_A[i][i - 1]) * f(t + O.RKCK_C[i - 1] * dt, ys[i - 1])
        ys.append(nxt)
    ynew = sum(float(bstar[j]) * ys[j] for j in range(6)) + dt * float(CK_B[5]) * f(t + O.RKCK_C[5] * dt, ys[5])
    want = O.rkck_step(grid, pot, g, t, dt, y0, 7)
    assert np.max(np.abs(ynew - want)) < 1e-13 * np.max(np.abs(want))


# ---- P17: the 19-point higher-order compact stencil (PAPER.md:341-343 Eq. B2) ----------------------------------
def test_P17_19pt_weights_symbol_and_kronecker():
    gold = json.load(open(os.path.join(GOLD, "paper_values.json")))["nineteen_point_isotropic"]["value"]
    n, h = 7, 0.5
    box, grid = full_box_grid(n, n, n, h, radius=1)
    # (a) weights: apply to a unit vector at the centre of the box
    c = (n // 2 * n + n // 2) * n + n // 2
    e = np.zeros(n ** 3, np.complex128)
    e[c] = 1.0
    lap = (-2.0 * O.apply_T(grid, e, 19)).real.reshape(n, n, n) * h * h
    m = n // 2
    assert abs(lap[m, m, m] - float(Fraction(gold["centre"]))) < 1e-13
    for off in [(1, 0, 0), (0, -1, 0), (0, 0, 1)]:
        assert abs(lap[m + off[0], m + off[1], m + off[2]] - float(Fraction(gold["face"]))) < 1e-13
    for off in [(1, 1, 0), (-1, 0, 1), (0, 1, -1)]:
        assert abs(lap[m + off[0], m + off[1], m + off[2]] - float(Fraction(gold["edge"]))) < 1e-13
    assert abs(lap[m + 1, m + 1, m + 1]) == 0 and np.count_nonzero(lap) == 19 and abs(lap.sum()) < 1e-12
    # (b) sine modes of the Dirichlet box are exact eigenvectors: s_x + s_y + s_z + h^2/6 (s_x s_y + s_x s_z + s_y s_z)
    mode = (2, 1, 3)
    psi = sine_mode(n, n, n, mode).ravel()
    sx, sy, sz = [-(4 / h ** 2) * math.sin(math.pi * mm / (2 * (n + 1))) ** 2 for mm in mode]
    lam = sx + sy + sz + h * h / 6 * (sx * sy + sx * sz + sy * sz)
    assert np.max(np.abs(O.apply_T(grid, psi, 19) + 0.5 * lam * psi)) < 1e-12
    # (c) Eq. B2 as Kronecker products with rows / columns deleted, random masks
    nx, ny, nz = 5, 6, 4
    d = lambda k: lap1d(k, h, 7)
    eye = np.eye
    k3 = lambda a, b, cc: np.kron(np.kron(a, b), cc)
    lap7 = k3(d(nx), eye(ny), eye(nz)) + k3(eye(nx), d(ny), eye(nz)) + k3(eye(nx), eye(ny), d(nz))
    lap19 = lap7 + (2 * h * h / 12) * (k3(d(nx), d(ny), eye(nz)) + k3(d(nx), eye(ny), d(nz)) + k3(eye(nx), d(ny), d(nz)))
    for seed, pr in ((31, 0.6), (32, 0.9)):
        act = I.random_mask_lin(seed, nx, ny, nz, pr)
        tmat = -0.5 * lap19[np.ix_(act, act)]
        g2 = O.SparseGrid(O.Box(nx, ny, nz, h), act, 1)
        psi = I.random_psi(seed, act.size)
        assert np.max(np.abs(O.apply_T(g2, psi, 19) - tmat @ psi)) < 1e-12 * np.max(np.abs(tmat)) * 8
        assert np.max(np.abs(tmat - tmat.T)) == 0          # Hermitian (principal sub-matrix)


def test_P17_19pt_leading_error_is_isotropic():
    """lap_19 u = lap u + h^2/12 lap^2 u + O(h^4): on a plane wave the symbol is -k^2 + h^2 k^4 / 12 to that order,
    a function of |k| only (the 7-point symbol has h^2/12 sum k_i^4 instead)."""
    h = 0.05
    for kv in ((1.0, 2.0, 2.0), (3.0, 0.0, 0.0), (0.0, 2.4, 1.8)):      # all |k| = 3
        s = [-(4 / h ** 2) * math.sin(k * h / 2) ** 2 for k in kv]
        lam19 = sum(s) + h * h / 6 * (s[0] * s[1] + s[0] * s[2] + s[1] * s[2])
        assert abs(lam19 - (-9.0 + h * h * 81.0 / 12)) < 5e-5 * 9


# ---- P18: anisotropic spacing d_x != d_y != d_z (App. B) -----------------------------------------
def test_P18_anisotropic_spacing():
    nx, ny, nz = 6, 7, 5
    dx, dy, dz = 0.5, 0.8, 0.3
    box = O.Box(nx, ny, nz, dx, (0.1, -0.2, 0.3), dy, dz)
    full = np.arange(nx * ny * nz, dtype=np.int64)
    grid = O.SparseGrid(box, full, 2)
    # (a) 7-point: sine modes are exact eigenvectors, each axis with its own step (Eq. B1)
    mode = (2, 3, 1)
    psi = sine_mode(nx, ny, nz, mode).ravel()
    lam = sum(-(4 / d ** 2) * math.sin(math.pi * m / (2 * (n + 1))) ** 2 for d, m, n in zip((dx, dy, dz), mode, (nx, ny, nz)))
    assert np.max(np.abs(O.apply_T(grid, psi, 7) + 0.5 * lam * psi)) < 1e-12
    # (b) Kronecker forms with per-axis second differences, rows / columns deleted, 7 / 13 / 19 points
    eye = np.eye
    k3 = lambda a, b, c: np.kron(np.kron(a, b), c)
    for stencil in (7, 13, 19):
        st = 7 if stencil == 19 else stencil
        ddx, ddy, ddz = lap1d(nx, dx, st), lap1d(ny, dy, st), lap1d(nz, dz, st)
        lap = k3(ddx, eye(ny), eye(nz)) + k3(eye(nx), ddy, eye(nz)) + k3(eye(nx), eye(ny), ddz)
        if stencil == 19:
            lap = lap + ((dx * dx + dy * dy) * k3(ddx, ddy, eye(nz)) + (dx * dx + dz * dz) * k3(ddx, eye(ny), ddz)
                         + (dy * dy + dz * dz) * k3(eye(nx), ddy, ddz)) / 12
        act = I.random_mask_lin(41, nx, ny, nz, 0.7)
        g2 = O.SparseGrid(box, act, 2)
        tmat = -0.5 * lap[np.ix_(act, act)]
        phi = I.random_psi(42, act.size)
        assert np.max(np.abs(O.apply_T(g2, phi, stencil) - tmat @ phi)) < 1e-12 * np.max(np.abs(tmat)) * 8
        if stencil != 19:
            mask = np.zeros(nx * ny * nz, bool)
            mask[act] = True
            dense = np.zeros(nx * ny * nz, np.complex128)
            dense[act] = phi
            got = O.dense_apply_T(box, mask.reshape(nx, ny, nz), dense.reshape(nx, ny, nz), stencil).ravel()[act]
            assert np.max(np.abs(got - tmat @ phi)) < 1e-12 * np.max(np.abs(tmat)) * 8
    # (c) coordinates, volume element, separable harmonic ground state
    assert abs(O.norm(grid, np.ones(full.size, np.complex128)) - full.size * dx * dy * dz) < 1e-12
    v = O.potential_at(box, O.Potential(kind=O.HARMONIC, ax=1.0, ay=2.0, az=3.0), full, 0.0).reshape(nx, ny, nz)
    x = (np.arange(nx) - 0.5 * (nx - 1)) * dx + 0.1
    y = (np.arange(ny) - 0.5 * (ny - 1)) * dy - 0.2
    z = (np.arange(nz) - 0.5 * (nz - 1)) * dz + 0.3
    assert np.max(np.abs(v - 0.5 * (x[:, None, None] ** 2 + 2 * y[None, :, None] ** 2 + 3 * z[None, None, :] ** 2))) < 1e-14
    n = 16
    boxh = O.Box(n, n, n, 0.5, (0.0, 0.0, 0.0), 0.6, 0.7)
    gh = O.SparseGrid(boxh, np.arange(n ** 3, dtype=np.int64), 1)
    es, vs = zip(*[ho_ground_state_1d(n, d, 7) for d in (0.5, 0.6, 0.7)])
    psi = (vs[0][:, None, None] * vs[1][None, :, None] * vs[2][None, None, :]).ravel().astype(np.complex128)
    psi /= math.sqrt(O.norm(gh, psi))
    e = O.energy(gh, O.Potential(kind=O.HARMONIC), 0.0, 0.0, psi, 7)
    assert abs(e["total"] - sum(es)) < 1e-12 and abs(e["mu"] - sum(es)) < 1e-12


# ---- P19: the 27-point compact stencil with caller-supplied weights ("HOC stencils of shape 3^3") ------
def test_P19_compact27_reductions_and_brute_force():
    nx, ny, nz = 6, 5, 7
    dx, dy, dz = 0.5, 0.7, 0.4
    box = O.Box(nx, ny, nz, dx, (0.0, 0.0, 0.0), dy, dz)
    act = I.random_mask_lin(51, nx, ny, nz, 0.75)
    grid = O.SparseGrid(box, act, 1)
    psi = I.random_psi(52, act.size)
    ia = [1 / dx ** 2, 1 / dy ** 2, 1 / dz ** 2]
    # (a) weights of Eq. B1 -> the 7-point operator; weights of Eq. B2 -> the 19-point operator
    w7 = O.Compact27(-2 * sum(ia), tuple(ia), (0.0, 0.0, 0.0), 0.0)
    assert np.max(np.abs(O.apply_T(grid, psi, w7) - O.apply_T(grid, psi, 7))) < 1e-12 * 40
    cxy, cxz, cyz = (ia[0] + ia[1]) / 12, (ia[0] + ia[2]) / 12, (ia[1] + ia[2]) / 12
    w19 = O.Compact27(-2 * sum(ia) + 4 * (cxy + cxz + cyz),
                      (ia[0] - 2 * (cxy + cxz), ia[1] - 2 * (cxy + cyz), ia[2] - 2 * (cxz + cyz)), (cxy, cxz, cyz), 0.0)
    assert np.max(np.abs(O.apply_T(grid, psi, w19) - O.apply_T(grid, psi, 19))) < 1e-12 * 40
    # (b) brute force with all four classes non-zero: dense 3x3x3 correlation on the zero-extended box
    w = O.Compact27(-3.1, (0.7, 0.5, 0.9), (0.11, 0.13, 0.17), 0.03)
    dense = np.zeros((nx + 2, ny + 2, nz + 2), np.complex128)
    ix, iy, iz = O.unravel(box, act)
    dense[ix + 1, iy + 1, iz + 1] = psi
    out = np.zeros(act.size, np.complex128)
    for a in (-1, 0, 1):
        for b in (-1, 0, 1):
            for c in (-1, 0, 1):
                k = abs(a) + abs(b) + abs(c)
                if k == 0:
                    wt = w.centre
                elif k == 1:
                    wt = w.face[0] if a else (w.face[1] if b else w.face[2])
                elif k == 2:
                    wt = w.edge[0] if c == 0 else (w.edge[1] if b == 0 else w.edge[2])
                else:
                    wt = w.corner
                out += wt * dense[ix + 1 + a, iy + 1 + b, iz + 1 + c]
    assert np.max(np.abs(O.apply_T(grid, psi, w) + 0.5 * out)) < 1e-13
    # (c) the tensor-product stencil (1 + a dxx)(1 + b dyy)(1 + c dzz) - 1 has all four classes: Kronecker form
    eye = np.eye
    k3 = lambda p, q, r: np.kron(np.kron(p, q), r)
    A, B, C = 0.02, 0.03, 0.05
    mats = [eye(n) + co * lap1d(n, d, 7) for n, d, co in ((nx, dx, A), (ny, dy, B), (nz, dz, C))]
    full = k3(*mats) - eye(nx * ny * nz)
    fx, fy, fz = A * ia[0], B * ia[1], C * ia[2]                       # off-diagonal entries of the 1-D factors
    px, py, pz = 1 - 2 * fx, 1 - 2 * fy, 1 - 2 * fz                    # diagonal entries
    wt = O.Compact27(px * py * pz - 1, (fx * py * pz, px * fy * pz, px * py * fz), (fx * fy * pz, fx * py * fz, px * fy * fz), fx * fy * fz)
    tm = -0.5 * full[np.ix_(act, act)]
    assert np.max(np.abs(O.apply_T(grid, psi, wt) - tm @ psi)) < 1e-13


# ---- P20: a fixed point of the normalised Euler iteration is a stationary state (g > 0) ----------------------------
def _stationary_shell(g=300.0, dt=8e-3, nsteps=3200):
    """Imaginary time on a small dressed shell until psi <- normalise((1 - dt H[psi]) psi) no longer moves."""
    from helpers import oracle_objs
    w = I.small_shell(24, 13)
    box, pot, act = oracle_objs(w)
    grid = O.SparseGrid(box, act, 2)
    psi = np.abs(I.make_psi0(w, act)).astype(np.complex128)
    psi /= math.sqrt(O.norm(grid, psi))
    psi = O.run_imag(grid, pot, g, 0.0, dt, nsteps, psi, 13)
    return box, pot, act, grid, psi


def test_P20_imag_step_fixed_point_is_stationary_state_g_positive():
    """PAPER.md:25 Eq. 1 (H psi = mu psi) and :35 (imaginary time converges to the ground state): a fixed point of
    psi <- normalise((1 - dt H[psi]) psi) satisfies H[psi] psi = mu psi exactly, for any dt, with
    mu = <psi|H psi>/<psi|psi>.  apply_H is pinned separately (P5, P11), so this pins the g > 0 arithmetic of
    imag_step (a doubled or dropped g |psi|^2 term moves the fixed point away from Eq. 1) and energy()['mu']
    (kin + pot + 2 inter; with 1 inter the residual below is O(inter))."""
    g = 300.0
    box, pot, act, grid, psi = _stationary_shell(g)
    e = O.energy(grid, pot, g, 0.0, psi, 13)
    hp = O.apply_H(grid, pot, g, 0.0, psi, 13)
    assert e["inter"] > 0.05 * abs(e["mu"])            # the nonlinear term matters in this state
    res = np.max(np.abs(hp - e["mu"] * psi)) / np.max(np.abs(e["mu"] * psi))
    assert res < 1e-8
    # the fixed point does not depend on dt: one step with another dt leaves it in place
    again = O.imag_step(grid, pot, g, 0.0, 2e-3, psi, 13)
    assert np.max(np.abs(again - psi)) < 1e-9 * np.max(np.abs(psi))
    # the explicit-loop C restatement has the same fixed point and the same mu
    from oracle.c_oracle import COracle
    co = COracle(box, pot, act, 13)
    ec = co.energy(g, 0.0, psi)
    assert abs(ec["mu"] - e["mu"]) < 1e-12 * abs(e["mu"])
    hc = co.apply_H(g, 0.0, psi)
    assert np.max(np.abs(hc - ec["mu"] * psi)) / np.max(np.abs(ec["mu"] * psi)) < 1e-8
    stepc = co.run_imag(g, 0.0, 2e-3, 1, psi)
    assert np.max(np.abs(stepc - psi)) < 1e-9 * np.max(np.abs(psi))


# ---- P21: mu is the Rayleigh quotient of H[psi] (definition, Eq. 1), on a random state with g > 0 ---------------
@pytest.mark.parametrize("stencil", [7, 13])
def test_P21_mu_is_rayleigh_quotient_of_apply_H(stencil):
    from helpers import oracle_objs
    w = I.small_shell(24, stencil)
    box, pot, act = oracle_objs(w)
    grid = O.SparseGrid(box, act, 2)
    psi = I.random_psi(77, len(act))
    g = 431.0
    hp = O.apply_H(grid, pot, g, 0.3, psi, stencil)
    rq = box.cell * float(np.sum((np.conj(psi) * hp).real)) / (box.cell * float(np.sum(np.abs(psi) ** 2)))
    e = O.energy(grid, pot, g, 0.3, psi, stencil)
    assert abs(e["mu"] - rq) < 1e-12 * abs(rq)
    assert abs(e["norm"] - box.cell * float(np.sum(np.abs(psi) ** 2))) < 1e-13 * e["norm"]
    # the interaction energy is half the interaction part of <H>: E = <H> - inter, so total = mu norm - inter
    assert abs(e["total"] - (e["mu"] * e["norm"] - e["inter"])) < 1e-12 * abs(e["total"])
    from oracle.c_oracle import COracle
    ec = COracle(box, pot, act, stencil).energy(g, 0.3, psi)
    assert abs(ec["mu"] - rq) < 1e-12 * abs(rq)


# ---- P22: Thomas-Fermi limit of the converged state (Eq. 5) ------------------------------------------------
def test_P22_thomas_fermi_limit_for_large_g():
    """For large g the kinetic term is a small correction and the stationary state obeys
    g |psi|^2 = mu - V where mu > V (Eq. 5).  Harmonic trap, g = 4000: the Thomas-Fermi chemical
    potential is mu_TF = (15 g / (4 pi))^(2/5) / 2 and the density follows (mu - V)/g away from the cloud's edge."""
    n, h, g = 28, 0.5, 4000.0
    box = O.Box(n, n, n, h)
    pot = O.Potential(kind=O.HARMONIC)
    act = O.active_indices(box, pot, 22.0)                  # V < 22: a ball that contains the cloud (mu_TF ~ 9.2)
    grid = O.SparseGrid(box, act, 1)
    v = O.potential_at(box, pot, act, 0.0)
    mu_tf = 0.5 * (15.0 * g / (4.0 * math.pi)) ** 0.4
    psi = np.sqrt(np.maximum(mu_tf - v, 0.0) / g).astype(np.complex128) + 1e-3
    psi /= math.sqrt(O.norm(grid, psi))
    psi = O.run_imag(grid, pot, g, 0.0, 4e-3, 1500, psi, 7)
    e = O.energy(grid, pot, g, 0.0, psi, 7)
    assert abs(e["mu"] - mu_tf) < 0.02 * mu_tf              # kinetic correction ~ (1/R_TF^2) ln R_TF
    bulk = v < 0.6 * e["mu"]
    dens = np.abs(psi[bulk]) ** 2
    assert np.max(np.abs(g * dens - (e["mu"] - v[bulk]))) < 0.03 * e["mu"]
    assert e["kin"] < 0.05 * e["mu"]


# ---- P23: the paper's split iteration agrees with the Euler step to first order in dt for g > 0 -----------------
def test_P23_split_step_equals_euler_step_to_second_order_g_positive():
    """D K K D with the linearised interaction factor and one Euler step of the full H differ by
    O(dt^2) per step; a wrong g, dt/2 or ordering in diag_propagator shows up at O(dt).  With P20 this pins
    imag_split_step for g > 0."""
    from helpers import oracle_objs
    w = I.small_shell(24, 13)
    box, pot, act = oracle_objs(w)
    grid = O.SparseGrid(box, act, 2)
    psi = np.abs(I.make_psi0(w, act)).astype(np.complex128)
    psi /= math.sqrt(O.norm(grid, psi))
    g = 300.0
    d = []
    for dt in (1e-3, 5e-4, 2.5e-4):
        a = O.imag_split_step(grid, pot, g, 0.0, dt, psi, 13)
        b = O.imag_step(grid, pot, g, 0.0, dt, psi, 13)
        d.append(np.max(np.abs(a - b)))
    assert 3.6 < d[0] / d[1] < 4.4 and 3.6 < d[1] / d[2] < 4.4
    # the test can see an O(dt) defect of the nonlinear term: that term's whole effect at the smallest dt is several
    # times the O(dt^2) difference measured there
    lin = np.max(np.abs(O.imag_step(grid, pot, g, 0.0, 2.5e-4, psi, 13) - O.imag_step(grid, pot, 0.0, 0.0, 2.5e-4, psi, 13)))
    assert lin > 3 * d[2]
