"""The explicit-loop C oracle (oracle/gpe_oracle_c.c) against the pinned numpy oracle.

The numpy oracle is pinned to the paper and the mathematics in test_oracle_pins.py; the C
version exists so that full-size parity cases and the timed CPU baseline finish in
reasonable time.  It is a second, independently written implementation (binary-search
neighbours, explicit loops) of the same definitions, so agreement here is also a
cross-check of both.  All CPU.
"""
import numpy as np
import pytest

from oracle import gpe_oracle as O
from oracle import c_oracle as CO
import gpe_inputs as I


def _objs(w):
    box = O.Box(w.nx, w.ny, w.nz, w.h, w.center, w.hy, w.hz)
    pot = O.Potential(w.kind, w.ax, w.ay, w.az, w.delta0, w.delta1, w.t_ramp, w.omega)
    act = O.active_indices(box, pot, w.v_cut, w.mask_mode)
    return box, pot, act


def _rel(a, b):
    return float(np.max(np.abs(a - b)) / np.max(np.abs(b)))


@pytest.mark.parametrize("stencil", [7, 13])
def test_c_apply_H_matches_numpy(stencil):
    w = I.small_shell(24, stencil).with_(delta0=3.0, delta1=9.0, t_ramp=0.5)
    box, pot, act = _objs(w)
    grid = O.SparseGrid(box, act, 2)
    co = CO.COracle(box, pot, act, stencil)
    psi = I.random_psi(7, act.size)
    for t in (0.0, 0.2, 0.9):
        assert _rel(co.apply_H(w.g, t, psi), O.apply_H(grid, pot, w.g, t, psi, stencil)) < 1e-14


def test_c_neighbours_match_numpy_on_random_mask():
    box = O.Box(9, 7, 11, 0.3)
    act = I.random_mask_lin(3, 9, 7, 11, 0.4)
    grid = O.SparseGrid(box, act, 2)
    co = CO.COracle(box, O.Potential(), act, 13)
    nbr = co.nbr.reshape(act.size, 3, 4)
    for axis in range(3):
        for j, s in enumerate((-2, -1, 1, 2)):
            assert np.array_equal(nbr[:, axis, j], grid.nbr[(axis, s)])


def test_c_rk4_imag_energy_match_numpy():
    w = I.small_shell(20, 13).with_(delta0=2.0, delta1=8.0, t_ramp=0.01)
    box, pot, act = _objs(w)
    grid = O.SparseGrid(box, act, 2)
    co = CO.COracle(box, pot, act, 13)
    psi = I.make_psi0(w, act)
    a = co.run_rk4(w.g, 0.0, w.dt, 5, psi)
    b = O.run_rk4(grid, pot, w.g, 0.0, w.dt, 5, psi, 13)
    assert _rel(a, b) < 1e-13
    a = co.run_imag(w.g, 0.003, 1e-3, 7, psi)
    b = O.run_imag(grid, pot, w.g, 0.003, 1e-3, 7, psi, 13)
    assert _rel(a, b) < 1e-13
    ea, eb = co.energy(w.g, 0.004, psi), O.energy(grid, pot, w.g, 0.004, psi, 13)
    for k in eb:
        assert abs(ea[k] - eb[k]) <= 1e-13 * max(1.0, abs(eb[k]))
    assert abs(co.norm(psi) - O.norm(grid, psi)) < 1e-14
