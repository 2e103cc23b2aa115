"""Shared test helpers: build oracle objects / product objects from a gpe_inputs.Workload."""
import numpy as np

import gpe_inputs as I
from oracle import gpe_oracle as O


def oracle_objs(w, active=None):
    box = O.Box(w.nx, w.ny, w.nz, w.h, w.center, w.hy, w.hz)
    pot = O.Potential(w.kind, w.ax, w.ay, w.az, w.delta0, w.delta1, w.t_ramp, w.omega)
    act = O.active_indices(box, pot, w.v_cut, w.mask_mode) if active is None else np.asarray(active, np.int64)
    return box, pot, act


def rel_max(a, b):
    """max_p |a_p - b_p| / max_p |b_p|  (R10)."""
    a = np.asarray(a)
    b = np.asarray(b)
    if b.size == 0:
        return 0.0
    return float(np.max(np.abs(a - b)) / np.max(np.abs(b)))


RADIUS = {7: 1, 13: 2, 19: 1}
