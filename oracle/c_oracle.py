"""ctypes wrapper of oracle/gpe_oracle_c.c.  TEST INFRASTRUCTURE ONLY (see that file's header).

``build()`` compiles the C file with gcc (no CUDA, no product code); ``COracle`` runs the
explicit-loop operator / textbook RK4 / imaginary-time steps on numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "gpe_oracle_c.c")
LIB = os.path.join(HERE, "libgpe_oracle.so")


class _Problem(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("kind", C.c_int32),
                ("h", C.c_double), ("cx", C.c_double), ("cy", C.c_double), ("cz", C.c_double),
                ("ax", C.c_double), ("ay", C.c_double), ("az", C.c_double),
                ("delta0", C.c_double), ("delta1", C.c_double), ("t_ramp", C.c_double),
                ("omega", C.c_double), ("hy", C.c_double), ("hz", C.c_double)]


def build(force: bool = False) -> str:
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < os.path.getmtime(SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC",
               SRC, "-o", LIB, "-lm"]
        subprocess.run(cmd, check=True)
    return LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(LIB)
        _lib.orc_num_threads.restype = C.c_int
        _lib.orc_norm.restype = C.c_double
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


class COracle:
    def __init__(self, box, pot, active: np.ndarray, stencil: int):
        self.lib = _load()
        self.prob = _Problem(box.nx, box.ny, box.nz, pot.kind, box.h, box.center[0], box.center[1],
                             box.center[2], pot.ax, pot.ay, pot.az, pot.delta0, pot.delta1,
                             pot.t_ramp, pot.omega, box.spacing[1], box.spacing[2])
        self.active = np.ascontiguousarray(active, dtype=np.int64)
        self.n = self.active.size
        self.R = {7: 1, 13: 2}[stencil]
        self.nbr = np.empty(self.n * 6 * self.R, dtype=np.int64)
        self.lib.orc_build_neighbours(C.byref(self.prob), _p(self.active), C.c_int64(self.n),
                                      C.c_int(self.R), _p(self.nbr))

    @property
    def threads(self) -> int:
        return int(self.lib.orc_num_threads())

    def set_threads(self, n: int):
        """OpenMP threads of the loops (0 = all cores)."""
        self.lib.orc_set_num_threads(C.c_int(int(n)))

    def apply_H(self, g, t, psi):
        psi = np.ascontiguousarray(psi, dtype=np.complex128)
        out = np.empty_like(psi)
        self.lib.orc_apply_H(C.byref(self.prob), _p(self.active), _p(self.nbr), C.c_int64(self.n),
                             C.c_int(self.R), C.c_double(g), C.c_double(t), _p(psi), _p(out))
        return out

    def run_rk4(self, g, t0, dt, nsteps, psi):
        psi = np.array(psi, dtype=np.complex128, copy=True)
        work = np.empty(5 * self.n, dtype=np.complex128)
        self.lib.orc_run_rk4(C.byref(self.prob), _p(self.active), _p(self.nbr), C.c_int64(self.n),
                             C.c_int(self.R), C.c_double(g), C.c_double(t0), C.c_double(dt),
                             C.c_int64(nsteps), _p(psi), _p(work))
        return psi

    def run_imag(self, g, t, dt, nsteps, psi, n_target=1.0):
        psi = np.array(psi, dtype=np.complex128, copy=True)
        work = np.empty(self.n, dtype=np.complex128)
        self.lib.orc_run_imag(C.byref(self.prob), _p(self.active), _p(self.nbr), C.c_int64(self.n),
                              C.c_int(self.R), C.c_double(g), C.c_double(t), C.c_double(dt),
                              C.c_int64(nsteps), C.c_double(n_target), _p(psi), _p(work))
        return psi

    def norm(self, psi):
        psi = np.ascontiguousarray(psi, dtype=np.complex128)
        return float(self.lib.orc_norm(C.byref(self.prob), C.c_int64(self.n), _p(psi)))

    def energy(self, g, t, psi):
        psi = np.ascontiguousarray(psi, dtype=np.complex128)
        work = np.empty(self.n, dtype=np.complex128)
        out = np.zeros(6, dtype=np.float64)
        self.lib.orc_energy(C.byref(self.prob), _p(self.active), _p(self.nbr), C.c_int64(self.n),
                            C.c_int(self.R), C.c_double(g), C.c_double(t), _p(psi), _p(work), _p(out))
        return dict(zip(("kin", "pot", "inter", "total", "mu", "norm"), out.tolist()))
