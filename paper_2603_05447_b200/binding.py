"""ctypes binding of libgpe_b200.so (include/gpe.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI.  PyTorch is used for device memory
and streams.  There is no CPU fallback: if the library cannot be loaded, importing this module raises.
Names follow include/gpe.h (gpe_grid_create -> Grid(...), gpe_step_rk4 -> Sim.step_rk4, ...).
"""
from __future__ import annotations

import ctypes as C
import math
import os

import numpy as np

from . import build as _build

HARMONIC, DRESSED = 0, 1
MASK_AT_DELTA0, MASK_AT_DELTA1, MASK_UNION = 0, 1, 2
C64, C128, R64 = 0, 1, 2
OPT_FUSED_K1, OPT_RK4_GRAPH, OPT_PDL = 0, 1, 2

ERR_NAMES = {-1: "GPE_ERR_INVALID_ARG", -2: "GPE_ERR_OUT_OF_MEMORY", -3: "GPE_ERR_CUDA",
             -4: "GPE_ERR_UNSUPPORTED", -5: "GPE_ERR_STATE"}


class GpeError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"{ERR_NAMES.get(code, code)}: {msg}")
        self.code = code


class Box(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("reserved", C.c_int32),
                ("h", C.c_double), ("center", C.c_double * 3), ("hy", C.c_double), ("hz", C.c_double)]


class Potential(C.Structure):
    _fields_ = [("kind", C.c_int32), ("mask_mode", C.c_int32), ("ax", C.c_double), ("ay", C.c_double),
                ("az", C.c_double), ("delta0", C.c_double), ("delta1", C.c_double), ("t_ramp", C.c_double),
                ("omega", C.c_double)]


class LayoutInfo(C.Structure):
    _fields_ = [("tx", C.c_int32), ("ty", C.c_int32), ("zt", C.c_int32), ("halo_width", C.c_int32),
                ("n_active", C.c_int64), ("n_tiles", C.c_int64), ("n_slabs", C.c_int64), ("n_work", C.c_int64)]


class LayoutTables(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in (
        "tile_xy", "tile_zlo", "tile_zhi", "tile_entry_base", "tile_nbr", "slab_mask", "slab_base",
        "wi_tile", "wi_z0", "wi_nz", "storage_to_canonical")]


class EnergyOut(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("kin", "pot", "inter", "total", "mu", "norm")]


# every symbol include/gpe.h declares (tests check that the library exports all of them)
SYMBOLS = (
    "gpe_last_error", "gpe_grid_create", "gpe_grid_create_from_indices", "gpe_grid_destroy",
    "gpe_grid_num_active", "gpe_grid_num_stored", "gpe_grid_layout_info", "gpe_grid_active_indices",
    "gpe_grid_stored_indices", "gpe_grid_layout_tables", "gpe_sim_state_bytes", "gpe_sim_create",
    "gpe_sim_destroy", "gpe_set_psi", "gpe_get_psi", "gpe_set_psi_host", "gpe_get_psi_host",
    "gpe_set_time", "gpe_get_time", "gpe_apply_H", "gpe_step_rk4", "gpe_run_rk4", "gpe_imag_step",
    "gpe_run_imag", "gpe_norm", "gpe_energy", "gpe_sim_kernel_launches", "gpe_sim_time_stages",
    "gpe_sim_stage_time_ms", "gpe_sim_set_planes_per_block", "gpe_imag_split_step", "gpe_run_imag_split",
    "gpe_remap_psi", "gpe_step_rkhe3", "gpe_run_rkhe3", "gpe_step_rkck", "gpe_run_rkck", "gpe_sim_set_compact_weights",
    "gpe_norm_noalloc", "gpe_sim_set_option",
)

NORM_NOALLOC_MAX_VALUES = 1 << 29       # GPE_NORM_NOALLOC_MAX_VALUES

_lib = None


def lib():
    """Load (building first if the in-tree .so is missing or stale) libgpe_b200.so."""
    global _lib
    if _lib is None:
        path = _build.build()
        _lib = C.CDLL(path)
        _lib.gpe_last_error.restype = C.c_char_p
        for name in SYMBOLS:
            getattr(_lib, name)  # AttributeError if the library does not export it
    return _lib


def _check(rc: int):
    if rc != 0:
        raise GpeError(rc, lib().gpe_last_error().decode())


def _np_ptr(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


class Grid:
    """gpe_grid_create / gpe_grid_create_from_indices (host only; no CUDA call)."""

    def __init__(self, nx, ny, nz, h, kind=HARMONIC, ax=1.0, ay=1.0, az=1.0, delta0=0.0, delta1=0.0,
                 t_ramp=0.0, omega=0.0, mask_mode=MASK_AT_DELTA0, v_cut=math.inf, halo_width=2,
                 center=(0.0, 0.0, 0.0), active=None, hy=0.0, hz=0.0):
        self.box = Box(nx, ny, nz, 0, h, (C.c_double * 3)(*center), hy, hz)
        self.pot = Potential(kind, mask_mode, ax, ay, az, delta0, delta1, t_ramp, omega)
        self._h = C.c_void_p()
        L = lib()
        if active is None:
            _check(L.gpe_grid_create(C.byref(self.box), C.byref(self.pot), C.c_double(v_cut),
                                     C.c_int(halo_width), C.byref(self._h)))
        else:
            act = np.ascontiguousarray(active, dtype=np.int64)
            _check(L.gpe_grid_create_from_indices(C.byref(self.box), C.byref(self.pot), _np_ptr(act),
                                                  C.c_int64(act.size), C.c_int(halo_width), C.byref(self._h)))

    @classmethod
    def from_workload(cls, w, active=None):
        return cls(w.nx, w.ny, w.nz, w.h, w.kind, w.ax, w.ay, w.az, w.delta0, w.delta1, w.t_ramp, w.omega,
                   w.mask_mode, w.v_cut, w.halo_width, w.center, active=active, hy=getattr(w, "hy", 0.0),
                   hz=getattr(w, "hz", 0.0))

    def close(self):
        if self._h:
            _check(lib().gpe_grid_destroy(self._h))
            self._h = C.c_void_p()

    def __del__(self):
        try:
            if self._h:
                lib().gpe_grid_destroy(self._h)
        except Exception:
            pass

    @property
    def n_active(self) -> int:
        v = C.c_int64()
        _check(lib().gpe_grid_num_active(self._h, C.byref(v)))
        return v.value

    @property
    def n_stored(self) -> int:
        v = C.c_int64()
        _check(lib().gpe_grid_num_stored(self._h, C.byref(v)))
        return v.value

    def layout_info(self) -> LayoutInfo:
        info = LayoutInfo()
        _check(lib().gpe_grid_layout_info(self._h, C.byref(info)))
        return info

    def active_indices(self) -> np.ndarray:
        out = np.empty(self.n_active, dtype=np.int64)
        _check(lib().gpe_grid_active_indices(self._h, _np_ptr(out)))
        return out

    def stored_indices(self) -> np.ndarray:
        out = np.empty(self.n_stored, dtype=np.int64)
        _check(lib().gpe_grid_stored_indices(self._h, _np_ptr(out)))
        return out

    def layout_tables(self) -> dict:
        i = self.layout_info()
        t = {
            "tile_xy": np.empty((i.n_tiles, 2), np.int32), "tile_zlo": np.empty(i.n_tiles, np.int32),
            "tile_zhi": np.empty(i.n_tiles, np.int32), "tile_entry_base": np.empty(i.n_tiles, np.int64),
            "tile_nbr": np.empty((i.n_tiles, 4), np.int32), "slab_mask": np.empty(i.n_slabs, np.uint64),
            "slab_base": np.empty(i.n_slabs, np.int64), "wi_tile": np.empty(i.n_work, np.int32),
            "wi_z0": np.empty(i.n_work, np.int32), "wi_nz": np.empty(i.n_work, np.int32),
            "storage_to_canonical": np.empty(i.n_active, np.int64),
        }
        s = LayoutTables(**{k: _np_ptr(v) for k, v in t.items()})
        _check(lib().gpe_grid_layout_tables(self._h, C.byref(s)))
        t.update(tx=i.tx, ty=i.ty, zt=i.zt, n_tiles=i.n_tiles)
        return t


def _stream_ptr(stream=None):
    import torch
    st = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(st.cuda_stream)


def norm_noalloc(psi_dev, cell_volume: float, out_dev, stream=None, n=None):
    """gpe_norm_noalloc: out_dev[0] = cell_volume * sum |psi_dev[k]|^2 without a Sim and without any allocation.

    For programs that cannot let the library call cudaMalloc: all device memory already belongs to torch's caching
    allocator, or the check runs between time steps while other streams must not be stalled, or there is only an array
    and no Sim.  The caller supplies both tensors (this wrapper creates none): psi_dev a contiguous CUDA tensor of
    complex128, complex64 or float64 values in any order, out_dev a one-element float64 CUDA tensor on the same device,
    which must be the current one.  Asynchronous on `stream`: synchronise before reading out_dev.  At most
    NORM_NOALLOC_MAX_VALUES values (2^29); more raises GpeError(GPE_ERR_UNSUPPORTED).  Calls share one scratch array
    inside the library, so do not let two of them run concurrently on one GPU; make the first call on a device during
    start-up (it resolves the scratch address).  `n` (default: psi_dev.numel()) only exists so that the size check can be
    exercised without allocating 2^29 values."""
    name = str(psi_dev.dtype).replace("torch.", "")
    code = {"complex128": C128, "complex64": C64, "float64": R64}.get(name)
    if code is None:
        raise ValueError(f"psi_dev must be complex128, complex64 or float64, not {psi_dev.dtype}")
    assert psi_dev.is_cuda and psi_dev.is_contiguous()
    assert out_dev.is_cuda and out_dev.numel() == 1 and str(out_dev.dtype) == "torch.float64"
    _check(lib().gpe_norm_noalloc(C.c_void_p(psi_dev.data_ptr()), C.c_int64(psi_dev.numel() if n is None else n),
                                  C.c_int(code), C.c_double(cell_volume), C.c_void_p(out_dev.data_ptr()),
                                  _stream_ptr(stream)))


class Sim:
    """gpe_sim_create: one wavefunction on a grid.  State memory is a caller-owned torch buffer."""

    def __init__(self, grid: Grid, dtype="complex128", stencil=7, g=0.0, n_target=1.0, device="cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise GpeError(-3, "no CUDA device: the GPE path has no CPU fallback")
        self.torch = torch
        self.grid = grid
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        name = str(dtype).replace("torch.", "")
        if name not in ("complex128", "complex64", "float64"):
            raise ValueError(f"dtype must be complex128, complex64 or float64 (real-valued ground states), not {dtype}")
        self.dtype_code = {"complex128": C128, "complex64": C64, "float64": R64}[name]
        self.cdtype = {C128: torch.complex128, C64: torch.complex64, R64: torch.float64}[self.dtype_code]
        self.npdtype = {C128: np.complex128, C64: np.complex64, R64: np.float64}[self.dtype_code]
        self.n = grid.n_active
        nbytes = C.c_size_t()
        _check(lib().gpe_sim_state_bytes(grid._h, C.c_int(self.dtype_code), C.byref(nbytes)))
        self.state = torch.empty(nbytes.value + 256, dtype=torch.uint8, device=self.device)
        off = (-self.state.data_ptr()) % 256
        self._state_ptr = self.state.data_ptr() + off
        self._h = C.c_void_p()
        _check(lib().gpe_sim_create(grid._h, C.c_int(self.dtype_code), C.c_int(stencil), C.c_double(g),
                                    C.c_double(n_target), C.c_void_p(self._state_ptr), C.c_size_t(nbytes.value),
                                    _stream_ptr(), C.byref(self._h)))

    def close(self):
        if self._h:
            self.torch.cuda.synchronize(self.device)
            _check(lib().gpe_sim_destroy(self._h))
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- psi in canonical order (ascending L over M) -------------------------------------------
    def _check_dev(self, x):
        assert x.is_cuda and x.dtype == self.cdtype and x.is_contiguous() and x.numel() == self.n

    def set_psi(self, psi_dev, stream=None):
        self._check_dev(psi_dev)
        _check(lib().gpe_set_psi(self._h, C.c_void_p(psi_dev.data_ptr()), _stream_ptr(stream)))

    def get_psi(self, out=None, stream=None):
        if out is None:
            out = self.torch.empty(self.n, dtype=self.cdtype, device=self.device)
        self._check_dev(out)
        _check(lib().gpe_get_psi(self._h, C.c_void_p(out.data_ptr()), _stream_ptr(stream)))
        return out

    def set_psi_host(self, psi: np.ndarray, stream=None):
        a = np.ascontiguousarray(psi, dtype=self.npdtype)
        assert a.size == self.n
        _check(lib().gpe_set_psi_host(self._h, _np_ptr(a), _stream_ptr(stream)))

    def get_psi_host(self, out: np.ndarray | None = None, stream=None) -> np.ndarray:
        if out is None:
            out = np.empty(self.n, dtype=self.npdtype)
        assert out.dtype == self.npdtype and out.flags.c_contiguous and out.size == self.n
        _check(lib().gpe_get_psi_host(self._h, _np_ptr(out), _stream_ptr(stream)))
        return out

    # -- clock -------------------------------------------------------------------------------------
    @property
    def time(self) -> float:
        t = C.c_double()
        _check(lib().gpe_get_time(self._h, C.byref(t)))
        return t.value

    @time.setter
    def time(self, t: float):
        _check(lib().gpe_set_time(self._h, C.c_double(t)))

    # -- operator and steppers -----------------------------------------------------------------------
    def apply_H(self, t, psi_in_dev, out=None, stream=None):
        self._check_dev(psi_in_dev)
        if out is None:
            out = self.torch.empty_like(psi_in_dev)
        self._check_dev(out)
        _check(lib().gpe_apply_H(self._h, C.c_double(t), C.c_void_p(psi_in_dev.data_ptr()),
                                 C.c_void_p(out.data_ptr()), _stream_ptr(stream)))
        return out

    def step_rk4(self, dt, stream=None):
        _check(lib().gpe_step_rk4(self._h, C.c_double(dt), _stream_ptr(stream)))

    def run_rk4(self, dt, nsteps, stream=None):
        _check(lib().gpe_run_rk4(self._h, C.c_double(dt), C.c_int64(nsteps), _stream_ptr(stream)))

    def step_rkhe3(self, dt, stream=None):
        _check(lib().gpe_step_rkhe3(self._h, C.c_double(dt), _stream_ptr(stream)))

    def run_rkhe3(self, dt, nsteps, stream=None):
        _check(lib().gpe_run_rkhe3(self._h, C.c_double(dt), C.c_int64(nsteps), _stream_ptr(stream)))

    def step_rkck(self, dt, stream=None):
        _check(lib().gpe_step_rkck(self._h, C.c_double(dt), _stream_ptr(stream)))

    def run_rkck(self, dt, nsteps, stream=None):
        _check(lib().gpe_run_rkck(self._h, C.c_double(dt), C.c_int64(nsteps), _stream_ptr(stream)))

    def imag_step(self, dt, stream=None):
        _check(lib().gpe_imag_step(self._h, C.c_double(dt), _stream_ptr(stream)))

    def run_imag(self, dt, nsteps, stream=None):
        _check(lib().gpe_run_imag(self._h, C.c_double(dt), C.c_int64(nsteps), _stream_ptr(stream)))

    def imag_split_step(self, dt, stream=None):
        _check(lib().gpe_imag_split_step(self._h, C.c_double(dt), _stream_ptr(stream)))

    def run_imag_split(self, dt, nsteps, stream=None):
        _check(lib().gpe_run_imag_split(self._h, C.c_double(dt), C.c_int64(nsteps), _stream_ptr(stream)))

    def remap_from(self, src: "Sim", stream=None):
        """Re-gridding: take src's state on the shared points, 0 on the new ones."""
        _check(lib().gpe_remap_psi(src._h, self._h, _stream_ptr(stream)))

    # -- reductions (synchronise the stream) ------------------------------------------------------------
    def norm(self, stream=None) -> float:
        v = C.c_double()
        _check(lib().gpe_norm(self._h, C.byref(v), _stream_ptr(stream)))
        return v.value

    def energy(self, stream=None) -> dict:
        e = EnergyOut()
        _check(lib().gpe_energy(self._h, C.byref(e), _stream_ptr(stream)))
        return {k: getattr(e, k) for k, _ in EnergyOut._fields_}

    # -- instrumentation ----------------------------------------------------------------------------------
    @property
    def kernel_launches(self) -> int:
        v = C.c_int64()
        _check(lib().gpe_sim_kernel_launches(self._h, C.byref(v)))
        return v.value

    def time_stages(self, on: bool):
        _check(lib().gpe_sim_time_stages(self._h, C.c_int(1 if on else 0)))

    def stage_time_ms(self):
        ms = (C.c_double * 4)()
        cnt = (C.c_int64 * 4)()
        _check(lib().gpe_sim_stage_time_ms(self._h, ms, cnt))
        return list(ms), list(cnt)

    def set_compact_weights(self, centre, face, edge, corner):
        """Weights of the 3x3x3 compact Laplacian (stencil 19 / 27): centre, face (x, y, z), edge (xy, xz, yz), corner."""
        f = (C.c_double * 3)(*face)
        e = (C.c_double * 3)(*edge)
        _check(lib().gpe_sim_set_compact_weights(self._h, C.c_double(centre), f, e, C.c_double(corner)))

    def set_option(self, option: int, value: int):
        """gpe_sim_set_option: OPT_FUSED_K1 / OPT_RK4_GRAPH / OPT_PDL, value 0 or 1 (bit-identical forms of the same path)."""
        _check(lib().gpe_sim_set_option(self._h, C.c_int(option), C.c_int(value)))

    def set_planes_per_block(self, kz: int):
        _check(lib().gpe_sim_set_planes_per_block(self._h, C.c_int(kz)))
