"""gpe_norm_noalloc: the norm for callers that must not allocate, checked against the existing gpe_norm path.

Who needs it: a program in which torch's caching allocator (or another framework's) already owns nearly all GPU
memory, so that a cudaMalloc made inside the library would fail; a norm check that runs between time steps while
other streams are busy and must not be stalled by cudaMalloc / cudaFree, which wait for the whole device; code that
holds only an array of wavefunction values and no Sim.  gpe_norm_noalloc serves them from a fixed 512 KiB scratch
array compiled into the library (include/gpe.h), at the price of a size limit (2^29 values) and of calls that must
not overlap on one GPU.

The scratch array is shared by every call and keeps what the previous call left in it, so each case below makes two
calls in a row -- a larger array first, then a smaller one with different values -- and compares both with
Sim.norm() of the same state at the 1e-12 relative tolerance the norm checks in test_gpu_parity.py use (the two paths
sum in a different order: canonical against storage order).  The file name sorts after every other test file, so
under `pytest -x` a failure here cannot hide another test; nothing here relies on what earlier tests did, and the
first case also works as the very first CUDA call of a fresh process (the entry point resolves its scratch address
on its first call per device).
"""
import numpy as np
import pytest

import gpe_inputs as I

pytestmark = pytest.mark.gpu

TOL = 1e-12   # relative; |norm| is O(1) in every case, as in test_gpu_parity.py's norm checks


@pytest.fixture(scope="module")
def P():
    import paper_2603_05447_b200 as P
    return P


def _state(P, w, dtype, seed_scale):
    """A Sim holding a seeded state on w's shell, the same state as a canonical device tensor, the cell volume."""
    import torch
    grid = P.Grid.from_workload(w)
    sim = P.Sim(grid, dtype, w.stencil, w.g)
    psi = I.make_psi0(w, grid.active_indices()) * seed_scale
    if dtype == "float64":
        psi = np.ascontiguousarray(psi.real)
    d = torch.from_numpy(np.ascontiguousarray(psi)).to("cuda:0").to(getattr(torch, dtype))
    sim.set_psi(d)
    h3 = w.h * (w.hy if w.hy > 0 else w.h) * (w.hz if w.hz > 0 else w.h)
    return sim, d, h3


@pytest.mark.parametrize("dtype", ["complex128", "complex64", "float64"])
def test_noalloc_norm_matches_sim_norm_on_two_calls_in_a_row(P, dtype):
    import torch
    torch.cuda.set_device(0)
    out = torch.full((1,), -7.0, dtype=torch.float64, device="cuda:0")   # the caller's output, deliberately not zero
    # first call: BASELINE configs[1]'s bubble with a non-constant seeded state, 1.2e6 values (147 scratch slots, ragged
    # last block); second call: a 2e4-value shell (3 slots) with other values
    big = _state(P, I.config2().with_(psi0="shell", seed=21), dtype, 1.0)
    small = _state(P, I.small_shell(33, 7).with_(center=(0.3, -0.2, 0.1)), dtype, 1.7)
    assert big[1].numel() > 100 * 8192 and small[1].numel() < 4 * 8192
    for sim, d, h3 in (big, small):
        want = sim.norm()
        assert want > 0.1
        P.norm_noalloc(d, h3, out)
        torch.cuda.synchronize()
        got = float(out.item())
        assert abs(got - want) <= TOL * want, (dtype, d.numel(), got, want)
    # and once more on the first array: what the second call left in the scratch does not leak into the result,
    # and the same array gives the same bits
    sim, d, h3 = big
    P.norm_noalloc(d, h3, out)
    torch.cuda.synchronize()
    first = float(out.item())
    P.norm_noalloc(d, h3, out)
    torch.cuda.synchronize()
    assert float(out.item()) == first
    assert abs(first - sim.norm()) <= TOL * first


def test_noalloc_norm_same_array_same_order_is_bit_identical_to_gpe_norm(P):
    """Given the sim's own storage-order array (the first n values of its state block), the static-scratch variant sums
    in gpe_norm's order below 19 398 656 values: same bits.  Two arrays in a row, as above."""
    import torch
    torch.cuda.set_device(0)
    out = torch.empty(1, dtype=torch.float64, device="cuda:0")
    for w in (I.config2().with_(psi0="shell", seed=22), I.small_shell(40, 13)):
        sim, d, h3 = _state(P, w, "complex128", 1.0)
        off = sim._state_ptr - sim.state.data_ptr()
        storage = sim.state[off: off + 16 * sim.n].view(torch.complex128)
        P.norm_noalloc(storage, h3, out)
        torch.cuda.synchronize()
        assert float(out.item()) == sim.norm()


def test_noalloc_norm_empty_and_limits(P):
    import torch
    torch.cuda.set_device(0)
    out = torch.full((1,), 3.0, dtype=torch.float64, device="cuda:0")
    d = torch.ones(100, dtype=torch.complex128, device="cuda:0")
    P.norm_noalloc(d[:0], 0.5, out)
    torch.cuda.synchronize()
    assert float(out.item()) == 0.0
    P.norm_noalloc(d, 0.5, out)
    torch.cuda.synchronize()
    assert float(out.item()) == 50.0
    # over the limit: refused before anything is launched (the array is not touched, so a small one will do), with text
    # that names the limit; the output keeps its value
    with pytest.raises(P.GpeError) as ei:
        P.norm_noalloc(d, 0.5, out, n=P.NORM_NOALLOC_MAX_VALUES + 1)
    assert ei.value.code == -4 and "GPE_NORM_NOALLOC_MAX_VALUES" in str(ei.value)
    torch.cuda.synchronize()
    assert float(out.item()) == 50.0
    # a host array is not memory of the device: INVALID_ARG, nothing launched
    import ctypes as C
    host = np.ones(4, np.complex128)
    rc = P.lib().gpe_norm_noalloc(host.ctypes.data_as(C.c_void_p), C.c_int64(4), C.c_int(P.C128), C.c_double(1.0),
                                  C.c_void_p(out.data_ptr()), C.c_void_p(0))
    assert rc == -1 and "current CUDA device" in P.lib().gpe_last_error().decode()
    torch.cuda.synchronize()
    assert float(out.item()) == 50.0
