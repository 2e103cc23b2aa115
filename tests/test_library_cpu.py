"""CPU-side checks of the product library: it loads, exports every symbol include/gpe.h declares, and
its HOST layout builder (no CUDA call) is bit-exact against the oracle's independent Python builder
(DESIGN.md "Layout tables").  No compute call is made here."""
import json
import os
import re

import numpy as np
import pytest

import gpe_inputs as I
import paper_2603_05447_b200 as P
from oracle import gpe_oracle as O
from helpers import oracle_objs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "gpe.h")).read()
    declared = set(re.findall(r"\b(gpe_[a-zA-Z0-9_]+)\s*\(", hdr))
    declared -= {"gpe_grid_stored_indices()"}
    assert declared, "no declarations parsed"
    L = P.lib()
    for name in sorted(declared):
        assert hasattr(L, name), name
    assert declared == set(P.SYMBOLS)


def _compare_tables(w, active=None, zt=32):
    box, pot, act = oracle_objs(w, active)
    g = P.Grid.from_workload(w, active=active)
    assert g.n_active == act.size
    assert np.array_equal(g.active_indices(), act)
    ref = O.tile_layout(box, act, 8, 8, zt)
    got = g.layout_tables()
    for k, v in ref.items():
        assert np.array_equal(np.asarray(v), np.asarray(got[k])), k
    assert np.array_equal(g.stored_indices(), O.stored_indices(box, act, w.halo_width))
    return g


@pytest.mark.parametrize("wl", [I.config1(), I.small_shell(40, 13), I.small_shell(24, 7, aniso=False),
                                I.small_shell(33, 13).with_(center=(0.3, -0.2, 0.1)),
                                I.small_shell(40, 13).with_(hy=0.4, hz=0.65)])
def test_layout_tables_bit_exact(wl):
    _compare_tables(wl)


def test_layout_union_mask_and_ramp():
    w = I.small_shell(36, 7).with_(delta0=0.0, delta1=20.0, t_ramp=1.0, mask_mode=I.MASK_UNION)
    _compare_tables(w)
    _compare_tables(w.with_(mask_mode=I.MASK_AT_DELTA1))
    _compare_tables(w.with_(mask_mode=I.MASK_AT_DELTA0, v_cut=3.0))


@pytest.mark.parametrize("dims,p,seed", [((9, 7, 11), 0.4, 3), ((17, 16, 40), 0.1, 4), ((8, 8, 70), 0.9, 5),
                                         ((6, 6, 6), 1.1, 6)])
def test_layout_from_random_indices(dims, p, seed):
    nx, ny, nz = dims
    w = I.Workload(name="rnd", nx=nx, ny=ny, nz=nz, h=0.3, kind=I.HARMONIC)
    act = I.random_mask_lin(seed, nx, ny, nz, p)
    _compare_tables(w, active=act)


def test_layout_edge_cases():
    w = I.Workload(name="one", nx=5, ny=4, nz=3, h=0.5, kind=I.HARMONIC)
    g = _compare_tables(w, active=np.array([17], np.int64))
    assert g.n_active == 1
    # empty mask is valid
    g = P.Grid.from_workload(w.with_(v_cut=-1.0))
    assert g.n_active == 0 and g.active_indices().size == 0 and g.n_stored == 0
    assert g.layout_info().n_tiles == 0


def test_config2_counts_match_fixture():
    gold = json.load(open(os.path.join(ROOT, "tests", "golden", "counts.json")))
    w = I.config2()
    g = P.Grid.from_workload(w)
    assert g.n_active == gold[w.name]["n_active"]
    box, pot, act = oracle_objs(w)
    assert np.array_equal(g.active_indices(), act)
    assert g.n_stored == gold[w.name]["n_stored"]


def test_argument_errors():
    w = I.config1()
    with pytest.raises(P.GpeError) as e:
        P.Grid.from_workload(w.with_(h=-1.0))
    assert e.value.code == -1
    with pytest.raises(P.GpeError):
        P.Grid.from_workload(w.with_(nx=0))
    with pytest.raises(P.GpeError):
        P.Grid.from_workload(w, active=np.array([5, 3], np.int64))      # not ascending
    with pytest.raises(P.GpeError):
        P.Grid.from_workload(w, active=np.array([48 ** 3], np.int64))   # outside the box
    with pytest.raises(P.GpeError):
        P.Grid.from_workload(w.with_(halo_width=9))


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    g = P.Grid.from_workload(I.small_shell(24, 7))
    with pytest.raises(P.GpeError) as e:
        P.Sim(g, "complex128", 7, 1.0)
    assert e.value.code == -3
