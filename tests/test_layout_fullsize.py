"""Bit-exact active set and layout tables at BASELINE.json's FULL sizes (north_star: "active-set and neighbour
tables must be bit-exact ... on all five configs"; PAPER.md:50-58 mask, :81-85 tables): the library's host builder
(csrc/gpe_layout.cpp, no CUDA call) against the oracle's independent Python builder, every table, every entry,
for configs 3a (union mask over the ramp), 3b (final shell), 4 (1024^3 ellipsoid, tips clipped by the box face)
and the 1e7-point shell of the configs[4] sweep.  The point counts are also pinned to the numbers the survey
session computed with its own script (SURVEY.md:237-241) and to tests/golden/counts.json (written by
tests/golden/make_counts.py from the oracle only).  The comparison itself is host-only; it is part of the `-m gpu` run
because it takes minutes (the CPU suite is sized for a few minutes in all): run it anywhere with
`pytest tests/test_layout_fullsize.py -m gpu` on a machine with a GPU, or drop the marker."""
import json
import os

import numpy as np
import pytest

import gpe_inputs as I
import paper_2603_05447_b200 as P
from oracle import gpe_oracle as O
from helpers import oracle_objs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
GOLD = json.load(open(os.path.join(ROOT, "tests", "golden", "counts.json")))

# SURVEY.md:237-241 (section 8, "Workload sizes"): n_a = |M| and the star halo (R = 2) of each config
SURVEY_COUNTS = {
    "cfg3a_ramp_union_512": (38495288, 922496),
    "cfg3b_ramp_final_512": (9730864, 1671856),
    "cfg4_ellipsoid_1024_c128": (31523416, 5942744),
}

pytestmark = [pytest.mark.gpu, pytest.mark.slow]

CASES = [I.config3(True), I.config3(False), I.config4(), I.config5_shell(1e7, 24, 13, "complex128", 4)]


@pytest.mark.parametrize("w", CASES, ids=[w.name for w in CASES])
def test_fullsize_layout_bit_exact(w):
    box, pot, act = oracle_objs(w)                       # plane-by-plane NumPy mask (reading R2: fixed order, no FMA)
    g = P.Grid.from_workload(w)
    gold = GOLD[w.name]
    assert g.n_active == act.size == gold["n_active"]
    if w.name in SURVEY_COUNTS:
        assert act.size == SURVEY_COUNTS[w.name][0]
    assert np.array_equal(g.active_indices(), act)
    ref = O.tile_layout(box, act, 8, 8, 32)
    got = g.layout_tables()
    info = g.layout_info()
    assert (info.n_tiles, info.n_slabs, info.n_work) == (gold["n_tiles"], gold["n_slabs"], gold["n_work"])
    for k, v in ref.items():
        assert np.array_equal(np.asarray(v), np.asarray(got[k])), k
    del ref, got
    # stored set S = M + star halo: the count against the fixture (the oracle wrote it) and the survey's halo size;
    # the index arrays themselves where the oracle's np.unique pass is short
    assert g.n_stored == gold["n_stored"]
    if w.name in SURVEY_COUNTS:
        assert g.n_stored - act.size == SURVEY_COUNTS[w.name][1]
    if act.size < 2e7:
        assert np.array_equal(g.stored_indices(), O.stored_indices(box, act, w.halo_width))
