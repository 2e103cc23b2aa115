"""Writes tests/golden/counts.json (active / stored point counts and layout-table sizes of BASELINE configs 1-4
and of the 1e7-point shell of the configs[4] sweep).

Calls only oracle/ and gpe_inputs; never the CUDA path.  Run: python tests/golden/make_counts.py
"""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import gpe_oracle as O  # noqa: E402
import gpe_inputs as I  # noqa: E402

out = {}
for w in (I.config1(), I.config2(), I.config3(True), I.config3(False), I.config4(), I.config5_shell(1e7, 24, 13, "complex128", 4)):
    box = O.Box(w.nx, w.ny, w.nz, w.h, w.center)
    pot = O.Potential(w.kind, w.ax, w.ay, w.az, w.delta0, w.delta1, w.t_ramp, w.omega)
    act = O.active_indices(box, pot, w.v_cut, w.mask_mode)
    st = O.stored_indices(box, act, w.halo_width)
    lay = O.tile_layout(box, act)
    out[w.name] = {"n_active": int(act.size), "n_stored": int(st.size), "n_tiles": int(lay["n_tiles"]),
                   "n_slabs": int(lay["slab_mask"].size), "n_work": int(lay["wi_tile"].size)}
json.dump(out, open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "counts.json"), "w"), indent=1)
print(out)
