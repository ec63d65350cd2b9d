"""Writes tests/golden/tiny_ps_populations.txt: site populations after each of the 20 TDVP-PS
steps of BASELINE.json configs[0] (M = 16, k = 10, dt = 10 fs), computed by oracle/ ONLY.
Run from the repo root:  python tests/golden/make_golden.py"""
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
import synthetic_inputs as si                      # noqa: E402
from oracle import model, observables, tdvp_ps      # noqa: E402

cfg = si.CONFIGS["tiny"]
params = si.draw_vibronic_params(cfg)
mpo = model.build_mpo(params)
mps = si.padded_product_mps(si.site_dims(params), si.initial_occupations(params), cfg.M, cfg.pad_seed)
st = tdvp_ps.PSState(mpo, mps)
rows = []
for _ in range(cfg.n_steps):
    tdvp_ps.step_ps(st, cfg.dt_fs, cfg.krylov_dim)
    rows.append(observables.populations(st.mps))
out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "tiny_ps_populations.txt")
np.savetxt(out, np.array(rows), fmt="%.17e",
           header="oracle TDVP-PS populations, config 'tiny' (PAPER.md Eq. 42-44; SURVEY.md 8(d) config 1)")
