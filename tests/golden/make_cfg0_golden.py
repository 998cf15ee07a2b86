"""Writes tests/golden/cfg0_first4096.json.  Calls only oracle/ and the input generator;
never the CUDA path.  Run from the repo root:  python tests/golden/make_cfg0_golden.py
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle as O  # noqa: E402
from paper_1908_02219_b200 import workloads as W  # noqa: E402

cfg = W.scaled(W.CONFIGS["cfg0"], 4096)
m = W.generate(cfg, workers=1)
g = O.geom(cfg.ns, cfg.ntheta, cfg.nphi, rho_star=cfg.rho_star)
rho, _, npts = O.deposit(g, O.policy_fixed(4), *(m[f] for f in W.FIELDS), current=False)
nodes = [(3, 0, 0), (9, 16, 8), (15, 31, 15), (5, 7, 3), (12, 20, 1), (2, 5, 9)]
out = dict(source="oracle/orb_oracle.c via tests/golden/make_cfg0_golden.py",
           config="cfg0 (BASELINE.json configs[0]), first 4096 markers, fixed N_L=4, charge only",
           n_points=npts, sum=float(rho.sum()), max_abs=float(np.abs(rho).max()),
           nodes=nodes, values=[float(rho[n]) for n in nodes])
with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg0_first4096.json"), "w") as f:
    json.dump(out, f, indent=1)
print(out)
