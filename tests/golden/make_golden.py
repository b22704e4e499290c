"""Writes the stored expected values under tests/golden/ -- calls ONLY oracle/ and workloads/.

  python tests/golden/make_golden.py

cfg0_kn1_film.txt: BASELINE.json configs[0] (1-D gray film, Kn = 1, 200 cells, 16-pt GL,
200 source iterations); columns: x/L, dT [K], q_x [W/m^2].  The oracle behind these values
is pinned independently by tests/test_oracle_1d.py (integral-equation value 0.5532 of the
slab problem the paper validates against, ref. [59]).
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle  # noqa: E402
import workloads as W  # noqa: E402

here = os.path.dirname(os.path.abspath(__file__))
p = W.config(0)
r = oracle.RefSolver(p)
r.iterate(p.n_iter)
x = (np.arange(p.nx) + 0.5) / p.nx
np.savetxt(os.path.join(here, "cfg0_kn1_film.txt"),
           np.stack([x, r.temperature().ravel(), r.heat_flux()[0].ravel()], axis=1),
           fmt="%.17e", header="oracle-only; BASELINE.json configs[0]; x/L dT[K] qx[W/m^2]")
print("wrote cfg0_kn1_film.txt")
