"""Writes tests/golden/cfg1_first8.txt: E_loc and ln psi of the first 8 samples of config 1.

Calls ONLY oracle/ and the seeded input generators (never the CUDA path).  Run from the repo root:
    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import nk_oracle as orc                      # noqa: E402
from paper_2112_10526_b200 import inputs as inp          # noqa: E402

p = inp.make_config(1, n_samples=8)
e, lp = orc.local_energy(p.kind, p.sigma, p.bonds, p.colors, p.J, p.h, p.W, p.a, p.b)
np.savetxt(os.path.join(ROOT, "tests", "golden", "cfg1_first8.txt"), np.stack([e, lp], axis=1), fmt="%.17g",
           header="config 1 (BASELINE.json configs[0]), first 8 samples: E_loc, ln psi (float64 oracle, Eq. (12) L652)\n"
                  "written by tests/golden/make_golden.py; regression guard only, the pins are in test_oracle_pins.py")
