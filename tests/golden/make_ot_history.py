"""Writes tests/golden/ot_history_oracle.txt: the ORACLE's energy history of BASELINE.json config 1
(Orszag-Tang, 128x128x2, dt=1e-3, 2000 steps), every 50th step.  Calls only oracle/ and the seeded
input module.  Run from the repo root:  python tests/golden/make_ot_history.py   (~80 s on 8 cores)"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import Oracle  # noqa: E402
from paper_2511_21891_b200 import synth  # noqa: E402

n = 128
o = Oracle(n, n, 2)
o.set_state(synth.orszag_tang(n, n, 2))
o.step(1e-3, 2000)
h = o.energy_history()
rows = h[49::50]
out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "ot_history_oracle.txt")
with open(out, "w") as fh:
    fh.write("# oracle energy history, config 1 (Orszag-Tang 128x128x2, dt=1e-3), steps 50,100,...,2000\n")
    fh.write("# written by tests/golden/make_ot_history.py (oracle only).  columns: step t E_A E+ E- E_kin E_mag W_g\n")
    for i, r in enumerate(rows):
        fh.write(f"{50 * (i + 1)} " + " ".join(repr(float(v)) for v in r) + "\n")
print("wrote", out)
