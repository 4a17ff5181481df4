"""Writes tests/golden/config2_history_oracle.txt: the ORACLE's run of BASELINE.json config 2 as specified (64x64x32, M = 16,
dt = 5e-4, all 200 steps): the energy record every 10th step and 48 sampled coefficients of the final state.  Calls only
oracle/ and the seeded input modules.  Run from the repo root:  python tests/golden/make_config2_history.py  (~6 min, 16 cores)"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import Oracle  # noqa: E402
from paper_2511_21891_b200.workloads import config2  # noqa: E402


def sample_indices(nfields, shape_half, n=48, seed=20002):
    """(field, iz, iy, ix) of the sampled coefficients: retained modes only (|n| <= N/3), fixed by the seed."""
    nz, ny, hx = shape_half
    rng = np.random.default_rng(seed)
    out = []
    while len(out) < n:
        f, iz, iy, ix = int(rng.integers(nfields)), int(rng.integers(nz)), int(rng.integers(ny)), int(rng.integers(hx))
        mz, my = (iz if iz < nz // 2 else iz - nz), (iy if iy < ny // 2 else iy - ny)
        if 3 * abs(mz) <= nz and 3 * abs(my) <= ny and 3 * ix <= 2 * (hx - 1):
            out.append((f, iz, iy, ix))
    return out


if __name__ == "__main__":
    prm, z, g, run = config2()
    o = Oracle(*run["shape"], **prm)
    o.set_state(z, g)
    o.step(run["dt"], run["steps"])
    h = o.energy_history()
    zeta, gm = o.get_state()
    allf = np.concatenate([zeta, gm])
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config2_history_oracle.txt")
    with open(out, "w") as fh:
        fh.write("# oracle run of BASELINE config 2 (64x64x32, M=16, dt=5e-4, 200 steps); written by tests/golden/make_config2_history.py (oracle only)\n")
        fh.write("# H rows: step t E_A E+ E- E_kin E_mag W_g (every 10th step);  S rows: field iz iy ix re im of the final state (zeta+-, then g_m)\n")
        for i in range(9, h.shape[0], 10):
            fh.write(f"H {i + 1} " + " ".join(repr(float(v)) for v in h[i]) + "\n")
        for (f, iz, iy, ix) in sample_indices(allf.shape[0], allf.shape[1:]):
            v = allf[f, iz, iy, ix]
            fh.write(f"S {f} {iz} {iy} {ix} {float(v.real)!r} {float(v.imag)!r}\n")
    print("wrote", out)
