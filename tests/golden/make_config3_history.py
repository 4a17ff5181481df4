"""Writes tests/golden/config3_history_oracle.txt: the ORACLE's run of BASELINE.json config 3 at its full size (128x128x64,
M = 32, white-noise forcing of Eq. 25, CFL dt of Eq. 16, kperp^8 and kz^8 hyperdissipation) over the window
SURVEY.md 8(d) names, "the first 10 and 100 steps":
  run A  config 3 as written (C = 0.3): 10 steps -- record and 48 sampled coefficients at step 10;
  run B  the same with C = 0.03: 100 steps -- records every 10th step, 48 sampled coefficients at steps 10 and 100.
         As written (C = 0.3, M = 32) the explicit RK2 of the Hermite couplings is unstable and W_g overflows within ~40 steps
         in the oracle and in the CUDA path alike (Q28), so the 100-step window uses the stable C.
Calls only oracle/ and the seeded input modules.  Run from the repo root:  python tests/golden/make_config3_history.py
(about an hour on 8 cores: the oracle needs 20-40 s per step at this size)."""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import Oracle  # noqa: E402
from paper_2511_21891_b200.workloads import config3  # noqa: E402

CFL_STABLE = 0.03


def sample_indices(nfields, shape_half, n=48, seed=30003):
    """(field, iz, iy, ix) of the sampled coefficients: retained modes only (3|n| <= N), fixed by the seed; the first 12 are
    drawn from zeta+- so that both the potentials and the moments are covered."""
    nz, ny, hx = shape_half
    rng = np.random.default_rng(seed)
    out = []
    while len(out) < n:
        f = int(rng.integers(2)) if len(out) < 12 else int(rng.integers(nfields))
        iz, iy, ix = int(rng.integers(nz)), int(rng.integers(ny)), int(rng.integers(hx))
        mz, my = (iz if iz < nz // 2 else iz - nz), (iy if iy < ny // 2 else iy - ny)
        if 3 * abs(mz) <= nz and 3 * abs(my) <= ny and 3 * ix <= 2 * (hx - 1):
            out.append((f, iz, iy, ix))
    return out


def dump(fh, tag, o, every, after):
    """T row, the H rows of every `every`-th step later than step `after`, and the S rows of the current state."""
    t, step, last_dt = o.time()
    h = o.energy_history()
    fh.write(f"T {tag} {step} {float(t)!r} {float(last_dt)!r}\n")
    for i in range(every - 1, h.shape[0], every):
        if i + 1 > after:
            fh.write(f"H {tag} {i + 1} " + " ".join(repr(float(v)) for v in h[i]) + "\n")
    zeta, gm = o.get_state()
    allf = np.concatenate([zeta, gm])
    for (f, iz, iy, ix) in sample_indices(allf.shape[0], allf.shape[1:]):
        v = allf[f, iz, iy, ix]
        fh.write(f"S {tag} {step} {f} {iz} {iy} {ix} {float(v.real)!r} {float(v.imag)!r}\n")
    fh.flush()


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config3_history_oracle.txt")
    prm, z, g, run = config3()
    assert run["shape"] == (128, 128, 64) and prm["M"] == 32 and prm["cfl"] == 0.3
    t0 = time.time()
    with open(out, "w") as fh:
        fh.write("# oracle runs of BASELINE config 3 (128x128x64, M=32, forcing, CFL dt, kperp^8 / kz^8 hyperdissipation); written by "
                 "tests/golden/make_config3_history.py (oracle only)\n")
        fh.write("# run A: cfl = 0.3 (as written), 10 steps;  run B: cfl = 0.03 (stable, DESIGN.md Q28), 100 steps\n")
        fh.write("# T rows: run step t last_dt;  H rows: run step t E_A E+ E- E_kin E_mag W_g;  S rows: run step field iz iy ix re im (zeta+-, then g_m)\n")
        o = Oracle(*run["shape"], **prm)
        o.set_state(z, g)
        o.step(0.0, 10)
        dump(fh, "A", o, 10, 0)
        print("run A done", round(time.time() - t0), "s", flush=True)
        del o
        o = Oracle(*run["shape"], **dict(prm, cfl=CFL_STABLE))
        o.set_state(z, g)
        for k in range(10):
            o.step(0.0, 10)
            if k in (0, 9):
                dump(fh, "B", o, 10, 0 if k == 0 else 10)
            print("run B step", 10 * (k + 1), round(time.time() - t0), "s", flush=True)
    print("wrote", out)
