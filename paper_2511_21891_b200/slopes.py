"""The two statistical numbers of the paper, measured with the library (PARITY UNPINNED: statistics of long runs).

  python -m paper_2511_21891_b200.slopes [out.json]        (one B200, about two minutes)

E4, velocity-space benchmark: 32^3, M = 128, nu = 0.25, p = 6, dt = 0.01, white-noise forcing of g_0 at
k = (0,0,1), brackets off; C_m (Eq. 27) sampled every 100 steps and averaged over three time windows, least-squares slope in
log-log over three ranges of m, two seeds, both closures (paper: -0.50 +- 0.02).
Config 3, driven turbulence (BASELINE config 3 with cfl = 0.03, Q28): 80 000 steps, E(k_perp)
(Eq. 26) sampled every 500 steps over the second half and averaged; slope over k in [2, 12] (paper: -5/3).
Only the public binding is used (Gandalf.step / hermite_spectrum / kperp_spectrum); results: profiles/r02_slopes.md."""
import json
import sys
import time

import numpy as np

from .gandalf import Gandalf
from . import workloads


def hermite_slopes(closure, seed, t_end=400.0):
    shape, M = (32, 32, 32), 128
    g = Gandalf(*shape, M=M, nu_coll=0.25, p=6.0, force_g_amp=0.0035, force_g_nz=1, seed=seed, nonlinear=0, closure=closure)
    g.set_state(np.zeros((2, 32, 32, 17)), np.zeros((M, 32, 32, 17)))
    wins = {"25-50": (25, 50), "25-200": (25, 200), "50-400": (50, 400)}
    sums = {k: [np.zeros(M), 0] for k in wins}
    for _ in range(int(round(t_end))):
        g.step(0.01, 100)
        t, c = g.time()[0], g.hermite_spectrum()
        for k, (a, b) in wins.items():
            if a <= t <= b + 1e-9:
                sums[k][0] += c
                sums[k][1] += 1
    out = {}
    for k in wins:
        cm = sums[k][0] / sums[k][1]
        for lo, hi in ((2, 20), (4, 40), (8, 64)):
            ms = np.arange(lo, hi + 1)
            out[f"{k} m{lo}-{hi}"] = round(float(np.polyfit(np.log(ms), np.log(cm[lo:hi + 1]), 1)[0]), 3)
    g.close()
    return out


def driven_spectrum_slopes(nsamples=160, every=500, nbins=44):
    prm, z, gm, run = workloads.config3()
    prm = dict(prm, cfl=0.03)
    g = Gandalf(*run["shape"], **prm)
    g.set_state(z, gm)
    acc, n, snaps = np.zeros(nbins), 0, []
    for it in range(nsamples):
        g.step(0.0, every)
        if it >= nsamples // 2:
            sp = g.kperp_spectrum(nbins)
            acc += sp
            n += 1
            if it % 20 == 0:
                snaps.append(sp)
    sp, ks, out = acc / n, np.arange(nbins), {}
    for lo, hi in ((2, 12), (3, 10), (4, 16)):
        sel = (ks >= lo) & (ks <= hi)
        out[f"avg k{lo}-{hi}"] = round(float(np.polyfit(np.log(ks[sel]), np.log(sp[sel]), 1)[0]), 3)
        out[f"snapshots k{lo}-{hi}"] = [round(float(np.polyfit(np.log(ks[sel]), np.log(s[sel]), 1)[0]), 3) for s in snaps]
    out.update(t_end=g.time()[0], E_A=float(g.energy()[0]), n_avg=n)
    g.close()
    return out


def main():
    res, t0 = {}, time.time()
    for closure in (0, 1):
        for seed in (2024, 7):
            res[f"E4 closure={closure} seed={seed}"] = hermite_slopes(closure, seed)
            print("E4", closure, seed, res[f"E4 closure={closure} seed={seed}"], flush=True)
    res["config3"] = driven_spectrum_slopes()
    print("config3", res["config3"], f"{time.time() - t0:.0f} s", flush=True)
    if len(sys.argv) > 1:
        json.dump(res, open(sys.argv[1], "w"), indent=1)


if __name__ == "__main__":
    main()
