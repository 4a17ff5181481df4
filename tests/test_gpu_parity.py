"""-m gpu: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  Tolerances are BASELINE.json north_star's: 1e-12 relative L2 per RHS evaluation,
1e-10 after 10 steps, 1e-9 on energy histories."""
import os

import numpy as np
import pytest

from paper_2511_21891_b200.workloads import config0, config1, config2, config3, rel_l2
from paper_2511_21891_b200 import synth

pytestmark = pytest.mark.gpu

TOL_RHS, TOL_10STEPS, TOL_ENERGY = 1e-12, 1e-10, 1e-9


def _pair(shape, prm):
    from oracle import Oracle
    from paper_2511_21891_b200.gandalf import Gandalf
    nx, ny, nz = shape
    o = Oracle(nx, ny, nz, **prm)
    g = Gandalf(nx, ny, nz, **prm)
    return o, g


def _check_rhs(o, g, tol=TOL_RHS):
    dw_o, dg_o = o.rhs()
    dw_g, dg_g = g.rhs()
    for a in range(2):
        assert rel_l2(dw_g[a], dw_o[a]) <= tol, ("dw", a, rel_l2(dw_g[a], dw_o[a]))
    if o.M:
        # per moment, relative to the largest moment's RHS norm (moments that start at zero have tiny RHS)
        ref = max(np.linalg.norm(dg_o[m]) for m in range(o.M))
        for m in range(o.M):
            assert np.linalg.norm(dg_g[m] - dg_o[m]) <= tol * ref, ("dg", m)
        assert rel_l2(dg_g, dg_o) <= tol
    # removed modes are exactly zero on the GPU side too
    assert np.count_nonzero(dw_g[:, :, :, o.nx // 3 + 1:]) == 0


def _check_state(o, g, tol):
    zo, go = o.get_state()
    zg, gg = g.get_state()
    assert rel_l2(zg, zo) <= tol, rel_l2(zg, zo)
    if o.M:
        assert rel_l2(gg, go) <= tol, rel_l2(gg, go)


def _check_history(o, g, tol=TOL_ENERGY):
    ho, hg = o.energy_history(), g.energy_history()
    assert ho.shape == hg.shape and ho.shape[0] > 0
    assert np.abs(hg[:, 0] - ho[:, 0]).max() <= 1e-12 * max(1.0, abs(ho[-1, 0]))
    scale = np.abs(ho[:, 1:]).max(axis=0)
    for k in range(6):
        if scale[k] > 0:
            assert np.abs(hg[:, 1 + k] - ho[:, 1 + k]).max() <= tol * scale[k], k


def test_config0_rmhd_decay():
    prm, z, _, run = config0()
    o, g = _pair(run["shape"], prm)
    o.set_state(z); g.set_state(z)
    _check_state(o, g, 1e-14)
    assert np.abs(g.energy() - o.energy()).max() <= 1e-13
    _check_rhs(o, g)
    o.step(run["dt"], 10); g.step(run["dt"], 10)
    _check_state(o, g, TOL_10STEPS)
    o.step(run["dt"], 90); g.step(run["dt"], 90)
    _check_state(o, g, 1e-9)
    _check_history(o, g)
    assert g.time()[1] == 100 and abs(g.time()[0] - 0.1) < 1e-12


def test_config2_krmhd_hermite():
    prm, z, gm, run = config2()
    o, g = _pair(run["shape"], prm)
    o.set_state(z, gm); g.set_state(z, gm)
    _check_rhs(o, g)
    o.step(run["dt"], 10); g.step(run["dt"], 10)
    _check_state(o, g, TOL_10STEPS)
    _check_rhs(o, g)                      # RHS on an evolved state (all moments populated up to m=10)
    o.step(run["dt"], 30); g.step(run["dt"], 30)
    _check_history(o, g)


def test_config2_all_200_steps_against_the_oracle_written_golden():
    """BASELINE config 2 AS SPECIFIED (64x64x32, M = 16, dt = 5e-4, all 200 steps): energy record every 10th step (1e-9) and 48
    sampled coefficients of the final state against tests/golden/config2_history_oracle.txt, which
    tests/golden/make_config2_history.py wrote from the oracle alone (six minutes of CPU: too slow to repeat in the test)."""
    import os
    from paper_2511_21891_b200.gandalf import Gandalf
    prm, z, gm, run = config2()
    g = Gandalf(*run["shape"], **prm)
    g.set_state(z, gm)
    g.step(run["dt"], run["steps"])
    hist = g.energy_history()
    zeta, gg = g.get_state()
    allf = np.concatenate([zeta, gg])
    nH = nS = 0
    for ln in open(os.path.join(os.path.dirname(__file__), "golden", "config2_history_oracle.txt")):
        if ln.startswith("H "):
            t = ln.split()
            step, want = int(t[1]), np.array([float(x) for x in t[2:]])
            got = hist[step - 1]
            assert abs(got[0] - want[0]) <= 1e-12 and np.abs(got[1:] - want[1:]).max() <= 1e-9 * max(1.0, np.abs(want[1:]).max()), step
            nH += 1
        elif ln.startswith("S "):
            t = ln.split()
            f, iz, iy, ix = (int(x) for x in t[1:5])
            want = complex(float(t[5]), float(t[6]))
            assert abs(allf[f, iz, iy, ix] - want) <= 1e-9 * np.abs(allf[f]).max(), (f, iz, iy, ix)
            nS += 1
    assert nH == 20 and nS == 48 and hist.shape[0] == 200


@pytest.mark.parametrize("shape,M", [((8, 8, 2), 0), ((16, 8, 4), 1), ((8, 16, 8), 2), ((32, 64, 16), 3),
                                     ((64, 32, 8), 5), ((128, 16, 4), 2), ((16, 128, 4), 2), ((256, 8, 2), 1),
                                     ((8, 256, 2), 1), ((512, 8, 2), 1), ((8, 512, 2), 2), ((8, 8, 64), 2),
                                     ((8, 8, 128), 1), ((8, 8, 256), 1), ((8, 8, 512), 1), ((16, 16, 32), 4)])
def test_rhs_all_transform_sizes_dense_state(shape, M):
    """Every FFT length on every axis, ragged tails, dense random input incl. modes set_state must project out."""
    nx, ny, nz = shape
    prm = dict(M=M)
    o, g = _pair(shape, prm)
    # rough |n|^-1.5 spectrum on every mode (w = -kperp^2 zeta GROWS with k): the 1e-12 bar holds here since the x-pass
    # transforms (A, bscale*B) -- round 1 needed |n|^-3 / |n|^-4 because B's round-off floor was set by A
    dec = 1.5
    z = synth.dense_random(nx, ny, nz, 2, seed=nx + 3 * ny + 7 * nz, decay=dec)
    gm = synth.dense_random(nx, ny, nz, M, seed=99 + nx, decay=dec) if M else None
    o.set_state(z, gm); g.set_state(z, gm)
    _check_state(o, g, 1e-14)
    _check_rhs(o, g)
    o.step(1e-3, 2); g.step(1e-3, 2)
    _check_state(o, g, TOL_10STEPS)


@pytest.mark.parametrize("opts", [dict(if_variant=1), dict(closure=1), dict(g_sign=-1), dict(hermite_coeff=1),
                                  dict(nonlinear=0), dict(eta=0.5, r=3, eta_normalized=1, eta_z=0.2, r_z=2, eta_g=0.3,
                                                          nu_coll=0.7, p=1.5),
                                  dict(Lx=3.0, Ly=5.0, Lz=11.0)])
def test_variants_and_options(opts):
    shape, M = (32, 16, 8), 4
    prm = dict(M=M, **opts)
    o, g = _pair(shape, prm)
    z = synth.dense_random(*shape, 2, seed=5)
    gm = synth.dense_random(*shape, M, seed=6)
    o.set_state(z, gm); g.set_state(z, gm)
    _check_rhs(o, g)
    o.step(2e-3, 10); g.step(2e-3, 10)
    _check_state(o, g, TOL_10STEPS)
    _check_history(o, g)


def test_rmhd_with_va_not_one():
    shape = (16, 16, 8)
    o, g = _pair(shape, dict(M=0, vA=2.5))
    z = synth.dense_random(*shape, 2, seed=8)
    o.set_state(z); g.set_state(z)
    o.step(5e-3, 10); g.step(5e-3, 10)
    _check_state(o, g, TOL_10STEPS)


def test_alfven_wave_exact_on_gpu():
    from paper_2511_21891_b200.gandalf import Gandalf
    g = Gandalf(32, 32, 16)
    z0 = synth.single_mode(32, 32, 16, (1, 0, 1), 0.01)
    g.set_state(z0)
    T = 2 * np.pi
    g.step(T / 4, 4)
    z, _ = g.get_state()
    assert abs(z[0, 1, 0, 1] - 0.01) <= 1e-16          # one full period: back to the start
    z[0, 1, 0, 1] = 0
    assert np.abs(z).max() == 0.0


def test_config3_forcing_and_cfl_window():
    """Scaled-down config 3 (forcing + adaptive CFL dt + k_z and k_perp hyperdissipation): trajectory parity
    over the first steps (Q20)."""
    prm, z, gm, run = config3(32, 32, 16, 4, eta=50.0)
    o, g = _pair(run["shape"], prm)
    o.set_state(z, gm); g.set_state(z, gm)
    o.step(0.0, 10); g.step(0.0, 10)
    to, tg = o.time(), g.time()
    assert tg[1] == 10 and abs(tg[0] - to[0]) <= 1e-12 * to[0] and abs(tg[2] - to[2]) <= 1e-12 * to[2]
    _check_state(o, g, TOL_10STEPS)
    _check_history(o, g)
    so, sg = o.kperp_spectrum(24), g.kperp_spectrum(24)
    assert np.abs(sg - so).max() <= 1e-10 * so.max()
    assert abs(sg.sum() - g.energy()[0]) <= 1e-12 * sg.sum()
    sl_o, sl_g = o.kperp_spectrum(24, True), g.kperp_spectrum(24, True)
    assert np.abs(sl_g - sl_o).max() <= 1e-10 * sl_o.max()


def test_config1_orszag_tang_energy_history():
    prm, z, _, run = config1()
    o, g = _pair(run["shape"], prm)
    o.set_state(z); g.set_state(z)
    e0 = g.energy()
    assert abs(e0[0] - 4.0) <= 1e-13 and abs(e0[3] - 2.0) <= 1e-13 and abs(e0[4] - 2.0) <= 1e-13
    n = 2000
    g.step(run["dt"], n)
    hg = g.energy_history()
    # BASELINE's IC has twice the paper's amplitude: the paper's 2 tau_A window is t in [0,1] here (golden/orszag_tang.txt)
    drift = np.abs(hg[:1000, 1] / 4.0 - 1.0).max()
    assert drift <= 1e-5, drift                      # paper: 1.6e-6 at 128^2 x 2
    o.step(run["dt"], 300)                           # oracle live over the first 300 steps ...
    ho = o.energy_history()
    assert np.abs(hg[:300, 1:] - ho[:, 1:]).max() <= TOL_ENERGY * 4.0
    gold = np.loadtxt(os.path.join(os.path.dirname(__file__), "golden", "ot_history_oracle.txt"))
    idx = gold[:, 0].astype(int) - 1                 # ... and its stored full history (written by make_ot_history.py)
    assert np.abs(hg[idx, 1:] - gold[:, 2:]).max() <= TOL_ENERGY * 4.0
    assert np.abs(hg[idx, 0] - gold[:, 1]).max() <= 1e-12
    assert hg[-1, 5] / hg[-1, 4] > 1.0               # selective decay direction


def test_device_pointer_entry_points():
    import torch
    from oracle import Oracle
    from paper_2511_21891_b200.gandalf import Gandalf
    shape, M = (32, 32, 8), 3
    z = synth.dense_random(*shape, 2, seed=1)
    gm = synth.dense_random(*shape, M, seed=2)
    g = Gandalf(*shape, M=M)
    zt = torch.from_numpy(z).cuda(); gt = torch.from_numpy(gm).cuda()
    g.set_state(zt, gt)
    dw, dg = g.rhs(device=True)
    torch.cuda.synchronize()
    o = Oracle(*shape, M=M)
    o.set_state(z, gm)
    dw_o, dg_o = o.rhs()
    assert rel_l2(dw.cpu().numpy(), dw_o) <= TOL_RHS and rel_l2(dg.cpu().numpy(), dg_o) <= TOL_RHS
    # a non-default stream supplied by torch
    s = torch.cuda.Stream()
    g2 = Gandalf(*shape, M=M, stream=s.cuda_stream)
    with torch.cuda.stream(s):
        g2.set_state(zt, gt)
        g2.step(1e-3, 3)
    zs, gs = g2.get_state()
    g.step(1e-3, 3)
    z1, g1 = g.get_state()
    assert np.array_equal(zs, z1) and np.array_equal(gs, g1)      # bit-reproducible across contexts/streams


def test_nonfinite_is_reported():
    from paper_2511_21891_b200.gandalf import Gandalf, GandalfError, ERR_NONFINITE
    g = Gandalf(16, 16, 4)
    z = synth.dense_random(16, 16, 4, 2, seed=3) * 1e200
    g.set_state(z)
    g.step(1.0, 3)
    with pytest.raises(GandalfError) as ei:
        g.energy_history()
    assert ei.value.code == ERR_NONFINITE


def test_launch_count_and_kernel_timing():
    from paper_2511_21891_b200.gandalf import Gandalf
    prm, z, gm, run = config2(32, 32, 16, 4)
    g = Gandalf(*run["shape"], **prm)
    g.set_state(z, gm)
    n0 = g.launch_count()
    g.kernel_timing(True)
    g.step(run["dt"], 2)
    kt = g.kernel_times()
    # per step: 2 x (P1 Elsasser + P1 moments, P2, P3 pair + P3 moments, P4) + dt + factor tables + 2 energy kernels
    assert g.launch_count() - n0 == 2 * 16
    assert kt["x_pass_P2"][1] == 4 and kt["x_pass_P2"][0] > 0
    assert kt["z_step_P4"][1] == 4 and kt["z_step_P4"][0] > 0


def test_hermite_and_parallel_spectra_match_oracle():
    prm, z, gm, run = config2(32, 32, 16, 6)
    o, g = _pair(run["shape"], prm)
    o.set_state(z, gm); g.set_state(z, gm)
    o.step(run["dt"], 5); g.step(run["dt"], 5)
    co, cg = o.hermite_spectrum(), g.hermite_spectrum()
    assert np.abs(cg - co).max() <= 1e-10 * co.max()
    ko, kg = o.kpar_spectrum(9), g.kpar_spectrum(9)
    assert np.abs(kg - ko).max() <= 1e-10 * ko.max()
    assert abs(kg.sum() - g.energy()[0]) <= 1e-12 * kg.sum() and abs(cg.sum() - 2 * g.energy()[5]) <= 1e-12 * cg.sum()


def test_velocity_space_benchmark_forced_g0_large_M():
    """SURVEY 8(f) rank 1 / PAPER.md:594: 32^3, M = 128, hyper-collisions nu = 0.25, p = 6, white-noise forcing of g_0 at
    k = (0,0,1), dt = 0.01 -- here with the brackets ON and a small Alfvenic field so that the Hermite sliding window of the
    x-pass runs at M = 128; trajectory parity over 20 steps and the Hermite spectrum."""
    shape, M = (32, 32, 32), 128
    prm = dict(M=M, nu_coll=0.25, p=6.0, force_g_amp=0.0035, force_g_nz=1, seed=99)
    o, g = _pair(shape, prm)
    z = 0.1 * synth.random_zeta(*shape, 5000)
    gm = synth.random_g(*shape, M, 5001, total=1e-4)
    o.set_state(z, gm); g.set_state(z, gm)
    _check_rhs(o, g)
    o.step(0.01, 20); g.step(0.01, 20)
    _check_state(o, g, TOL_10STEPS)
    _check_history(o, g)
    co, cg = o.hermite_spectrum(), g.hermite_spectrum()
    assert np.abs(cg - co).max() <= 1e-10 * co.max()


def test_velocity_space_benchmark_linear_cascade_slope_reported():
    """The linear phase-mixing run itself (brackets off, 20 000 steps to t = 200): the time-averaged C_m is reported with its
    fitted slope over m in [2, 20] and [8, 64] (paper: -0.50 +- 0.02, PAPER.md:617 -- a statistical result: PARITY UNPINNED,
    DESIGN.md section 7).  Round 1 reported -0.38 from 24 samples in t in [25, 50]; the white-noise forcing needs a longer
    average: over [25, 200] two seeds and both closures give -0.47 .. -0.49 on [2, 20] and -0.50 .. -0.51 on [8, 64]
    (BASELINE.md section 5).  Gated on the GPU/oracle agreement of the first 200 steps and on a loose band around -1/2."""
    from paper_2511_21891_b200.gandalf import Gandalf
    shape, M = (32, 32, 32), 128
    prm = dict(M=M, nu_coll=0.25, p=6.0, force_g_amp=0.0035, force_g_nz=1, seed=2024, nonlinear=0)
    o, g = _pair(shape, prm)
    zz = np.zeros((2, 32, 32, 17)); gz = np.zeros((M, 32, 32, 17))
    o.set_state(zz, gz); g.set_state(zz, gz)
    o.step(0.01, 200); g.step(0.01, 200)
    assert np.abs(g.hermite_spectrum() - o.hermite_spectrum()).max() <= 1e-10 * o.hermite_spectrum().max()
    acc, n = np.zeros(M), 0
    for _ in range(198):
        g.step(0.01, 100)
        if g.time()[0] >= 25.0:
            acc += g.hermite_spectrum(); n += 1
    cm = acc / n
    s1 = np.polyfit(np.log(np.arange(2, 21)), np.log(cm[2:21]), 1)[0]
    s2 = np.polyfit(np.log(np.arange(8, 65)), np.log(cm[8:65]), 1)[0]
    print(f"velocity-space benchmark: time-averaged C_m slope, t in [25,200]: {s1:.3f} over m in [2,20], {s2:.3f} over [8,64] "
          f"(paper: -0.50 +- 0.02)")
    assert np.isfinite(cm).all() and cm[2] > cm[20] > cm[100]
    assert -0.58 < s1 < -0.40 and -0.58 < s2 < -0.42


def test_truncation_ratio_matches_oracle():
    """E_M / E_total (Q32) after a few steps, one and two species."""
    for extra in (dict(), dict(nspecies=2)):
        prm, z, gm, run = config2(32, 32, 16, 6)
        prm = dict(prm, **extra)
        if extra:
            gm = np.concatenate([gm, 0.5 * gm])
        o, g = _pair(run["shape"], prm)
        o.set_state(z, gm); g.set_state(z, gm)
        o.step(run["dt"], 5); g.step(run["dt"], 5)
        ro, rg = o.truncation_ratio(), g.truncation_ratio()
        assert ro > 0 and abs(rg - ro) <= 1e-9 * ro


def test_repeated_runs_are_bit_identical():
    """No result depends on CTA scheduling: fixed-order reductions, no floating-point atomics (the CFL maximum is an
    order-independent atomicMax), persistent kernels that assign work by index.  Two runs of config 3 (forcing + CFL dt)
    must agree bit for bit -- also a race check for the TMA / mbarrier pipelines."""
    from paper_2511_21891_b200.gandalf import Gandalf
    prm, z, gm, run = config3(32, 32, 16, 6)
    outs = []
    for _ in range(2):
        g = Gandalf(*run["shape"], **prm)
        g.set_state(z, gm)
        g.step(0.0, 12)
        zz, gg = g.get_state()
        outs.append((zz.copy(), gg.copy(), g.energy_history().copy()))
        g.close()
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])
    assert np.array_equal(outs[0][2], outs[1][2])


@pytest.mark.parametrize("M,closure", [(3, 0), (4, 1), (1, 0)])
def test_two_species_match_oracle(M, closure):
    """nspecies = 2: g^+ and g^- share the Phi, Psi lines of the fused row pass; the species must not
    couple through the Hermite sliding window (x-pass) or the streaming stencil (P4)."""
    shape = (32, 32, 16)
    prm = dict(M=M, nspecies=2, closure=closure, nu_coll=0.5, p=2.0, eta=0.5, r=2, eta_normalized=1, eta_g=0.5)
    o, g = _pair(shape, prm)
    z = synth.random_zeta(*shape, 6000)
    gm = np.concatenate([synth.random_g(*shape, M, 6001, total=0.01, filled=min(2, M)),
                         synth.random_g(*shape, M, 6002, total=0.02, filled=min(2, M))])
    o.set_state(z, gm); g.set_state(z, gm)
    _check_rhs(o, g)
    o.step(5e-4, 10); g.step(5e-4, 10)
    _check_state(o, g, TOL_10STEPS)
    _check_history(o, g)
    assert np.abs(g.hermite_spectrum() - o.hermite_spectrum()).max() <= 1e-10 * o.hermite_spectrum().max()


def test_config3_full_size_first_steps():
    """BASELINE config 3 at its full size (128x128x64, M=32, forcing, CFL dt, k_perp^8 and k_z^8 hyperdissipation): the first
    two steps against the oracle on the same grid (the oracle needs ~15-30 s per step there; Q20)."""
    prm, z, gm, run = config3()
    assert run["shape"] == (128, 128, 64) and prm["M"] == 32
    o, g = _pair(run["shape"], prm)
    o.set_state(z, gm); g.set_state(z, gm)
    o.step(0.0, 2); g.step(0.0, 2)
    to, tg = o.time(), g.time()
    assert abs(tg[0] - to[0]) <= 1e-12 * to[0] and abs(tg[2] - to[2]) <= 1e-12 * to[2]
    _check_state(o, g, TOL_10STEPS)
    _check_history(o, g)


def _golden_rows(name):
    import os
    rows = {"T": [], "H": [], "S": []}
    for ln in open(os.path.join(os.path.dirname(__file__), "golden", name)):
        t = ln.split()
        if t and t[0] in rows:
            rows[t[0]].append(t[1:])
    return rows


def test_config3_full_size_10_and_100_steps_against_the_oracle_written_golden():
    """BASELINE config 3 at its full size over the window SURVEY.md 8(d) names ("the first 10 and 100 steps"), against
    tests/golden/config3_history_oracle.txt, which tests/golden/make_config3_history.py wrote from the oracle alone (about an
    hour of CPU: too slow to repeat here).  Run A is the config as written (C = 0.3), 10 steps; run B uses C = 0.03 for the
    100-step window, because as written the run overflows within ~40 steps in the oracle and here alike (Q28).
    Compared: time and the CFL dt of the last step (1e-12), the energy records (1e-9), 48 sampled coefficients of zeta+- and
    g_m at step 10 (1e-10 of the largest coefficient of the potentials / of all moments) and at step 100 (1e-9)."""
    from paper_2511_21891_b200.gandalf import Gandalf
    prm, z, gm, run = config3()
    assert run["shape"] == (128, 128, 64) and prm["M"] == 32 and prm["cfl"] == 0.3
    rows = _golden_rows("config3_history_oracle.txt")
    seen = {"T": 0, "H": 0, "S": 0}

    def check(g, tag, step, tol_s):
        t, nstep, last_dt = g.time()
        assert nstep == step
        hist = g.energy_history()
        zeta, gg = g.get_state()
        allf = np.concatenate([zeta, gg])
        for r in rows["T"]:
            if r[0] == tag and int(r[1]) == step:
                assert abs(t - float(r[2])) <= 1e-12 * float(r[2]) and abs(last_dt - float(r[3])) <= 1e-12 * float(r[3]), (tag, step)
                seen["T"] += 1
        for r in rows["H"]:
            if r[0] == tag and int(r[1]) <= step and (step == 10 or int(r[1]) > 10):
                want = np.array([float(x) for x in r[2:]])
                got = hist[int(r[1]) - 1]
                assert abs(got[0] - want[0]) <= 1e-12 * want[0], (tag, r[1])
                assert np.abs(got[1:] - want[1:]).max() <= TOL_ENERGY * max(1.0, np.abs(want[1:]).max()), (tag, r[1])
                seen["H"] += 1
        for r in rows["S"]:
            if r[0] == tag and int(r[1]) == step:
                f, iz, iy, ix = (int(x) for x in r[2:6])
                want = complex(float(r[6]), float(r[7]))
                # scale: the largest coefficient of the potentials / of ALL moments, as _check_state's joint relative L2 (a high
                # moment the cascade has not reached yet sits at 1e-17, the round-off floor of its neighbours' couplings)
                scale = np.abs(allf[:2]).max() if f < 2 else np.abs(allf[2:]).max()
                assert abs(allf[f, iz, iy, ix] - want) <= tol_s * scale, (tag, step, f, iz, iy, ix)
                seen["S"] += 1

    g = Gandalf(*run["shape"], **prm)                      # run A: as written
    g.set_state(z, gm)
    g.step(0.0, 10)
    check(g, "A", 10, TOL_10STEPS)
    g.close()
    g = Gandalf(*run["shape"], **dict(prm, cfl=0.03))      # run B: the stable C
    g.set_state(z, gm)
    g.step(0.0, 10)
    check(g, "B", 10, TOL_10STEPS)
    g.step(0.0, 90)
    check(g, "B", 100, 1e-9)
    assert seen == {"T": 3, "H": 1 + 1 + 9, "S": 3 * 48}, seen


def test_finding_q28_advective_cfl_is_not_sufficient_with_moments():
    """DESIGN.md Q28: with C = 0.3 on max|grad Phi| alone (Eq. 16) the explicit RK2 of the Hermite couplings
    sqrt(m/2){Psi, g_m+-1} is unstable once enough moments are kept (the oracle blows up with the same digits); C = 0.03
    ~ 0.3/(1+sqrt(2M)) is stable.  64x64x32, M = 16, config 3's forcing and dissipation."""
    from paper_2511_21891_b200.gandalf import Gandalf
    prm, z, gm, run = config3(64, 64, 32, 16)
    g = Gandalf(*run["shape"], **prm)
    g.set_state(z, gm)
    g.step(0.0, 40)
    assert g.energy_history()[-1, 6] > 1e10            # W_g (2.4720e+24 in the oracle and on the GPU)
    g2 = Gandalf(*run["shape"], **dict(prm, cfl=0.03))
    g2.set_state(z, gm)
    g2.step(0.0, 400)
    h = g2.energy_history()
    assert np.isfinite(h).all() and h[-1, 6] < 0.05 and 1.0 < h[-1, 1] < 3.0


@pytest.mark.parametrize("shape,M,extra,dt", [
    ((32, 16, 8), 4, dict(), 2e-3),
    ((16, 32, 16), 9, dict(if_variant=1, g_sign=-1, nu_coll=0.7, p=1.5, eta=0.5, r=2, eta_normalized=1, eta_g=0.3), 2e-3),
    ((32, 32, 8), 3, dict(nspecies=2), 2e-3),
    ((16, 16, 32), 16, dict(nonlinear=0), 0.4),            # a step the plain RK2 of Alg. 1 cannot take (dt kz sqrt(2M) >> 1)
    ((64, 64, 32), 16, dict(nu_coll=1.0, p=2.0, eta=1.0, r=2, eta_normalized=1), 5e-4),   # config 2's shape
])
def test_hermite_exact_propagator_matches_oracle(shape, M, extra, dt):
    """hermite_exact = 1 (Q30; PAPER.md:657, 829 name exponential integrators as future work): the streaming /
    phase-mixing terms of Eq. 6 by exp(s i kz (I - T) dt) per kz -- k_hermite_propagator / k_hermite_apply against the
    oracle's eigen-decomposition route, brackets by the midpoint rule on both sides."""
    prm = dict(M=M, hermite_exact=1, **extra)
    o, g = _pair(shape, prm)
    nsp = extra.get("nspecies", 1)
    z = synth.dense_random(*shape, 2, seed=31, decay=2.0)
    gm = synth.dense_random(*shape, M * nsp, seed=32, decay=2.0)
    o.set_state(z, gm); g.set_state(z, gm)
    o.step(dt, 10); g.step(dt, 10)
    _check_state(o, g, TOL_10STEPS)
    _check_history(o, g)
    if extra.get("nonlinear", 1) == 0 and not extra.get("nu_coll"):
        h = g.energy_history()
        assert abs(h[-1, 6] - h[0, 6]) <= 1e-12 * h[0, 6]      # unitary propagator: W_g conserved at any dt


def test_hermite_exact_rejects_unsupported_closure():
    from paper_2511_21891_b200.gandalf import Gandalf, GandalfError
    with pytest.raises(GandalfError):
        Gandalf(16, 16, 8, M=4, hermite_exact=1, closure=1)
