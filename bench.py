#!/usr/bin/env python
"""bench.py -- throughput of the GANDALF KRMHD hot path (RHS + integrating-factor step) on B200.

Workload: BASELINE.json config 4(a), 256x256x128 with M=32 Hermite moments, fp64, seeded synthetic
initial state, fixed dt.  One "step" = one complete Algorithm-2 step
(two RHS evaluations).  Prints ONE JSON line (see DESIGN.md for every key).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 4a|4b|2|0] [--impl reference]

--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
N > 1 (under torchrun) runs N independent replicas, one per GPU ("replicas only": north_star keeps the
path on one GPU).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

WORKLOADS = {
    "4a": ("config4a", dict(nx=256, ny=256, nz=128, M=32)),
    "4a2": ("config4a", dict(nx=256, ny=256, nz=128, M=32, nspecies=2)),     # both species: 2 + 64 fields
    "4b": ("config4b", dict(nx=512, ny=512, nz=256)),
    "0": ("config0", dict(nx=32, ny=32, nz=16)),          # the small configurations are launch-bound: they time the step's launch path
    "1": ("config1", dict(n=128)),
    "2": ("config2", dict(nx=64, ny=64, nz=32, M=16)),
    # driven turbulence; e.g. --steps 79990 --warmup 10 reaches the statistically steady state (t ~ 17).  cfl = 0.03, not
    # BASELINE's 0.3: with C = 0.3 on max|grad Phi| alone (Eq. 16) the explicit RK2 of the Hermite couplings
    # sqrt(m/2){Psi, g_m+-1} is unstable at M = 32 -- oracle and GPU blow up identically (Q28)
    "3": ("config3", dict(nx=128, ny=128, nz=64, M=32)),
    "0": ("config0", dict(nx=32, ny=32, nz=16)),
}


def make_workload(name, **override):
    from paper_2511_21891_b200 import workloads as cases
    fn, kw = WORKLOADS[name]
    kw = dict(kw)
    kw.update(override)
    if name == "1":
        kw.pop("nz", None)      # Orszag-Tang is z-uniform on two planes: the oracle's sample is the whole workload
    prm, z, g, run = getattr(cases, fn)(**kw)
    if name == "3":
        prm = dict(prm, cfl=0.03)
    return prm, z, g, run


def algorithmic_bytes(shape, M):
    """Algorithmic bytes per launch of each kernel class and per step for the 4-pass design, counting
    retained (dealiased) modes only -- DESIGN.md "Roofline", same formulas as SURVEY.md 8(d)."""
    nx, ny, nz = shape
    F = 2 + M
    Kx, Ky, Kz = nx // 3 + 1, 2 * (ny // 3) + 1, 2 * (nz // 3) + 1
    S_c, S_h, S_xy = 16 * Kx * Ky * Kz, 16 * Kx * Ky * nz, 16 * Kx * ny * nz
    per_launch = {
        "z_inverse": F * (S_c + S_h),
        "y_inverse_P1": F * S_h + 2 * (F + 2) * S_xy,
        "x_pass_P2": 2 * (F + 2) * S_xy + F * S_xy,
        "y_forward_P3": F * S_xy + F * S_h,
        # fused z-forward + update + z-inverse: per step 4F S_h + (3F + 2M) S_c (SURVEY 8(d) "P4"); per launch half of it
        "z_step_P4": 2 * F * S_h + (1.5 * F + M) * S_c,
    }
    p4 = 4 * F * S_h + (3 * F + 2 * M) * S_c
    step_4pass = 2 * (per_launch["y_inverse_P1"] + per_launch["x_pass_P2"] + per_launch["y_forward_P3"]) + p4
    return per_launch, step_4pass


def max_over_ranks(x, world, device="cuda"):
    """Replicas only: the job's time is the slowest replica's.  No data-path collective exists;
    this all-reduce(MAX) of one scalar is the only communication of the bench."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_steps_per_s(ms_max, steps, world):
    """Every rank advances its own replica by `steps` steps in `ms_max` (max over ranks): weak scaling."""
    return world * steps / (ms_max * 1e-3)


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, dev):
        self.dev, self.rows, self.proc = dev, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "50",
                                          "-i", str(self.dev)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


ORACLE_SLAB_NZ = 8          # z-planes of the oracle's timed sample (both the cpu_baseline leg and --impl reference)


def _oracle_slab(name, nz_s, threads=None):
    """One oracle context on a z-slab of the workload (full nx x ny, all moments, nz_s planes)."""
    import oracle
    from oracle import Oracle
    if threads is not None:
        oracle.set_num_threads(threads)
    prm, z, g, run = make_workload(name, nz=nz_s)
    o = Oracle(*run["shape"], **prm)
    o.set_state(z, g)
    return o, prm, run


def run_reference(args, rank, world):
    """The oracle, as it stands, on the host cores: each 'step' is one complete Algorithm-2 step on a bounded sample (a
    z-slab of ORACLE_SLAB_NZ planes, full nx x ny, all moments) of the workload.  ms_per_step is the MEASURED time of one
    sample step; `value` scales the sample's rate by slab/nz to the full grid (sample_scale)."""
    if rank != 0:
        return
    import oracle
    name = args.workload
    fn, kw = WORKLOADS[name]
    full = (kw["nx"], kw["ny"], kw["nz"]) if "nx" in kw else (kw["n"], kw["n"], 2)
    nz_s = min(ORACLE_SLAB_NZ, full[2])
    o, prm, run = _oracle_slab(name, nz_s)
    for _ in range(args.warmup):
        o.step(run["dt"], 1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.step(run["dt"], 1)
    el = time.perf_counter() - t0
    frac = nz_s / full[2]
    sample_steps_per_s = args.steps / el
    steps_per_s = sample_steps_per_s * frac
    M = prm.get("M", 0) * prm.get("nspecies", 1)
    wl = {"4a": "BASELINE config 4(a)", "4b": "BASELINE config 4(b)",
          "4a2": "BASELINE config 4(a) with both slow-mode species (2+64 fields)"}.get(name, f"BASELINE config {name}")
    line = {
        "impl": "reference", "metric": "RHS evals/s", "value": 2 * steps_per_s, "unit": "RHS evals/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 / sample_steps_per_s, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl, "grid": list(full), "M": M, "dt": run["dt"], "fields": 2 + M, "parallelism": "host cores (OpenMP)",
                   "l2": "n/a (CPU)"},
        "sample_scale": frac, "sample_grid": list(run["shape"]),
        "steps_per_s": steps_per_s, "grid_point_moments_per_s": steps_per_s * full[0] * full[1] * full[2] * (2 + M),
        "cpu_baseline": {"value": 2 * steps_per_s, "unit": "RHS evals/s", "cores": oracle.num_threads(), "kind": "oracle",
                         "sample": f"each timed step = one full Algorithm-2 step (2 RHS) on a {run['shape'][0]}x{run['shape'][1]}x{nz_s} "
                                   f"z-slab (all {M} moments): ms_per_step is that measured time; value = sample rate x {nz_s}/{full[2]}"},
        "e2e": {"value": 2 * steps_per_s, "unit": "RHS evals/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)


def cpu_baseline_sample(name, full_shape, full_rhs=False):
    """The oracle timed on the host cores: (i) all cores, one Algorithm-2 step on the ORACLE_SLAB_NZ-plane slab (the same
    sample --impl reference times), (ii) ONE thread on a 2-plane slab, (iii) with --oracle-full-rhs, one RHS evaluation at
    the FULL grid on all cores (tens of seconds and ~20 GB of host memory at 4a)."""
    import oracle
    nthreads = oracle.num_threads()
    nz_s = min(ORACLE_SLAB_NZ, full_shape[2])
    o, prm, run = _oracle_slab(name, nz_s)
    o.step(run["dt"], 1)                  # one untimed step first, as the reference arm does (page faults, thread start-up)
    t0 = time.perf_counter()
    o.step(run["dt"], 1)
    el = time.perf_counter() - t0
    frac = nz_s / full_shape[2]
    out = {"value": 2.0 / el * frac, "unit": "RHS evals/s", "cores": nthreads, "kind": "oracle", "seconds": el,
           "sample": f"one full Algorithm-2 step (2 RHS; after one untimed step) on a {run['shape'][0]}x{run['shape'][1]}x{nz_s} z-slab of the "
                     f"workload, all moments; rate scaled by {nz_s}/{full_shape[2]} to the full grid"}
    del o
    nz_1 = min(2, full_shape[2])
    o1, _, run1 = _oracle_slab(name, nz_1, threads=1)
    t0 = time.perf_counter()
    o1.rhs()
    el1 = time.perf_counter() - t0
    out["single_thread"] = {"value": 1.0 / el1 * nz_1 / full_shape[2], "unit": "RHS evals/s", "cores": 1, "seconds": el1,
                            "sample": f"one RHS evaluation on a {run1['shape'][0]}x{run1['shape'][1]}x{nz_1} z-slab, one thread; "
                                      f"rate scaled by {nz_1}/{full_shape[2]}"}
    del o1
    oracle.set_num_threads(nthreads)
    if full_rhs:
        # the slab flatters the oracle (its z transforms shrink with the slab): where the host has the memory, ONE RHS evaluation at
        # the full grid is the reported value and the slab figure moves to `slab_sample`
        of, _, runf = _oracle_slab(name, full_shape[2])
        t0 = time.perf_counter()
        of.rhs()
        elf = time.perf_counter() - t0
        del of
        out["slab_sample"] = {k: out[k] for k in ("value", "seconds", "sample")}
        out.update({"value": 1.0 / elf, "seconds": elf,
                    "sample": f"ONE RHS evaluation at the full {full_shape[0]}x{full_shape[1]}x{full_shape[2]} grid, all moments, no scaling "
                              f"(the slab figure, which --impl reference also uses, is in slab_sample)"})
    return out


def host_can_hold_full_oracle(shape, F):
    """The oracle keeps full complex spectra: about 12 arrays of nx*ny*nz complex per field at the RHS (measured ~20 GB at 4a)."""
    try:
        avail = os.sysconf("SC_AVPHYS_PAGES") * os.sysconf("SC_PAGE_SIZE")
    except (ValueError, OSError):
        return False
    return avail > 2.0 * 12 * F * shape[0] * shape[1] * shape[2] * 16


def cufft_comparison(sim, stream, shape, prm, reps=3):
    """Timed comparison ONLY (north_star: "cuFFT may appear only as a timed comparison"; BASELINE config 4): the same RHS
    evaluation written the way the paper describes its own code -- vendor FFT (torch.fft = cuFFT
    3-D D2Z/Z2D on the full grid, boolean-mask dealiasing) plus un-fused elementwise tensor ops -- with the SAME transform
    count as the product path (derivatives of xi+-, w+- once; two inverse transforms and one forward transform per moment).
    It is not on the product path and not the oracle; its result is compared with gandalf_rhs for the record."""
    import torch
    nx, ny, nz = shape
    M = prm.get("M", 0)
    dev = torch.device("cuda", sim.params.device)
    two_pi = 2.0 * np.pi
    Lx, Ly, Lz = (prm.get(k, two_pi) for k in ("Lx", "Ly", "Lz"))
    nxs = torch.arange(nx // 2 + 1, device=dev, dtype=torch.float64)
    nys = torch.fft.fftfreq(ny, 1.0 / ny, device=dev, dtype=torch.float64)
    nzs = torch.fft.fftfreq(nz, 1.0 / nz, device=dev, dtype=torch.float64)
    kx = (two_pi / Lx * nxs)[None, None, :]
    ky = (two_pi / Ly * nys)[None, :, None]
    kz = (two_pi / Lz * nzs)[:, None, None]
    mask = ((3 * nxs.abs() <= nx)[None, None, :] & (3 * nys.abs() <= ny)[None, :, None] & (3 * nzs.abs() <= nz)[:, None, None])
    k2 = kx * kx + ky * ky
    ik2 = torch.where(k2 > 0, 1.0 / k2, torch.zeros_like(k2))
    dn = [np.sqrt(m / 2.0) for m in range(M)]
    up = [np.sqrt((m + 1) / 2.0) for m in range(M)]
    if M:
        if prm.get("closure", 0) == 1 and M >= 2:
            dn[M - 1] += up[M - 1]
        up[M - 1] = 0.0
    sgn = float(prm.get("g_sign", 1))
    sz = (nz, ny, nx)

    def grad(fh):
        return (torch.fft.irfftn(1j * kx * fh, s=sz, norm="forward"), torch.fft.irfftn(1j * ky * fh, s=sz, norm="forward"))

    def fwd(f):
        return torch.fft.rfftn(f, s=sz, norm="forward") * mask

    def rhs(zeta, g):
        w = -k2 * zeta                                             # vorticities
        xpx, xpy = grad(zeta[0]); xmx, xmy = grad(zeta[1])
        wpx, wpy = grad(w[0]); wmx, wmy = grad(w[1])
        A = fwd(xpx * wmy - xpy * wmx + xmx * wpy - xmy * wpx)
        B = fwd(xpx * xmy - xpy * xmx)
        dw = torch.stack((-0.5 * A - 0.5 * k2 * B, -0.5 * A + 0.5 * k2 * B))
        del wpx, wpy, wmx, wmy, A, B
        phx, phy, psx, psy = 0.5 * (xpx + xmx), 0.5 * (xpy + xmy), 0.5 * (xpx - xmx), 0.5 * (xpy - xmy)
        dg = torch.empty_like(g)
        Qp = None; Ra = None
        for m in range(M):
            gx, gy = grad(g[m])
            P = phx * gy - phy * gx
            Q = psx * gy - psy * gx
            if m >= 1:
                dg[m - 1] = fwd(Ra + up[m - 1] * Q)
            Ra = (dn[m] * Qp - P) if m >= 1 else -P
            Qp = Q
        if M:
            dg[M - 1] = fwd(Ra)
            zero = torch.zeros_like(g[0])
            for m in range(M):
                lin = g[m] - dn[m] * (g[m - 1] if m >= 1 else zero) - up[m] * (g[m + 1] if m + 1 < M else zero)
                dg[m] = dg[m] + sgn * 1j * kz * lin
        return dw, dg

    with torch.cuda.stream(stream):                                # the context's stream: device-pointer calls are stream-ordered
        zeta, g = sim.get_state(device=True)
        dw_o, dg_o = sim.rhs(device=True)
    torch.cuda.synchronize()
    dw_c, dg_c = rhs(zeta, g)                                      # also warms cuFFT's plans
    err_w = float((dw_c - dw_o).norm() / dw_o.norm())
    err_g = float((dg_c - dg_o).norm() / dg_o.norm()) if M else 0.0
    del dw_c, dg_c, dw_o, dg_o
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        rhs(zeta, g)
    e1.record()
    torch.cuda.synchronize()
    ms_c = e0.elapsed_time(e1) / reps
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(stream):
        f0.record(stream)
        for _ in range(reps):
            sim.rhs(device=True)
        f1.record(stream)
    torch.cuda.synchronize()
    ms_o = f0.elapsed_time(f1) / reps
    return {"what": "one RHS evaluation: torch.fft (cuFFT) 3-D transforms on the full grid + un-fused elementwise ops, same transform count",
            "cufft_path_ms_per_rhs": ms_c, "cufft_path_rhs_per_s": 1e3 / ms_c,
            "gandalf_rhs_call_ms": ms_o, "note": "gandalf_rhs_call_ms includes exporting the RHS to the boundary layout",
            "rel_l2_vs_gandalf_rhs": {"dw": err_w, "dg": err_g}, "reps": reps}


def run_microbench(device=0, which=(0, 1, 2, 3)):
    """Measured ceilings of the units the hot path leans on (include/gandalf.h: gandalf_microbench)."""
    from paper_2511_21891_b200 import gandalf
    out = {}
    for w in which:
        v = gandalf.microbench(w, device)
        name = gandalf.MICROBENCHES[w]
        if w == 0:
            out[name] = {"tflops": v[0], "t_instr_per_s": v[1], "ms": v[2], "sms": int(v[3])}
        elif w == 1:
            out[name] = {"g_transforms_per_s_16x16_8warps_register_twiddles": v[0], "g_transforms_per_s_16x16_8warps_table_twiddles": v[1],
                         "g_transforms_per_s_8x8x4_16warps": v[2], "ms": v[3]}
        else:
            out[name] = {"bytes_per_clk_per_sm": v[0], "tb_per_s_chip": v[1], "ms": v[2], "cycles_per_cta": v[3]}
    return out


L2_BYTES = 126e6          # B200 L2 (B200_PROFILING.md)
CAPTURE_SOURCES = ("pass_x.cu", "passes_zy.cu", "fft.cuh", "common.cuh")      # what the kernels of the committed ncu captures are built from


def kernel_sources_sha256():
    """sha256 over the kernel sources the committed ncu figures (profiles/r0N_traffic.csv, _fp64_instr.csv) were captured from."""
    import hashlib
    h = hashlib.sha256()
    for fn_ in CAPTURE_SOURCES:
        h.update(open(os.path.join(ROOT, "paper_2511_21891_b200", "csrc", fn_), "rb").read())
    return h.hexdigest()


def captures_stale(tag="r02"):
    """True when the kernel sources differ from the ones hashed in profiles/<tag>_capture_sources.md at capture time (the
    committed traffic / instruction counts then describe another build); None when no hash was recorded."""
    try:
        txt = open(os.path.join(ROOT, "profiles", f"{tag}_capture_sources.md")).read()
    except OSError:
        return None
    import re
    m = re.search(r"sha256[^0-9a-f]*([0-9a-f]{64})", txt)
    return None if not m else m.group(1) != kernel_sources_sha256()


def classify_bound(dom_bytes, hbm_floor_ms, alu_floor_ms):
    """Which roof bounds the dominant kernel, and the L2 note of the timing rules, from the workload itself:
    a launch whose algorithmic bytes fit the L2 is not an HBM measurement at all (the small grids are launch / latency
    bound); otherwise the larger of the HBM floor and the fp64-instruction floor (when one is known)."""
    if dom_bytes <= L2_BYTES:
        return ("launch/latency",
                "NOT flushed: the dominant kernel moves %.1f MB per launch, which fits the 126 MB L2 -- this grid is launch / latency bound "
                "(DESIGN.md 5b) and the HBM fraction below says nothing about the kernels" % (dom_bytes / 1e6))
    l2 = "no flush needed: the dominant kernel streams %.2f GB per launch, far more than the 126 MB L2" % (dom_bytes / 1e9)
    if alu_floor_ms is not None and alu_floor_ms > hbm_floor_ms:
        return "alu", l2
    return "hbm", l2


def quick_time(workload, local, warmup=10, steps=50):
    """ms per step and roofline fractions of another workload, timed like the headline (CUDA events on the context's stream, then a
    per-kernel pass): used to put BASELINE config 4(b) into the default line (extra.config4b)."""
    import torch
    from paper_2511_21891_b200.gandalf import Gandalf, KERNEL_CLASSES
    prm, z, g, run = make_workload(workload)
    shape, dt, M = run["shape"], run["dt"], prm.get("M", 0) * prm.get("nspecies", 1)
    stream = torch.cuda.Stream()
    sim = Gandalf(*shape, device=local, stream=stream.cuda_stream, **prm)
    zd = torch.from_numpy(z).cuda()
    gd = torch.from_numpy(g).cuda() if M else None
    sampler = ClockSampler(local)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(stream):
        sim.set_state(zd, gd)
        sim.step(dt, warmup)
    torch.cuda.synchronize()
    sampler.start()
    with torch.cuda.stream(stream):
        e0.record(stream)
        sim.step(dt, steps)
        e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    sim.kernel_timing(True)
    with torch.cuda.stream(stream):
        sim.step(dt, 10)
    torch.cuda.synchronize()
    kt = sim.kernel_times()
    sim.kernel_timing(False)
    clocks = sampler.stop()
    assert np.isfinite(sim.energy_history()).all()
    sim.close()
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    peak = peaks.get("hbm_gbs", 6650.0)
    per_launch, step_bytes = algorithmic_bytes(shape, M)
    kern = {k: {"avg_ms": kt[k][0], "frac_of_hbm_peak": per_launch[k] / 1e9 / (kt[k][0] * 1e-3) / peak}
            for k in KERNEL_CLASSES if kt[k][1] and k != "z_inverse"}
    dom = max(kern, key=lambda k: kern[k]["avg_ms"])
    return {"workload": f"BASELINE config {workload}", "grid": list(shape), "M": M, "steps": steps, "warmup": warmup, "ms_per_step": ms,
            "value": 2e3 / ms, "unit": "RHS evals/s", "step_algorithmic_gb": step_bytes / 1e9,
            "step_frac_of_measured_hbm_peak": step_bytes / 1e9 / (ms * 1e-3) / peak, "dominant_kernel": dom,
            "dominant_kernel_frac": kern[dom]["frac_of_hbm_peak"], "kernels": kern, "clocks": clocks}


def run_mshard(args, rank, world, local):
    """ONE run of the workload sharded by Hermite moment over the ranks (strong scaling): xi+- replicated, one halo moment per
    neighbour exchanged twice per step with NCCL point-to-point copies in place on the library's buffers (sharded.py)."""
    import torch
    import torch.distributed as dist
    from paper_2511_21891_b200 import sharded
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    prm, z, g, run = make_workload(args.workload)
    shape, dt, M = run["shape"], run["dt"], prm.get("M", 0)
    emu = args.emulate_ranks if world == 1 else 0
    nranks = emu if emu else world
    if M < nranks or prm.get("nspecies", 1) != 1:
        raise SystemExit("mshard needs one species and at least one moment per rank")
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    stream = torch.cuda.current_stream()        # NCCL orders its copies against torch's current stream: the contexts run on it
    lays = [sharded.ShardLayout.make(M, nranks, r) for r in range(nranks)]
    mine = lays if emu else [lays[rank]]
    shards = [sharded.GandalfShard(*shape, lay, device=local, stream=stream.cuda_stream, **prm) for lay in mine]
    for sh in shards:
        sh.set_state(z, g)
    if emu or world == 1:
        def advance(n):
            sharded.step_all(shards, mine, dt, n)
    else:
        stepper = sharded.ShardedStepper(shards[0], mine[0], sharded.DistExchange())
        advance = lambda n: stepper.step(dt, n)                   # noqa: E731
    advance(args.warmup)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    sampler.start()
    n0 = sum(sh.g.launch_count() for sh in shards)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    advance(args.steps)
    e1.record()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    ms = max_over_ranks(e0.elapsed_time(e1), world)
    clocks = sampler.stop()
    launches = sum(sh.g.launch_count() for sh in shards) - n0
    if world > 1:
        en = np.array([stepper.energy()])                          # W_g summed over the ranks by DistExchange (a CUDA tensor under NCCL)
        wg = float(en[0, 5])
    else:
        en = np.array([sh.energy() for sh in shards])
        wg = float(en[:, 5].sum())
    if rank == 0:
        steps_per_s = args.steps / (ms * 1e-3)                     # ONE run: the ranks share the work (strong scaling)
        halo_bytes = 16 * (shape[0] // 3 + 1) * (2 * (shape[1] // 3) + 1) * (2 * (shape[2] // 3) + 1)
        print(json.dumps({
            "metric": "RHS evals/s", "value": 2 * steps_per_s, "unit": "RHS evals/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"BASELINE config {args.workload}", "grid": list(shape), "M": M,
                       "parallelism": f"m-shard, {nranks} ranks" + (" EMULATED in one process on one GPU (path check, not a scaling number)" if emu else ""),
                       "moments_per_rank": [lay.hi - lay.lo for lay in lays], "halo_fields_per_rank": [lay.halo_lo + lay.halo_hi for lay in lays],
                       "halo_bytes_per_neighbour_per_exchange": halo_bytes, "exchanges_per_step": 2},
            "steps_per_s": steps_per_s, "grid_point_moments_per_s": shape[0] * shape[1] * shape[2] * (2 + M) * steps_per_s,
            "gpu_launches": int(launches), "clocks": clocks,
            "final_energy": {"E_A": float(en[0, 0]), "W_g": wg},
        }), flush=True)
    for sh in shards:
        sh.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--workload", default="4a", choices=sorted(WORKLOADS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-cufft-compare", action="store_true")
    ap.add_argument("--no-graph", action="store_true", help="plain stream launches instead of the replayed CUDA graph of one step")
    ap.add_argument("--oracle-full-rhs", action="store_true", help="also time one oracle RHS evaluation at the FULL grid (slow, ~20 GB host memory at 4a)")
    ap.add_argument("--no-oracle-full-rhs", action="store_true", help="cpu_baseline from the z-slab sample only (skips the ~30 s full-grid oracle RHS of the default 4a run)")
    ap.add_argument("--sustained-seconds", type=float, default=3.0, help="after the timed region, run about this many seconds of steps and report them as `sustained` (0 = off)")
    ap.add_argument("--no-4b", action="store_true", help="do not time BASELINE config 4(b) after the default 4a run")
    ap.add_argument("--microbench", action="store_true", help="print the measured unit ceilings (gandalf_microbench) and exit")
    ap.add_argument("--parallelism", default="replicas", choices=["replicas", "mshard"],
                    help="N > 1: independent replicas (default; north_star keeps the product on one GPU) or ONE run sharded by Hermite "
                         "moment with halo exchange over NCCL (paper_2511_21891_b200/sharded.py, DESIGN.md Q31)")
    ap.add_argument("--emulate-ranks", type=int, default=0, help="mshard on ONE GPU: emulate this many ranks in one process (checks the path; not a scaling number)")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    if args.microbench:
        if rank == 0:
            print(json.dumps(run_microbench(local)), flush=True)
        return
    if args.warmup < 3:
        args.warmup = 3
    if args.parallelism == "mshard":
        run_mshard(args, rank, world, local)
        return

    import torch
    import torch.distributed as dist
    from paper_2511_21891_b200.gandalf import Gandalf, KERNEL_CLASSES
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    prm, z, g, run = make_workload(args.workload)
    shape, dt, M = run["shape"], run["dt"], prm.get("M", 0) * prm.get("nspecies", 1)      # M = moment fields
    F = 2 + M
    stream = torch.cuda.Stream()
    sim = Gandalf(*shape, device=local, stream=stream.cuda_stream, **prm)
    if args.no_graph:
        sim.graph_mode(False)
    # device-resident inputs for the device-timed number
    zd = torch.from_numpy(z).cuda()
    gd = torch.from_numpy(g).cuda() if M else None
    with torch.cuda.stream(stream):
        sim.set_state(zd, gd)
        sim.step(dt, args.warmup)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    sampler.start()
    n0 = sim.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(stream):
        e0.record(stream)
        sim.step(dt, args.steps)
        e1.record(stream)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    launches = sim.launch_count() - n0
    graph_replays = sim.graph_mode()    # steps of the timed region replayed from the captured CUDA graph of one step (gandalf_graph_mode)
    ms = max_over_ranks(ms, world)
    # per-kernel CUDA-event times in a SECOND, untimed-for-the-headline pass (the events cost a little per launch)
    ksteps = min(args.steps, 10)
    sim.kernel_timing(True)
    k0, k1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(stream):
        k0.record(stream)
        sim.step(dt, ksteps)
        k1.record(stream)
    torch.cuda.synchronize()
    kms = k0.elapsed_time(k1)
    ktimes = sim.kernel_times()
    sim.kernel_timing(False)
    clocks = sampler.stop()             # sampled over the timed region and the per-kernel pass that follows it (same load)
    # a time stepper runs for minutes: the same steps over a few SECONDS, where the power cap has settled the clock
    sustained, nsus = None, 0
    if args.sustained_seconds > 0:
        nsus = max(args.steps, int(args.sustained_seconds / max(ms / args.steps * 1e-3, 1e-6)))
        nsus = min(nsus, 20000)
        s2 = ClockSampler(local)
        s2.start()
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(stream):
            s0.record(stream)
            sim.step(dt, nsus)
            s1.record(stream)
        torch.cuda.synchronize()
        sms = max_over_ranks(s0.elapsed_time(s1), world)
        sustained = {"steps": nsus, "seconds": sms * 1e-3, "ms_per_step": sms / nsus, "value": 2 * whole_job_steps_per_s(sms, nsus, world),
                     "unit": "RHS evals/s", "clocks": s2.stop()}
    hist = sim.energy_history()
    assert hist.shape[0] == args.warmup + args.steps + ksteps + nsus and np.isfinite(hist).all()
    spectrum = None
    if args.workload == "3":      # BASELINE config 3 "reports the k_perp energy spectrum" (Eq. 26; unpinned statistics)
        sp = sim.kperp_spectrum(44)
        ks = np.arange(44)
        sel = (ks >= 2) & (ks <= 12) & (sp > 0)
        slope = float(np.polyfit(np.log(ks[sel]), np.log(sp[sel]), 1)[0]) if sel.sum() >= 3 else None
        spectrum = {"E_kperp": [float(x) for x in sp], "fit_range": [2, 12], "slope": slope, "paper_slope": -5.0 / 3.0,
                    "t_end": float(hist[-1, 0]), "mean_dt": float(hist[-1, 0] / hist.shape[0])}
    steps_per_s = whole_job_steps_per_s(ms, args.steps, world)

    # ---- end to end through the C ABI with HOST (pinned) buffers: H2D state, one step, D2H energies
    e2e = None
    if args.e2e_steps > 0:
        zp = torch.empty(z.shape, dtype=torch.complex128, pin_memory=True)
        zp.copy_(torch.from_numpy(z))
        zh = zp.numpy()
        gh = None
        if M:
            gp = torch.empty(g.shape, dtype=torch.complex128, pin_memory=True)
            gp.copy_(torch.from_numpy(g))
            gh = gp.numpy()
        sim.set_state(zh, gh); sim.step(dt, 1); sim.energy()      # warm the host path
        torch.cuda.synchronize()
        b0 = sim.transfer_bytes()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            sim.set_state(zh, gh)           # host -> device copy of the step's input state inside the call
            sim.step(dt, 1)
            en = sim.energy_history()       # device -> host read of the step's result (energy record)
        torch.cuda.synchronize()
        el = time.perf_counter() - t0
        el = max_over_ranks(el, world)
        b1 = sim.transfer_bytes()           # counted by the library at the copies it issues (gandalf_transfer_bytes)
        energy_only = {"value": 2 * world * args.e2e_steps / el, "unit": "RHS evals/s",
                       "h2d_bytes_per_step": int((b1[0] - b0[0]) // args.e2e_steps), "d2h_bytes_per_step": int((b1[1] - b0[1]) // args.e2e_steps),
                       "what": "gandalf_set_state(host pinned) + gandalf_step(dt,1) + gandalf_energy_history(host): only the energy record comes back"}
        # the result of a step is the new STATE: read it back too, in the library's checkpoint format (gandalf_get_state_raw: the
        # retained modes of every field, the mirror of what set_state moves in), into pinned host memory
        rawp = torch.empty(sim.state_raw_doubles(), dtype=torch.float64, pin_memory=True)
        rawh = rawp.numpy()

        def read_state():
            sim.get_state_raw(out=rawh)
        read_state()
        torch.cuda.synchronize()
        b0 = sim.transfer_bytes()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            sim.set_state(zh, gh)
            sim.step(dt, 1)
            read_state()                    # device -> host: the new state (synchronises)
            en = sim.energy_history()       # and its energy record
        torch.cuda.synchronize()
        el = max_over_ranks(time.perf_counter() - t0, world)
        b1 = sim.transfer_bytes()
        assert np.isfinite(rawh).all() and np.abs(rawh).max() > 0
        e2e = {"value": 2 * world * args.e2e_steps / el, "unit": "RHS evals/s", "steps": args.e2e_steps,
               "h2d_bytes_per_step": int((b1[0] - b0[0]) // args.e2e_steps), "d2h_bytes_per_step": int((b1[1] - b0[1]) // args.e2e_steps),
               "host_array_bytes": int(z.nbytes + (g.nbytes if M else 0)),
               "what": "gandalf_set_state(host pinned) + gandalf_step(dt,1) + gandalf_get_state_raw(host pinned) + gandalf_energy_history(host) "
                       "per step: the state goes in and the new state comes back; both directions move only the modes Eq. 20 retains",
               "energy_only": energy_only}

    # ---- roofline of the dominant kernel (largest share of device time in the timed region)
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    peak_gbs, peak_src = (peaks["hbm_gbs"], "measured (MEASURED_PEAKS.json)") if "hbm_gbs" in peaks else (6650.0, "fallback")
    per_launch, step_bytes = algorithmic_bytes(shape, M)
    # the stand-alone z-inverse runs inside a step only after a forcing increment, on the forced fields alone (w+-: 2, g_0: 1)
    nzi = (2 if prm.get("force_eps", 0.0) > 0 else 0) + (1 if prm.get("force_g_amp", 0.0) > 0 else 0)
    if nzi:
        per_launch["z_inverse"] = per_launch["z_inverse"] / F * (nzi / ((prm.get("force_eps", 0.0) > 0) + (prm.get("force_g_amp", 0.0) > 0)))
    kern = {}
    for name in KERNEL_CLASSES:
        avg_ms, n = ktimes[name]
        if n:
            kern[name] = {"avg_ms": avg_ms, "launches": n, "share_of_step": avg_ms * n / kms,
                          "algorithmic_gb": per_launch[name] / 1e9, "achieved_gbs": per_launch[name] / 1e9 / (avg_ms * 1e-3),
                          "frac_of_hbm_peak": per_launch[name] / 1e9 / (avg_ms * 1e-3) / peak_gbs}
    dom = max(kern, key=lambda k: kern[k]["avg_ms"] * kern[k]["launches"])
    traffic, traffic_src = None, None   # dram bytes per launch of the dominant kernel from the committed ncu capture (profiles/)
    for fn_ in ("r02_traffic.csv",):
        try:
            for ln in open(os.path.join(ROOT, "profiles", fn_)).read().splitlines()[1:]:
                w, k, b = ln.split(",")
                if w == args.workload and k == dom:
                    traffic, traffic_src = float(b), f"profiles/{fn_} (ncu --set full dram__bytes_read+write per launch, committed; not measured in this run)"
        except Exception:
            pass
        if traffic is not None:
            break
    stale = captures_stale("r02")
    # fp64 side of the dominant kernel: 5 N log2 N flops per complex transform against the DFMA rate
    # measured on this device right now (gandalf_microbench 0)
    alu = None
    try:
        from paper_2511_21891_b200 import gandalf as _g
        mb = _g.microbench(0, local)
        nx_, ny_, nz_ = shape
        nfft = {"x_pass_P2": (4 + M + (2 + M + 1) // 2) * ny_ * nz_ * 5.0 * nx_ * np.log2(nx_),
                "y_inverse_P1": 2 * (F + 2) * nz_ * (nx_ // 3 + 1) * 5.0 * ny_ * np.log2(ny_),
                "y_forward_P3": F * nz_ * (nx_ // 3 + 1) * 5.0 * ny_ * np.log2(ny_),
                "z_step_P4": 2 * F * (nx_ // 3 + 1) * (2 * (ny_ // 3) + 1) * 5.0 * nz_ * np.log2(nz_)}
        alu = {"measured_fp64_fma_tflops": mb[0], "measured_fp64_t_instr_per_s": mb[1], "how": "gandalf_microbench(0): dependency-free DFMA chains, all SMs, best of 5",
               "kernels": {k: {"transform_gflop_per_launch": nfft[k] / 1e9, "achieved_tflops": nfft[k] / 1e12 / (kern[k]["avg_ms"] * 1e-3),
                               "frac_of_measured_fp64_peak": nfft[k] / 1e12 / (kern[k]["avg_ms"] * 1e-3) / mb[0]} for k in nfft if k in kern}}
        # instruction side: executed fp64 warp instructions per launch from the committed ncu capture (profiles/), against
        # the issue rate measured above -- the roofline that actually bounds the x-pass's transforms
        try:
            for ln in open(os.path.join(ROOT, "profiles", "r02_fp64_instr.csv")).read().splitlines()[1:]:
                w, k, n_ = ln.split(",")
                if w == args.workload and k == dom and k in kern:
                    rate = float(n_) * 32 / (kern[k]["avg_ms"] * 1e-3)
                    alu["instr"] = {"kernel": k, "fp64_warp_instructions_per_launch": float(n_), "achieved_t_instr_per_s": rate / 1e12,
                                    "frac_of_measured_issue_rate": rate / 1e12 / mb[1],
                                    "source": "profiles/r02_fp64_instr.csv (ncu source page, committed; not counted in this run)"}
        except Exception:
            pass
    except Exception as exc:
        alu = {"error": repr(exc)[:200]}
    step_ms = ms / args.steps
    bound_note = None
    hbm_floor = per_launch[dom] / 1e9 / peak_gbs * 1e3
    alu_floor = None
    if isinstance(alu, dict) and "instr" in alu:
        alu_floor = alu["instr"]["fp64_warp_instructions_per_launch"] * 32 / (alu["measured_fp64_t_instr_per_s"] * 1e12) * 1e3
    bound, l2_note = classify_bound(per_launch[dom], hbm_floor, alu_floor)
    hbm_side = {"achieved": kern[dom]["achieved_gbs"], "peak": peak_gbs, "unit": "GB/s", "frac": kern[dom]["achieved_gbs"] / peak_gbs,
                "floor_ms": hbm_floor}
    head = dict(hbm_side)
    if bound == "alu":       # the larger floor is the roof the kernel can actually reach: report against it, keep the HBM side beside it
        ins = alu["instr"]
        head = {"achieved": ins["achieved_t_instr_per_s"], "peak": alu["measured_fp64_t_instr_per_s"], "unit": "T fp64 thread-instr/s",
                "frac": ins["frac_of_measured_issue_rate"], "floor_ms": alu_floor}
        peak_src = "measured in this run (gandalf_microbench 0: fp64 issue rate of all SMs); the HBM side uses " + peak_src
        bound_note = ("%s sits on the ridge: HBM floor %.2f ms (algorithmic bytes at the measured copy bandwidth), fp64-instruction floor %.2f ms "
                      "(executed fp64 instructions at the measured issue rate), measured %.2f ms; the larger floor is the bound reported, the HBM "
                      "side is in roofline.hbm (the step as a whole is HBM-bound: roofline.step)" % (dom, hbm_floor, alu_floor, kern[dom]["avg_ms"]))
    elif bound == "launch/latency":
        bound_note = "the dominant kernel's bytes per launch fit the L2: neither roof applies, the step is a chain of short launches (cuda graph replay)"
    elif alu_floor is not None:
        bound_note = ("%s: HBM floor %.2f ms, fp64-instruction floor %.2f ms, measured %.2f ms" % (dom, hbm_floor, alu_floor, kern[dom]["avg_ms"]))
    roofline = {"bound": bound, "bound_note": bound_note, "kernel": dom, "achieved": head["achieved"], "peak": head["peak"], "peak_source": peak_src,
                "unit": head["unit"], "frac": head["frac"], "floor_ms": head["floor_ms"], "measured_ms": kern[dom]["avg_ms"], "hbm": hbm_side,
                "traffic": traffic, "traffic_source": traffic_src,
                "traffic_stale": stale, "traffic_stale_how": "sha256 of csrc/{%s} against profiles/r02_capture_sources.md" % ", ".join(CAPTURE_SOURCES),
                "algorithmic_bytes_per_launch": per_launch[dom],
                "note": "per-kernel times come from a second pass of %d steps with CUDA events around every launch (%.3f ms/step); the headline "
                        "ms_per_step is timed without them" % (ksteps, kms / ksteps),
                "step": {"algorithmic_gb_4pass_design": step_bytes / 1e9, "achieved_gbs": step_bytes / 1e9 / (step_ms * 1e-3),
                         "frac_of_measured_peak": step_bytes / 1e9 / (step_ms * 1e-3) / peak_gbs,
                         "frac_of_8TBs_nominal": step_bytes / 1e9 / (step_ms * 1e-3) / 8000.0},
                "alu": alu, "kernels": kern}

    cufft = None
    if rank == 0 and world == 1 and not args.no_cufft_compare and prm.get("nspecies", 1) == 1:
        try:
            cufft = cufft_comparison(sim, stream, shape, prm)
        except Exception as exc:                      # the comparison must never take the bench line down
            cufft = {"error": repr(exc)[:200]}
    if rank == 0:
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            full = args.oracle_full_rhs or (args.workload == "4a" and not args.no_oracle_full_rhs and host_can_hold_full_oracle(shape, F))
            cpu = cpu_baseline_sample(args.workload, shape, full_rhs=full)
        wl = {"4a": "BASELINE config 4(a)", "4b": "BASELINE config 4(b)",
              "4a2": "BASELINE config 4(a) with both slow-mode species (2+64 fields)"}.get(args.workload, f"BASELINE config {args.workload}")
        line = {
            "metric": "RHS evals/s", "value": 2 * steps_per_s, "unit": "RHS evals/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl, "grid": list(shape), "M": M, "dt": dt, "fields": F, "parallelism": "replicas only" if world > 1 else "1 GPU",
                       "l2": l2_note},
            "steps_per_s": steps_per_s, "grid_point_moments_per_s": steps_per_s * shape[0] * shape[1] * shape[2] * F,
            "clocks": clocks, "sustained": sustained, "e2e": e2e, "gpu_launches": launches,
            "launch_path": ("cuda graph of one step, replayed" if graph_replays else "plain stream launches"), "graph_replays": graph_replays, "roofline": roofline, "cpu_baseline": cpu, "cufft_comparison": cufft, "kperp_spectrum": spectrum,
            "final_energy": {"E_A": float(hist[-1, 1]), "W_g": float(hist[-1, 6])},
        }
        if args.workload == "4a" and world == 1 and not args.no_4b:
            # BASELINE config 4 names two sizes: the second one is timed in the same run (the 4a context is released first)
            sim.close()
            del zd, gd
            torch.cuda.empty_cache()
            try:
                line["extra"] = {"config4b": quick_time("4b", local)}
            except Exception as exc:                  # never take the headline down
                line["extra"] = {"config4b": {"error": repr(exc)[:200]}}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
