"""Workload definitions shared by the parity tests, smoke() and bench.py (no CUDA, no oracle import): the BASELINE.json configs
as (parameter dict, seeded inputs).  The dicts use the parameter names common to gandalf_params and
the oracle; nothing here computes any of the method's arithmetic."""
import numpy as np

from . import synth


def config0(nx=32, ny=32, nz=16, seed=1000):
    prm = dict(M=0, eta=1e-3, r=2, eta_normalized=0)
    return prm, synth.random_zeta(nx, ny, nz, seed), None, dict(dt=1e-3, steps=100, shape=(nx, ny, nz))


def config1(n=128):
    prm = dict(M=0)
    return prm, synth.orszag_tang(n, n, 2), None, dict(dt=1e-3, steps=2000, shape=(n, n, 2))


def config2(nx=64, ny=64, nz=32, M=16, seed=2000):
    prm = dict(M=M, nu_coll=1.0, p=2.0, eta=1.0, r=2, eta_normalized=1, eta_g=1.0)
    z = synth.random_zeta(nx, ny, nz, seed)
    g = synth.random_g(nx, ny, nz, M, seed + 1, total=0.01)
    return prm, z, g, dict(dt=5e-4, steps=200, shape=(nx, ny, nz))


def config3(nx=128, ny=128, nz=64, M=32, seed=3000, eta=3e3):
    prm = dict(M=M, nu_coll=1.0, p=2.0, eta=eta, r=4, eta_normalized=1, eta_z=eta, r_z=4, eta_g=eta,
               force_eps=1.0, force_nperp_min=1, force_nperp_max=2, force_nz_max=1, seed=seed + 2, cfl=0.3)
    z = synth.random_zeta(nx, ny, nz, seed)
    g = synth.random_g(nx, ny, nz, M, seed + 1, total=0.01)
    return prm, z, g, dict(dt=0.0, steps=2000, shape=(nx, ny, nz))


def config4a(nx=256, ny=256, nz=128, M=32, seed=4000, nspecies=1):
    prm, _, _, _ = config2(8, 8, 2, M)
    z = synth.random_zeta(nx, ny, nz, seed)
    g = synth.random_g(nx, ny, nz, M, seed + 1, total=0.01)
    if nspecies == 2:       # both slow-mode species (PAPER.md:357 layout): g^+ then g^-, 2M fields
        prm = dict(prm, nspecies=2)
        g = np.concatenate([g, synth.random_g(nx, ny, nz, M, seed + 2, total=0.01)])
    return prm, z, g, dict(dt=5e-4, steps=50, shape=(nx, ny, nz))


def config4b(nx=512, ny=512, nz=256, seed=4100):
    prm, _, _, _ = config0(8, 8, 2)
    return prm, synth.random_zeta(nx, ny, nz, seed), None, dict(dt=1e-3, steps=50, shape=(nx, ny, nz))


def rel_l2(a, b):
    a = np.asarray(a); b = np.asarray(b)
    den = np.linalg.norm(b.ravel())
    return float(np.linalg.norm((a - b).ravel()) / den) if den > 0 else float(np.linalg.norm(a.ravel()))
