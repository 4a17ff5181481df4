"""Oracle pins, round 3 (-m "not gpu"): the five one-line mistakes that still passed every pin after round 2.

P23  shell index of Eq. 26 (Q15): bin = floor(kperp/dk + 1/2), dk = 2 pi / max(Lx, Ly) -- single
     modes whose rounded and truncated bins differ, and an anisotropic box where max and min give different bins
P24  which of E+ / E- is which in the energy record (Q14): a pure xi+ (pure xi-) mode, closed form,
     for the instantaneous energies and for the per-step history record
P25  order of dissipation and forcing inside a step (Alg. 2 l.12-14; Q17: the increment is added AFTER the
     dissipation): one step from rest equals the undamped run bit for bit
P26  the printed coefficients of Eq. 6a/6b (Q24, hermite_coeff = 1): sqrt 2 and sqrt(3/2), closed form

Every expected value is typed from the paper's formula or is a closed form evaluated on the grid; none comes from the
oracle or from the CUDA path.
"""
import math

import numpy as np
import pytest

from oracle import Oracle
from paper_2511_21891_b200 import synth

TWO_PI = 2 * np.pi


def _grid(nx, ny, nz, Lx=TWO_PI, Ly=TWO_PI, Lz=TWO_PI):
    x = Lx * np.arange(nx) / nx
    y = Ly * np.arange(ny) / ny
    z = Lz * np.arange(nz) / nz
    return np.meshgrid(z, y, x, indexing="ij")


def _half(f):
    return (np.fft.fftn(f) / f.size)[:, :, : f.shape[-1] // 2 + 1]


# ---- P23 ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,bin_round,bin_trunc", [((2, 2, 1), 3, 2),       # kperp = sqrt 8  = 2.83
                                                    ((3, -2, 0), 4, 3),      # kperp = sqrt 13 = 3.61
                                                    ((1, 1, -1), 1, 1)])     # kperp = sqrt 2  = 1.41 (both rules agree: control)
def test_p23_shell_index_rounds_to_nearest(n, bin_round, bin_trunc):
    nx, ny, nz, amp = 16, 16, 8, 0.7 - 0.2j
    o = Oracle(nx, ny, nz)
    o.set_state(synth.single_mode(nx, ny, nz, n, amp, field=0))
    k2 = n[0] ** 2 + n[1] ** 2
    assert int(math.floor(math.sqrt(k2) + 0.5)) == bin_round and int(math.floor(math.sqrt(k2))) == bin_trunc
    s = o.kperp_spectrum(8)
    want = np.zeros(8)
    want[bin_round] = 2 * 0.25 * k2 * abs(amp) ** 2            # the mode and its conjugate partner, 1/4 kperp^2 |xi+|^2 each
    assert np.abs(s - want).max() <= 1e-14 * want.max()
    lit = o.kperp_spectrum(8, literal_eq26=True)               # Eq. 26 as printed: |xi+|^2 + |xi-|^2
    want_l = np.zeros(8)
    want_l[bin_round] = 2 * abs(amp) ** 2
    assert np.abs(lit - want_l).max() <= 1e-14 * want_l.max()


def test_p23_shell_width_uses_the_longer_box_side():
    """Lx = 2 pi, Ly = 4 pi: dk = 2 pi / max(Lx, Ly) = 1/2.  Mode (1,0): kperp = 1 -> bin 2 (bin 1 with min(Lx, Ly));
    mode (0,1): kperp = 2 pi / Ly = 1/2 -> bin 1; mode (1,1): kperp = sqrt(5)/2 = 1.118 -> 2.236 -> bin 2."""
    nx, ny, nz = 16, 16, 8
    for n, b in (((1, 0, 1), 2), ((0, 1, 0), 1), ((1, 1, 0), 2), ((2, 3, 0), 5)):        # (2,3): sqrt(4 + 2.25) = 2.5 -> 5.0 -> bin 5
        o = Oracle(nx, ny, nz, Lx=TWO_PI, Ly=2 * TWO_PI)
        o.set_state(synth.single_mode(nx, ny, nz, n, 1.0, field=1))
        kx, ky = n[0] * 1.0, n[1] * 0.5
        assert int(math.floor(math.sqrt(kx * kx + ky * ky) / 0.5 + 0.5)) == b
        s = o.kperp_spectrum(12)
        assert np.count_nonzero(s) == 1 and s[b] > 0, (n, s)
        assert abs(s[b] - 2 * 0.25 * (kx * kx + ky * ky)) <= 1e-14
    # the mirrored box gives the mirrored answer (the rule does not single out x or y)
    o = Oracle(nx, ny, nz, Lx=2 * TWO_PI, Ly=TWO_PI)
    o.set_state(synth.single_mode(nx, ny, nz, (0, 1, 0), 1.0, field=0))
    assert o.kperp_spectrum(12)[2] > 0


# ---- P24 ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("field", [0, 1])
def test_p24_plus_and_minus_energies_are_not_swapped(field):
    """xi+ alone (field 0) must show up as E+, xi- alone (field 1) as E-; record = {E_A, E+, E-, E_kin, E_mag, W_g} with
    E+- = 1/4 sum kperp^2 |xi+-|^2, Phi = (xi+ + xi-)/2, Psi = (xi+ - xi-)/2."""
    nx, ny, nz, n, amp = 16, 16, 8, (2, 1, 1), 0.6 + 0.3j
    k2 = n[0] ** 2 + n[1] ** 2
    EA = 0.25 * k2 * 2 * abs(amp) ** 2
    want = np.array([EA, EA if field == 0 else 0.0, EA if field == 1 else 0.0, EA / 2, EA / 2, 0.0])
    o = Oracle(nx, ny, nz, nonlinear=0)
    o.set_state(synth.single_mode(nx, ny, nz, n, amp, field=field))
    assert np.abs(o.energy() - want).max() <= 1e-15
    # the per-step history record uses the same order: a linear step only rotates the phase of the one mode
    o.step(0.05, 2)
    h = o.energy_history()
    assert h.shape == (2, 7) and abs(h[1, 0] - 0.1) <= 1e-15
    assert np.abs(h[:, 1:] - want).max() <= 1e-14


# ---- P25 ---------------------------------------------------------------------------------------------------------------
def test_p25_forcing_increment_is_added_after_the_dissipation():
    """From rest the only thing a step does is the forcing increment (Eq. 25).  Dissipation applied BEFORE it acts on zeros,
    so the result is bit for bit that of the undamped run; applied after it, it would shrink the increment by
    exp(-eta kperp^2 dt) <= 0.6 here (and the g_0 increment by the k_z factor)."""
    nx, ny, nz, M, dt = 16, 16, 8, 2, 0.1
    force = dict(force_eps=1.0, force_nperp_min=1, force_nperp_max=2, force_nz_max=1, seed=11, force_g_amp=0.3, force_g_nz=1)
    damp = dict(eta=5.0, r=1, eta_normalized=0, eta_z=3.0, r_z=1, eta_g=2.0, nu_coll=4.0, p=1.0)
    zero_z = np.zeros((2, nz, ny, nx // 2 + 1), dtype=np.complex128)
    zero_g = np.zeros((M, nz, ny, nx // 2 + 1), dtype=np.complex128)
    out = []
    for extra in ({}, damp):
        o = Oracle(nx, ny, nz, M=M, **force, **extra)
        o.set_state(zero_z, zero_g)
        o.step(dt, 1)
        out.append(o.get_state())
    (z0, g0), (z1, g1) = out
    assert np.abs(z0).max() > 1e-3 and np.abs(g0[0]).max() > 1e-3          # both forcings did something
    assert np.array_equal(z0, z1) and np.array_equal(g0, g1)
    # the damping is strong enough that the other order could not hide: a SECOND step damps the first increment
    o = Oracle(nx, ny, nz, M=M, **damp)
    o.set_state(z0, g0)
    o.step(dt, 1)
    z2, g2 = o.get_state()
    assert np.abs(z2).max() < 0.65 * np.abs(z0).max() and np.abs(g2[0]).max() < 0.999 * np.abs(g0[0]).max()


# ---- P26 ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("s", [+1, -1])
def test_p26_literal_eq6ab_coefficients_closed_form(s):
    """hermite_coeff = 1 (Q24): the coupling of g_0 to g_1 is sqrt 2 (Eq. 6a) and of g_1 to g_2 sqrt(3/2) (Eq. 6b); the
    downward couplings and every m >= 2 keep sqrt(m/2), sqrt((m+1)/2).  Single cosines, closed form as in P16."""
    nx, ny, nz, M = 16, 16, 16, 4
    Z, Y, X = _grid(nx, ny, nz)
    ph = lambda n: n[0] * X + n[1] * Y + n[2] * Z                                    # noqa: E731
    br = lambda p, q: (p[0] * q[1] - p[1] * q[0]) * np.sin(ph(p)) * np.sin(ph(q))    # noqa: E731  {cos p.x, cos q.x}
    a, b = (1, 2, 1), (2, -1, 0)
    c = [(1, 1, 1), (-1, 2, 2), (2, 1, -1), (1, -1, 2)]
    amp = [0.9, -0.6, 1.1, 0.5]
    fa, fb = 0.8, 1.2
    Phi, Psi = fa * np.cos(ph(a)), fb * np.cos(ph(b))
    g = [amp[m] * np.cos(ph(c[m])) for m in range(M)]
    dz = [-amp[m] * c[m][2] * np.sin(ph(c[m])) for m in range(M)]
    brPhi = [fa * amp[m] * br(a, c[m]) for m in range(M)]
    brPsi = [fb * amp[m] * br(b, c[m]) for m in range(M)]
    up = [math.sqrt(2.0), math.sqrt(1.5), math.sqrt(3 / 2.0), 0.0]                   # 6a, 6b, 6c at m = 2, absorbing end
    dn = [0.0, 1 / math.sqrt(2.0), math.sqrt(2 / 2.0), math.sqrt(3 / 2.0)]           # 6b, 6c
    zero = np.zeros_like(Phi)
    o = Oracle(nx, ny, nz, M=M, g_sign=s, hermite_coeff=1)
    o.set_state(np.stack([_half(Phi + Psi), _half(Phi - Psi)]), np.stack([_half(v) for v in g]))
    _, dg = o.rhs()
    for m in range(M):
        lo_b, lo_z = (brPsi[m - 1], dz[m - 1]) if m >= 1 else (zero, zero)
        hi_b, hi_z = (brPsi[m + 1], dz[m + 1]) if m + 1 < M else (zero, zero)
        H = -brPhi[m] + s * dz[m] + dn[m] * (lo_b - s * lo_z) + up[m] * (hi_b - s * hi_z)
        ref = _half(H)
        assert np.abs(dg[m] - ref).max() <= 2e-14 * max(1.0, np.abs(ref).max()), m
    # the default (Eq. 6c for every m) differs at m = 0 and m = 1 only
    o2 = Oracle(nx, ny, nz, M=M, g_sign=s, hermite_coeff=0)
    o2.set_state(np.stack([_half(Phi + Psi), _half(Phi - Psi)]), np.stack([_half(v) for v in g]))
    _, dg2 = o2.rhs()
    assert np.abs(dg2[0] - dg[0]).max() > 0.05 and np.abs(dg2[1] - dg[1]).max() > 0.05
    assert np.array_equal(dg2[2], dg[2]) and np.array_equal(dg2[3], dg[3])
