"""Pins for the CPU oracle (-m "not gpu"): every check compares oracle/ against something the
paper or the mathematics fixes, never against itself.  Pin numbers are DESIGN.md's P0..P11."""
import math
import os

import numpy as np
import pytest

import oracle
from oracle import Oracle
from paper_2511_21891_b200 import synth

GOLD = os.path.join(os.path.dirname(__file__), "golden")
TWO_PI = 2 * np.pi


def _rows(name):
    out = []
    with open(os.path.join(GOLD, name)) as fh:
        for line in fh:
            line = line.split("#")[0].strip()
            if line:
                out.append(line.split())
    return out


def _full_from_half(h, nx):
    """Hermitian completion of a (nz, ny, hx) half-spectrum to (nz, ny, nx) -- test-side helper."""
    nz, ny, hx = h.shape
    full = np.zeros((nz, ny, nx), dtype=np.complex128)
    full[:, :, :hx] = h
    for ix in range(1, nx // 2):
        src = h[:, :, ix]
        full[:, :, nx - ix] = np.conj(np.roll(np.flip(src, axis=(0, 1)), (1, 1), axis=(0, 1)))
    return full


# ---- P0: own FFT against the O(N^2) definition and against numpy ---------------------------
@pytest.mark.parametrize("n", [2, 4, 8, 16, 32, 64])
def test_p0_fft_matches_dft(n):
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    for sign in (-1, +1):
        a = oracle.fft1d(x, sign)
        b = oracle.dft1d(x, sign)
        ref = np.fft.fft(x) if sign < 0 else np.fft.ifft(x) * n
        assert np.linalg.norm(a - b) <= 1e-13 * np.linalg.norm(b)
        assert np.linalg.norm(b - ref) <= 1e-13 * np.linalg.norm(ref)
    back = oracle.fft1d(oracle.fft1d(x, -1), +1) / n
    assert np.linalg.norm(back - x) <= 1e-14 * np.linalg.norm(x)


# ---- P1: linear Alfven wave propagates with the exact phase (Table 1) ------
@pytest.mark.parametrize("row", _rows("alfven_table1.txt"), ids=lambda r: r[0])
@pytest.mark.parametrize("nonlinear", [0, 1])
def test_p1_alfven_wave_table1(row, nonlinear):
    label, frac, omega_paper, bound = row[0], int(row[1]), float(row[2]), float(row[3])
    T = TWO_PI
    if frac == 0:
        dt, nsteps = 0.01, 300
    else:
        dt, nsteps = T / frac, frac          # one period
    o = Oracle(16, 16, 8, nonlinear=nonlinear)
    z0 = synth.single_mode(16, 16, 8, (1, 0, 1), 0.01, field=0)
    o.set_state(z0)
    phases = [0.0]
    prev = z0[0, 1, 0, 1]
    for _ in range(nsteps):
        o.step(dt, 1)
        z, _g = o.get_state()
        cur = z[0, 1, 0, 1]
        phases.append(phases[-1] + np.angle(cur / prev))     # unwrapped increment; |dphi| < pi needs dt<T/2
        prev = cur
    z, _ = o.get_state()
    expect = 0.01 * np.exp(1j * 1.0 * 1.0 * dt * nsteps)
    assert abs(z[0, 1, 0, 1] - expect) <= 1e-15 * nsteps * 10 * 0.01 + 1e-17
    if frac != 2:   # at dt = T/2 the per-step phase is exactly pi and cannot be unwrapped
        t = dt * np.arange(nsteps + 1)
        omega = np.polyfit(t, np.array(phases), 1)[0]
        assert abs(omega - 1.0) <= bound
        assert abs(omega - 1.0) <= abs(omega_paper - 1.0) + 1e-13
    # nothing else got excited
    z[0, 1, 0, 1] = 0
    assert np.abs(z).max() == 0.0


def test_p1_alfven_minus_field_and_speed():
    o = Oracle(16, 16, 8, vA=2.5, nonlinear=1)
    z0 = synth.single_mode(16, 16, 8, (2, 1, -1), 0.3 - 0.1j, field=1)
    o.set_state(z0)
    o.step(0.37, 5)
    z, _ = o.get_state()
    kz = -1.0
    expect = (0.3 - 0.1j) * np.exp(-1j * kz * 2.5 * 0.37 * 5)     # xi^- carries exp(-i kz vA t)
    assert abs(z[1, 7, 1, 2] - expect) <= 1e-14


# ---- P2: bracket of single Fourier modes, closed form ---------------------------
def test_p2_bracket_single_modes_closed_form():
    nx, ny, nz = 16, 16, 4
    o = Oracle(nx, ny, nz)
    a, b = (1, 2, 1), (2, -1, 0)
    x = TWO_PI * np.arange(nx) / nx
    y = TWO_PI * np.arange(ny) / ny
    zc = TWO_PI * np.arange(nz) / nz
    Z, Y, X = np.meshgrid(zc, y, x, indexing="ij")
    f = np.cos(a[0] * X + a[1] * Y + a[2] * Z)
    g = np.cos(b[0] * X + b[1] * Y + b[2] * Z)
    cross = a[0] * b[1] - a[1] * b[0]
    amb = tuple(a[i] - b[i] for i in range(3))
    apb = tuple(a[i] + b[i] for i in range(3))
    exact = cross * 0.5 * (np.cos(amb[0] * X + amb[1] * Y + amb[2] * Z) - np.cos(apb[0] * X + apb[1] * Y + apb[2] * Z))
    fh, gh, eh = (np.fft.fftn(v) / v.size for v in (f, g, exact))
    out, max_imag = o.bracket_full(fh, gh)
    assert max_imag <= 1e-14
    assert np.abs(out - eh).max() <= 1e-14
    # antisymmetry and the sign convention {P,Q} = Px Qy - Py Qx
    out2, _ = o.bracket_full(gh, fh)
    assert np.abs(out + out2).max() <= 1e-15
    assert abs(cross) == 5 and np.abs(eh).max() > 1.0


# ---- P3: dealiased pseudo-spectral bracket == truncated convolution sum (brute force) --------
@pytest.mark.parametrize("shape", [(8, 8, 2), (8, 8, 4), (16, 8, 4)])
def test_p3_bracket_equals_convolution_sum(shape):
    nx, ny, nz = shape
    o = Oracle(nx, ny, nz)
    h = synth.dense_random(nx, ny, nz, 2, seed=7, decay=0.5)
    mx, my, mz = synth.mode_numbers(nx), synth.mode_numbers(ny), synth.mode_numbers(nz)
    keep = ((3 * np.abs(mz)[:, None, None] <= nz) & (3 * np.abs(my)[None, :, None] <= ny)
            & (3 * np.abs(mx)[None, None, :] <= nx))
    fulls = []
    for f in range(2):
        hf = h[f].copy()
        hf[:, :, 0] = 0.5 * (hf[:, :, 0] + np.conj(np.roll(np.flip(hf[:, :, 0], (0, 1)), (1, 1), (0, 1))))
        full = _full_from_half(hf, nx) * keep
        fulls.append(full)
    out, _ = o.bracket_full(fulls[0], fulls[1])
    modes = [(iz, iy, ix) for iz in range(nz) for iy in range(ny) for ix in range(nx) if keep[iz, iy, ix]]
    brute = np.zeros((nz, ny, nx), dtype=np.complex128)
    for (pz, py, px) in modes:
        fp = fulls[0][pz, py, px]
        for (qz, qy, qx) in modes:
            kx, ky, kz = mx[px] + mx[qx], my[py] + my[qy], mz[pz] + mz[qz]
            if 3 * abs(kx) > nx or 3 * abs(ky) > ny or 3 * abs(kz) > nz:
                continue
            # physical wavenumbers equal mode numbers on the 2 pi box
            coeff = -(mx[px] * my[qy] - my[py] * mx[qx])
            brute[kz % nz, ky % ny, kx % nx] += coeff * fp * fulls[1][qz, qy, qx]
    assert np.abs(out - brute).max() <= 1e-13 * max(1.0, np.abs(brute).max())
    assert np.abs(brute).max() > 1e-3
    assert np.abs(out[~keep]).max() == 0.0


# ---- P6: mask definition and retained counts (Eq. 20) ---------------------------
@pytest.mark.parametrize("row", _rows("retained_counts.txt"), ids=lambda r: "x".join(r[:3]))
def test_p6_retained_counts(row):
    nx, ny, nz, Kx, Ky, Kz = map(int, row)
    o = Oracle(nx, ny, nz, M=1)
    ones = np.ones((1, nz, ny, nx // 2 + 1), dtype=np.complex128)
    o.set_state(np.zeros((2, nz, ny, nx // 2 + 1)), ones)
    _, g = o.get_state()
    kept = g[0] != 0
    assert kept.sum() == Kx * Ky * Kz
    assert kept.any(axis=(0, 1)).sum() == Kx and kept.any(axis=(0, 2)).sum() == Ky and kept.any(axis=(1, 2)).sum() == Kz
    if nz == 2:
        assert not kept[1].any()      # only kz = 0 survives
