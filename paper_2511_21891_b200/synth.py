"""Seeded synthetic inputs shaped like the paper's workloads.

This module serves BOTH the CUDA path and the CPU oracle (tests, bench) and therefore holds none
of the method's arithmetic: it only draws random phases, places amplitudes on Fourier modes in
the boundary layout, and rescales them to a requested quadratic norm.  It imports neither the
CUDA binding nor the oracle.  numpy only.

Boundary layout (include/gandalf.h): complex128 arrays (fields, nz, ny, nx//2+1), kx = 0..nx/2
fastest, ky and kz in FFT order, physical normalisation f(x) = sum_k fhat(k) exp(+i k.x).
"""
from __future__ import annotations

import numpy as np

TWO_PI = 2.0 * np.pi


def mode_numbers(n: int) -> np.ndarray:
    """Signed integer mode numbers in FFT order: 0..n/2-1, -n/2..-1."""
    m = np.arange(n)
    return np.where(m < n // 2, m, m - n)


def _hermitian_fix_kx0(a: np.ndarray) -> np.ndarray:
    """Make the kx=0 plane of a (nz, ny, hx) half-spectrum self-consistent:
    f(0,-ky,-kz) = conj f(0,ky,kz), so the real-space field is real."""
    p = a[:, :, 0]
    flipped = np.roll(np.flip(p, axis=(0, 1)), shift=(1, 1), axis=(0, 1))   # index (-kz, -ky)
    a[:, :, 0] = 0.5 * (p + np.conj(flipped))
    return a


def _weights(nx: int) -> np.ndarray:
    """Half-plane multiplicities: kx=0 and kx=nx/2 count once, the others twice."""
    w = np.full(nx // 2 + 1, 2.0)
    w[0] = 1.0
    w[-1] = 1.0
    return w


def band_shape(nx, ny, nz, nperp_lo=1.0, nperp_hi=4.0, nz_hi=2, power=-2.0):
    """Amplitude envelope |f(k)| ~ nperp^power on nperp_lo <= nperp <= nperp_hi, |n_z| <= nz_hi
    (BASELINE.json config 0: "|zeta(k)| ~ kperp^-2 for 1<=kperp<=4 and |kz|<=2")."""
    hx = nx // 2 + 1
    mx = np.arange(hx)[None, None, :].astype(float)
    my = mode_numbers(ny)[None, :, None].astype(float)
    mz = mode_numbers(nz)[:, None, None]
    nperp = np.sqrt(mx * mx + my * my)
    sel = (nperp >= nperp_lo) & (nperp <= nperp_hi) & (np.abs(mz) <= nz_hi)
    # never populate Nyquist planes
    sel &= (mx < nx // 2) & (np.abs(my) < ny // 2) & ((np.abs(mz) < nz // 2) | (mz == 0))
    env = np.zeros((nz, ny, hx))
    env[sel] = np.broadcast_to(nperp, env.shape)[sel] ** power
    return env


def random_phase_field(rng, env):
    """One Hermitian-consistent half-spectrum with the given envelope and uniform random phases."""
    ph = rng.uniform(0.0, TWO_PI, size=env.shape)
    a = env * np.exp(1j * ph)
    return _hermitian_fix_kx0(a)


def quad_norm(a, nx, Lx=TWO_PI, Ly=TWO_PI, kperp_weight=False):
    """sum over the FULL spectrum of |a|^2 (optionally times kperp^2), from a half-plane array."""
    nz, ny, hx = a.shape[-3:]
    w = _weights(nx)[None, None, :]
    v = np.abs(a) ** 2 * w
    if kperp_weight:
        kx = TWO_PI * np.arange(hx)[None, None, :] / Lx
        ky = TWO_PI * mode_numbers(ny)[None, :, None] / Ly
        v = v * (kx * kx + ky * ky)
    return float(v.sum())


def random_zeta(nx, ny, nz, seed, Lx=TWO_PI, Ly=TWO_PI, energy=1.0, nperp_hi=4.0, nz_hi=2):
    """Elsasser potentials zeta^+- (2, nz, ny, hx): random phases, |amp| ~ nperp^-2 in the band,
    rescaled so that 1/4 sum_k kperp^2 (|zeta+|^2 + |zeta-|^2) = energy."""
    rng = np.random.default_rng(seed)
    env = band_shape(nx, ny, nz, 1.0, nperp_hi, nz_hi, -2.0)
    z = np.stack([random_phase_field(rng, env), random_phase_field(rng, env)])
    e = 0.25 * (quad_norm(z[0], nx, Lx, Ly, True) + quad_norm(z[1], nx, Lx, Ly, True))
    z *= np.sqrt(energy / e)
    return z


def random_g(nx, ny, nz, M, seed, total=0.01, nperp_hi=4.0, nz_hi=2, filled=2):
    """Hermite moments (M, nz, ny, hx): the first `filled` moments get random-phase nperp^-2 amplitudes,
    each rescaled to 1/2 sum_k |g_m|^2 = total/filled; higher moments start at zero (config 2)."""
    rng = np.random.default_rng(seed)
    g = np.zeros((M, nz, ny, nx // 2 + 1), dtype=np.complex128)
    # include kperp = 0? no: the envelope starts at nperp = 1
    env = band_shape(nx, ny, nz, 1.0, nperp_hi, nz_hi, -2.0)
    for m in range(min(filled, M)):
        a = random_phase_field(rng, env)
        w = 0.5 * quad_norm(a, nx)
        g[m] = a * np.sqrt((total / filled) / w)
    return g


def dense_random(nx, ny, nz, nfields, seed, decay=1.5, amp=1.0):
    """Random complex amplitudes on EVERY half-plane mode (including ones the 2/3 rule removes and
    the Nyquist planes), decaying like (1+|n|)^-decay: exercises the projection in set_state and
    fills the whole retained band for parity tests."""
    rng = np.random.default_rng(seed)
    hx = nx // 2 + 1
    mx = np.arange(hx)[None, None, :].astype(float)
    my = mode_numbers(ny)[None, :, None].astype(float)
    mz = mode_numbers(nz)[:, None, None].astype(float)
    env = amp * (1.0 + np.sqrt(mx * mx + my * my + mz * mz)) ** (-decay)
    out = np.empty((nfields, nz, ny, hx), dtype=np.complex128)
    for f in range(nfields):
        out[f] = env * (rng.standard_normal(env.shape) + 1j * rng.standard_normal(env.shape))
    return out


def orszag_tang(nx, ny, nz):
    """BASELINE.json config 1: Phi = -2(cos x + cos y), Psi = cos 2x + 2 cos y on a 2 pi box,
    uniform in z; returns zeta^+- = Phi +- Psi as half-plane coefficients."""
    hx = nx // 2 + 1
    phi = np.zeros((nz, ny, hx), dtype=np.complex128)
    psi = np.zeros((nz, ny, hx), dtype=np.complex128)
    # cos x -> 1/2 at kx=+-1 (only +1 stored); cos y -> 1/2 at ky=+-1 on the kx=0 plane
    phi[0, 0, 1] = -1.0
    phi[0, 1, 0] = -1.0
    phi[0, ny - 1, 0] = -1.0
    psi[0, 0, 2] = 0.5
    psi[0, 1, 0] = 1.0
    psi[0, ny - 1, 0] = 1.0
    return np.stack([phi + psi, phi - psi])


def single_mode(nx, ny, nz, n, amp, field=0, nfields=2):
    """One Fourier mode n = (n_x >= 0, n_y, n_z) (and its conjugate partner when n_x = 0)."""
    hx = nx // 2 + 1
    a = np.zeros((nfields, nz, ny, hx), dtype=np.complex128)
    ix, iy, iz = n[0], n[1] % ny, n[2] % nz
    assert 0 <= ix < hx
    a[field, iz, iy, ix] = amp
    if ix == 0:
        a[field, (-n[2]) % nz, (-n[1]) % ny, 0] = np.conj(amp)
    return a
