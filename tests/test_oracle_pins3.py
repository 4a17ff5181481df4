"""Oracle pins, round 2 (-m "not gpu"): the parts a one-line mistake could slip through before.

P15  sign and scale of N+- (Eq. 1): single-cosine Elsasser potentials, closed form
P16  signs of the three bracket terms of H_m and of the streaming terms (Eq. 6): closed form
P17  advective CFL step (Eq. 16): Orszag-Tang max|grad Phi| = 2 sqrt 2, anisotropic grids, C, dt_max
P18  perpendicular / parallel hyperdissipation on g_m (eta_g, Q9): closed-form decay
P19  one complete Algorithm-1 step (Eq. 15) re-evaluated by brute force on a tiny grid: brackets from
     the truncated convolution sum (no FFT anywhere), phases typed from the paper; both integrating-factor variants
P20  restart: N steps == N/2 steps + (state, time, step) carried to a NEW context + N/2 steps, forcing on (bit exact)

Every expected value here is a closed form evaluated on the grid (numpy's FFT only converts it to coefficients) or a
brute-force sum; none comes from the oracle or from the CUDA path.
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
    return np.meshgrid(z, y, x, indexing="ij")       # Z, Y, X with shape (nz, ny, nx)


def _half(f):
    """real-space field (nz, ny, nx) -> half-plane coefficients with the physical normalisation (Eq. 9)."""
    nx = f.shape[-1]
    return (np.fft.fftn(f) / f.size)[:, :, : nx // 2 + 1]


def _ph(n, X, Y, Z):
    return n[0] * X + n[1] * Y + n[2] * Z


def _br_cos(p, q, X, Y, Z):
    """{cos p.x, cos q.x} = (p_x q_y - p_y q_x) sin(p.x) sin(q.x)  from {P,Q} = Px Qy - Py Qx."""
    return (p[0] * q[1] - p[1] * q[0]) * np.sin(_ph(p, X, Y, Z)) * np.sin(_ph(q, X, Y, Z))


# ---- P15: N+- of Eq. 1 for xi+ = alpha cos a.x, xi- = beta cos b.x ---------------------------------------------------
@pytest.mark.parametrize("a,b", [((1, 2, 1), (3, -1, 0)), ((2, 1, -1), (1, -3, 1)), ((3, 0, 1), (1, 1, 1))])
def test_p15_elsasser_rhs_sign_and_scale_closed_form(a, b):
    nx, ny, nz = 16, 16, 8
    al, be = 0.7, -1.3
    Z, Y, X = _grid(nx, ny, nz)
    a2, b2 = a[0] ** 2 + a[1] ** 2, b[0] ** 2 + b[1] ** 2
    assert a2 != b2 and a[0] * b[1] - a[1] * b[0] != 0
    xp, xm = al * np.cos(_ph(a, X, Y, Z)), be * np.cos(_ph(b, X, Y, Z))
    # w+- = lap xi+- = -|a|^2 xi+, -|b|^2 xi-  =>  {xi+,w-} + {xi-,w+} = (-|b|^2 + |a|^2) {xi+,xi-}
    C = al * be * _br_cos(a, b, X, Y, Z)                       # {xi+, xi-}
    A = (a2 - b2) * C
    amb = tuple(a[i] - b[i] for i in range(3))
    apb = tuple(a[i] + b[i] for i in range(3))
    cross = a[0] * b[1] - a[1] * b[0]
    # C = al be cross/2 [cos((a-b).x) - cos((a+b).x)]  =>  lap C termwise
    lapC = al * be * cross * 0.5 * (-(amb[0] ** 2 + amb[1] ** 2) * np.cos(_ph(amb, X, Y, Z))
                                    + (apb[0] ** 2 + apb[1] ** 2) * np.cos(_ph(apb, X, Y, Z)))
    assert np.abs(C - al * be * cross * 0.5 * (np.cos(_ph(amb, X, Y, Z)) - np.cos(_ph(apb, X, Y, Z)))).max() < 1e-13
    Np = -0.5 * (A - lapC)                                       # Eq. 1, upper signs
    Nm = -0.5 * (A + lapC)                                       # Eq. 1, lower signs
    o = Oracle(nx, ny, nz)
    o.set_state(np.stack([_half(xp), _half(xm)]))
    dw, _ = o.rhs()
    scale = max(np.abs(_half(Np)).max(), np.abs(_half(Nm)).max())
    assert scale > 0.1
    assert np.abs(dw[0] - _half(Np)).max() <= 1e-14 * scale
    assert np.abs(dw[1] - _half(Nm)).max() <= 1e-14 * scale
    # the two signs of the lap{xi+,xi-} term are really different here (a wrong sign cannot hide)
    assert np.abs(_half(Np) - _half(Nm)).max() > 0.1 * scale


# ---- P16: H_m of Eq. 6 for single-cosine Phi, Psi, g_0, g_1, g_2 -------------------------------------------------------
@pytest.mark.parametrize("s", [+1, -1])
@pytest.mark.parametrize("closure", [0, 1])
def test_p16_hermite_rhs_signs_closed_form(s, closure):
    nx, ny, nz, M = 16, 16, 16, 4
    Z, Y, X = _grid(nx, ny, nz)
    a, b = (1, 2, 1), (2, -1, 0)                                 # Phi, Psi
    c = [(1, 1, 1), (-1, 2, 2), (2, 1, -1), (1, -1, 2)]          # g_0 .. g_3
    amp = [0.9, -0.6, 1.1, 0.5 if closure else 0.0]              # absorbing case: g_3 = 0 exercises the one-sided rows
    fa, fb = 0.8, 1.2
    Phi, Psi = fa * np.cos(_ph(a, X, Y, Z)), fb * np.cos(_ph(b, X, Y, Z))
    g = [amp[m] * np.cos(_ph(c[m], X, Y, Z)) for m in range(M)]
    dz = [-amp[m] * c[m][2] * np.sin(_ph(c[m], X, Y, Z)) for m in range(M)]          # d g_m / dz
    brPhi = [fa * amp[m] * _br_cos(a, c[m], X, Y, Z) for m in range(M)]              # {Phi, g_m}
    brPsi = [fb * amp[m] * _br_cos(b, c[m], X, Y, Z) for m in range(M)]              # {Psi, g_m}
    zero = np.zeros_like(Phi)
    H = []
    for m in range(M):
        dn, up = math.sqrt(m / 2.0), math.sqrt((m + 1) / 2.0)                        # Eq. 6c
        lo_b, lo_z = (brPsi[m - 1], dz[m - 1]) if m >= 1 else (zero, zero)
        if m + 1 < M:
            hi_b, hi_z = brPsi[m + 1], dz[m + 1]
        elif closure == 1:                                                           # g_M := g_{M-2}  (Q23)
            hi_b, hi_z = brPsi[M - 2], dz[M - 2]
        else:
            hi_b, hi_z = zero, zero
        # d g_m/dt = -{Phi,g_m} +- dz g_m + dn [{Psi,g_{m-1}} -+ dz g_{m-1}] + up [{Psi,g_{m+1}} -+ dz g_{m+1}]   (Eq. 6)
        H.append(-brPhi[m] + s * dz[m] + dn * (lo_b - s * lo_z) + up * (hi_b - s * hi_z))
    o = Oracle(nx, ny, nz, M=M, g_sign=s, closure=closure)
    o.set_state(np.stack([_half(Phi + Psi), _half(Phi - Psi)]), np.stack([_half(v) for v in g]))
    _, dg = o.rhs()
    for m in range(M):
        ref = _half(H[m])
        assert np.abs(ref).max() > 0.05
        assert np.abs(dg[m] - ref).max() <= 2e-14 * max(1.0, np.abs(ref).max()), m
    # each of the three bracket terms and the streaming term matters in this configuration
    assert min(np.abs(v).max() for v in brPhi[:3]) > 0.1 and min(np.abs(v).max() for v in brPsi[:3]) > 0.1


# ---- P17: Eq. 16 --------------------------------------------------------------------------------------------------------
def test_p17_cfl_dt_orszag_tang_exact():
    # Phi = -2(cos x + cos y): |grad Phi|^2 = 4 (sin^2 x + sin^2 y), max 8 at x = y = pi/2, a grid point when 4 | N
    for n in (16, 32):
        o = Oracle(n, n, 2)
        o.set_state(synth.orszag_tang(n, n, 2))
        o.step(0.0, 1)
        t, step, last = o.time()
        expect = 0.3 * (TWO_PI / n) / (2.0 * math.sqrt(2.0))
        assert step == 1 and abs(last - expect) <= 1e-15 and abs(t - expect) <= 1e-15


@pytest.mark.parametrize("Lx,Ly,nx,ny", [(TWO_PI, 2 * TWO_PI, 16, 16), (2 * TWO_PI, TWO_PI, 16, 16), (TWO_PI, TWO_PI, 32, 16),
                                         (TWO_PI, TWO_PI, 16, 32)])
def test_p17_cfl_uses_min_spacing_sqrt_of_max_and_C(Lx, Ly, nx, ny):
    # Phi = 2A cos(2 pi x / Lx):  max |grad Phi| = 2A * 2 pi / Lx  (attained on the grid: 4 | nx);  xi+ = xi- = Phi
    A, C = 0.37, 0.25
    ph = np.zeros((8, ny, nx // 2 + 1), dtype=np.complex128)
    ph[0, 0, 1] = A
    o = Oracle(nx, ny, 8, Lx=Lx, Ly=Ly, cfl=C)
    o.set_state(np.stack([ph, ph]))
    o.step(-1.0, 1)
    vmax = 2 * A * TWO_PI / Lx
    expect = C * min(Lx / nx, Ly / ny) / vmax
    assert abs(o.time()[2] - expect) <= 1e-15
    assert abs(vmax - 1.0) > 0.05 and Lx / nx != Ly / ny        # sqrt and min are both discriminating here
    # dt_max caps it
    o2 = Oracle(nx, ny, 8, Lx=Lx, Ly=Ly, cfl=C, dt_max=0.5 * expect)
    o2.set_state(np.stack([ph, ph]))
    o2.step(-1.0, 1)
    assert abs(o2.time()[2] - 0.5 * expect) <= 1e-16


def test_p17_cfl_zero_flow_is_an_error_unless_dt_max():
    nx, ny, nz, M = 8, 8, 4, 2
    g = synth.dense_random(nx, ny, nz, M, seed=3)
    o = Oracle(nx, ny, nz, M=M)
    o.set_state(np.zeros((2, nz, ny, nx // 2 + 1)), g)
    before = o.get_state()[1].copy()
    with pytest.raises(RuntimeError):
        o.step(0.0, 1)
    assert np.array_equal(o.get_state()[1], before) and o.time()[1] == 0        # state untouched
    o2 = Oracle(nx, ny, nz, M=M, dt_max=1e-2)
    o2.set_state(np.zeros((2, nz, ny, nx // 2 + 1)), g)
    o2.step(0.0, 2)
    assert abs(o2.time()[0] - 2e-2) <= 1e-16


# ---- P18: eta_g --------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("normalized", [0, 1])
def test_p18_eta_g_decay_closed_form(normalized):
    nx, ny, nz, M = 16, 16, 8, 4
    eta, eta_g, r, nu, p, eta_z, r_z = 0.7, 0.45, 2, 0.9, 2.0, 0.3, 2
    o = Oracle(nx, ny, nz, M=M, eta=eta, r=r, eta_normalized=normalized, nu_coll=nu, p=p, nonlinear=0, eta_z=eta_z, r_z=r_z,
               eta_g=eta_g)
    mode, m = (1, 2, 0), 3                                        # kz = 0: no streaming, the amplitude only decays
    o.set_state(np.zeros((2, nz, ny, nx // 2 + 1)), synth.single_mode(nx, ny, nz, mode, 0.25, field=m, nfields=M))
    dt, n = 0.05, 7
    o.step(dt, n)
    k2 = float(mode[0] ** 2 + mode[1] ** 2)
    k2max = (np.pi * nx / TWO_PI) ** 2 + (np.pi * ny / TWO_PI) ** 2
    shape = (k2 / k2max) ** r if normalized else k2 ** r
    rate = eta_g * shape + nu * (m / M) ** (2 * p)                # kz = 0: the eta_z factor is 1
    got = abs(o.get_state()[1][m, 0, 2, 1])
    assert abs(got - 0.25 * math.exp(-rate * dt * n)) <= 1e-15
    assert abs(math.exp(-eta_g * shape * dt * n) - 1.0) > 1e-4    # eta_g matters at this mode
    # with kz != 0 and streaming switched off by M = 1 ... the parallel factor multiplies too (g_0 alone: H_0 = s i kz g_0)
    o2 = Oracle(nx, ny, nz, M=1, nonlinear=0, eta_z=eta_z, r_z=r_z, eta_g=eta_g, eta_normalized=normalized, r=r)
    o2.set_state(np.zeros((2, nz, ny, nx // 2 + 1)), synth.single_mode(nx, ny, nz, (1, 2, 2), 0.25, field=0, nfields=1))
    o2.step(1e-3, 4)
    kzmax2 = (np.pi * nz / TWO_PI) ** 2
    rate2 = eta_g * shape + eta_z * (4.0 / kzmax2) ** r_z
    # |g_0| under RK2 of dg/dt = i kz g: |1 + i th - th^2/2| per step, th = kz dt
    th = 2.0 * 1e-3
    amp = abs(1 + 1j * th - 0.5 * th * th) ** 4
    assert abs(abs(o2.get_state()[1][0, 2, 2, 1]) - 0.25 * amp * math.exp(-rate2 * 4e-3)) <= 1e-15


# ---- P19: one full Algorithm-1 step by brute force --------------------------------------------------------------------
def _modes(n):
    return [i if i < n // 2 else i - n for i in range(n)]


def _conv_bracket(f, g, nx, ny, nz):
    """Truncated convolution sum of {f,g}^(k) = sum_{p+q=k} (p_y q_x - p_x q_y) f(p) g(q) over the nonzero entries of the
    full spectra f, g (dict mode -> coefficient), k restricted to the retained band 3|n| <= N (Eq. 20).
    {P,Q} = Px Qy - Py Qx with d/dx -> i k: (i p_x)(i q_y) - (i p_y)(i q_x) = p_y q_x - p_x q_y."""
    out = {}
    for p, fp in f.items():
        for q, gq in g.items():
            k = (p[0] + q[0], p[1] + q[1], p[2] + q[2])
            if 3 * abs(k[0]) > nx or 3 * abs(k[1]) > ny or 3 * abs(k[2]) > nz:
                continue
            out[k] = out.get(k, 0.0) + (p[1] * q[0] - p[0] * q[1]) * fp * gq
    return out


def _add(*terms):
    out = {}
    for c, d in terms:
        for k, v in d.items():
            out[k] = out.get(k, 0.0) + c * v
    return out


def _rhs_brute(w, g, nx, ny, nz, s):
    """Eq. 1 and Eq. 6 (L = 2 pi so k = n) on dict spectra; w = [w+, w-], g = [g_0..g_{M-1}] (absorbing closure)."""
    xi = [{k: -v / (k[0] ** 2 + k[1] ** 2) for k, v in wf.items() if k[0] ** 2 + k[1] ** 2 > 0} for wf in w]
    A = _add((1.0, _conv_bracket(xi[0], w[1], nx, ny, nz)), (1.0, _conv_bracket(xi[1], w[0], nx, ny, nz)))
    B = _conv_bracket(xi[0], xi[1], nx, ny, nz)
    lapB = {k: -(k[0] ** 2 + k[1] ** 2) * v for k, v in B.items()}
    N = [_add((-0.5, A), (+0.5, lapB)), _add((-0.5, A), (-0.5, lapB))]                # -1/2 [A -+ lap B]
    Phi, Psi = _add((0.5, xi[0]), (0.5, xi[1])), _add((0.5, xi[0]), (-0.5, xi[1]))
    M = len(g)
    H = []
    for m in range(M):
        dn, up = math.sqrt(m / 2.0), math.sqrt((m + 1) / 2.0)
        terms = [(-1.0, _conv_bracket(Phi, g[m], nx, ny, nz)), (1.0, {k: 1j * s * k[2] * v for k, v in g[m].items()})]
        if m >= 1:
            terms += [(dn, _conv_bracket(Psi, g[m - 1], nx, ny, nz)), (-dn, {k: 1j * s * k[2] * v for k, v in g[m - 1].items()})]
        if m + 1 < M:
            terms += [(up, _conv_bracket(Psi, g[m + 1], nx, ny, nz)), (-up, {k: 1j * s * k[2] * v for k, v in g[m + 1].items()})]
        H.append(_add(*terms))
    return N, H


def _to_dict(full, nx, ny, nz):
    mx, my, mz = _modes(nx), _modes(ny), _modes(nz)
    return {(mx[ix], my[iy], mz[iz]): full[iz, iy, ix] for iz in range(nz) for iy in range(ny) for ix in range(nx)
            if full[iz, iy, ix] != 0}


@pytest.mark.parametrize("if_variant", [0, 1])
def test_p19_one_step_brute_force(if_variant):
    nx, ny, nz, M, s, vA, dt = 8, 8, 8, 2, 1, 1.0, 0.05
    o = Oracle(nx, ny, nz, M=M, if_variant=if_variant, g_sign=s, vA=vA)
    o.set_state(synth.dense_random(nx, ny, nz, 2, seed=51, decay=2.0), synth.dense_random(nx, ny, nz, M, seed=52, decay=2.0))
    w = [_to_dict(o.get_full(f), nx, ny, nz) for f in range(2)]
    g = [_to_dict(o.get_full(2 + m), nx, ny, nz) for m in range(M)]
    sg = [+1.0, -1.0]

    def phase(k, frac, a):
        return np.exp(1j * sg[a] * k[2] * vA * dt * frac)        # exp(+-i kz vA dt * frac)

    N0, H0 = _rhs_brute(w, g, nx, ny, nz, s)
    keys = set().union(*[set(d) for d in w + g + N0 + H0])
    wh = []
    for a in range(2):
        d = {}
        for k in keys:
            wn, Nn = w[a].get(k, 0.0), N0[a].get(k, 0.0)
            if if_variant == 0:                                  # Eq. 15 / Alg. 1 l.3: the phase appears twice
                d[k] = phase(k, 0.5, a) * (wn + phase(k, 0.5, a) * 0.5 * dt * Nn)
            else:                                                # standard integrating-factor midpoint (Q6)
                d[k] = phase(k, 0.5, a) * (wn + 0.5 * dt * Nn)
        wh.append(d)
    gh = [{k: g[m].get(k, 0.0) + 0.5 * dt * H0[m].get(k, 0.0) for k in keys} for m in range(M)]      # Alg. 1 l.4
    N1, H1 = _rhs_brute(wh, gh, nx, ny, nz, s)
    keys = keys.union(*[set(d) for d in N1 + H1])
    o.step(dt, 1)
    scale = max(np.abs(o.get_full(f)).max() for f in range(2 + M))
    for a in range(2):
        got = _to_dict(o.get_full(a), nx, ny, nz)
        for k in keys:
            wn, Nh = w[a].get(k, 0.0), N1[a].get(k, 0.0)
            if if_variant == 0:                                  # Alg. 1 l.8
                ref = phase(k, 1.0, a) * (wn + phase(k, 1.0, a) * dt * Nh)
            else:
                ref = phase(k, 1.0, a) * wn + phase(k, 0.5, a) * dt * Nh
            assert abs(got.get(k, 0.0) - ref) <= 1e-13 * scale, (a, k)
    for m in range(M):
        got = _to_dict(o.get_full(2 + m), nx, ny, nz)
        for k in keys:
            ref = g[m].get(k, 0.0) + dt * H1[m].get(k, 0.0)      # Alg. 1 l.9
            assert abs(got.get(k, 0.0) - ref) <= 1e-13 * scale, (m, k)
    # the two variants differ by far more than the tolerance on this state (kz != 0, N != 0)
    o2 = Oracle(nx, ny, nz, M=M, if_variant=1 - if_variant, g_sign=s, vA=vA)
    o2.set_state(synth.dense_random(nx, ny, nz, 2, seed=51, decay=2.0), synth.dense_random(nx, ny, nz, M, seed=52, decay=2.0))
    o2.step(dt, 1)
    assert max(np.abs(o2.get_full(f) - o.get_full(f)).max() for f in range(2)) > 1e-6 * scale


def test_p9_orders_separate_the_two_variants():
    """DESIGN.md Q6: the paper-literal double phase is first order, the standard integrating-factor midpoint second."""
    def _run_cfg0_like(if_variant, dt, tend):
        nx, ny, nz = 16, 16, 8
        o = Oracle(nx, ny, nz, if_variant=if_variant, vA=1.0)
        o.set_state(synth.random_zeta(nx, ny, nz, seed=5, energy=1.0, nperp_hi=3.0, nz_hi=2))
        o.step(dt, int(round(tend / dt)))
        return o.get_state()[0].ravel()

    tend = 0.2
    orders = {}
    for v in (0, 1):
        ref = _run_cfg0_like(v, tend / 256, tend)
        e = [np.linalg.norm(_run_cfg0_like(v, tend / n, tend) - ref) for n in (16, 32)]
        orders[v] = math.log2(e[0] / e[1])
    assert 0.9 < orders[0] < 1.3, orders
    assert 1.9 < orders[1] < 2.1, orders


# ---- P20: restart through get_state / set_state / set_time -------------------------------------------------------------
def test_p20_restart_is_bit_exact_with_forcing():
    nx, ny, nz, M, dt = 8, 8, 8, 3, 2e-3
    kw = dict(M=M, force_eps=0.7, seed=99, force_g_amp=0.2, force_g_nz=1, nu_coll=0.3, p=2.0, eta=0.2, r=2, eta_normalized=1)
    z = synth.dense_random(nx, ny, nz, 2, seed=61, decay=2.0)
    g = synth.dense_random(nx, ny, nz, M, seed=62, decay=2.0)
    a = Oracle(nx, ny, nz, **kw)
    a.set_state(z, g)
    a.step(dt, 6)
    b = Oracle(nx, ny, nz, **kw)
    b.set_state(z, g)
    b.step(dt, 3)
    t, step, _ = b.time()
    full = [b.get_full(f) for f in range(2 + M)]                  # exact checkpoint of the evolved variables w+-, g_m
    c = Oracle(nx, ny, nz, **kw)
    for f in range(2 + M):
        c.set_full(f, full[f])
    c.set_time(t, step)
    c.step(dt, 3)
    for f in range(2 + M):
        assert np.array_equal(c.get_full(f), a.get_full(f)), f
    assert c.time()[:2] == a.time()[:2]
    # without set_time the forcing sequence restarts from counter 0: a different trajectory
    d = Oracle(nx, ny, nz, **kw)
    for f in range(2 + M):
        d.set_full(f, full[f])
    d.step(dt, 3)
    assert not np.array_equal(d.get_full(0), a.get_full(0))


# ---- P21: exact propagator of the Hermite streaming terms (hermite_exact = 1; Q30) ---------------------------
def _jacobi(M):
    T = np.zeros((M, M))
    for m in range(1, M):
        T[m, m - 1] = T[m - 1, m] = math.sqrt(m / 2.0)
    return T


@pytest.mark.parametrize("sign", [+1, -1])
def test_p21_exact_streaming_closed_form_at_any_dt(sign):
    """Brackets off: g(t) = exp(s i kz (I - T) t) g(0).  From g = delta_{m0} the infinite hierarchy gives
    e^{i s a} e^{-a^2/4} (-i s a/sqrt 2)^m / sqrt(m!), a = kz t (generating function of the Hermite functions); M = 40
    reproduces it to 1e-12 at a = 2.  With the exact propagator this holds for ONE step of dt = 1 as well as for 7."""
    import scipy.linalg
    nx, ny, nz, M, kz, tend = 8, 8, 8, 40, 2, 1.0
    a = kz * tend
    closed = np.array([np.exp(1j * sign * a) * math.exp(-a * a / 4) * (-1j * sign * a / math.sqrt(2)) ** m / math.sqrt(math.factorial(m))
                       for m in range(M)])
    lib = scipy.linalg.expm(1j * sign * kz * (np.eye(M) - _jacobi(M)) * tend)[:, 0]
    assert np.abs(lib - closed).max() <= 1e-12
    g0 = synth.single_mode(nx, ny, nz, (1, 0, kz), 1.0, field=0, nfields=M)
    for nsteps in (1, 7):
        o = Oracle(nx, ny, nz, M=M, nonlinear=0, g_sign=sign, hermite_exact=1)
        o.set_state(np.zeros((2, nz, ny, nx // 2 + 1)), g0)
        w0 = o.energy()[5]
        o.step(tend / nsteps, nsteps)
        got = o.get_state()[1][:, kz, 0, 1]
        assert np.abs(got - closed).max() <= 1e-12, nsteps
        assert abs(o.energy()[5] - w0) <= 1e-13 * w0                 # the propagator is unitary: W_g exactly conserved
    # the plain RK2 of Alg. 1 l.4/l.9 is unstable at this step (|1 + i th - th^2/2| > 1): that is the constraint this lifts
    o = Oracle(nx, ny, nz, M=M, nonlinear=0, g_sign=sign)
    o.set_state(np.zeros((2, nz, ny, nx // 2 + 1)), g0)
    o.step(tend, 1)
    assert np.abs(o.get_state()[1][:, kz, 0, 1] - closed).max() > 0.1


def test_p21_exact_streaming_reflecting_closure_vs_library_expm():
    import scipy.linalg
    nx, ny, nz, M, kz = 8, 8, 8, 6, 1
    T = _jacobi(M)
    T[M - 1, M - 2] += math.sqrt(M / 2.0)                             # g_M := g_{M-2}  (Q23)
    exact = scipy.linalg.expm(1j * kz * (np.eye(M) - T) * 0.9)[:, 0]
    o = Oracle(nx, ny, nz, M=M, nonlinear=0, closure=1, hermite_exact=1)
    o.set_state(np.zeros((2, nz, ny, nx // 2 + 1)), synth.single_mode(nx, ny, nz, (1, 0, kz), 1.0, field=0, nfields=M))
    o.step(0.3, 3)
    assert np.abs(o.get_state()[1][:, kz, 0, 1] - exact).max() <= 1e-13


def test_p21_exact_streaming_with_brackets_is_second_order_and_consistent():
    nx, ny, nz, M, tend = 16, 16, 8, 4, 0.2
    z = synth.random_zeta(nx, ny, nz, seed=5, energy=1.0, nperp_hi=3.0, nz_hi=2)
    g = synth.random_g(nx, ny, nz, M, seed=6, total=0.05, nperp_hi=3.0)

    def run(exact, n):
        o = Oracle(nx, ny, nz, M=M, if_variant=1, hermite_exact=exact)
        o.set_state(z, g)
        o.step(tend / n, n)
        return o.get_state()[1].ravel()

    ref = run(1, 256)
    e = [np.linalg.norm(run(1, n) - ref) for n in (8, 16, 32)]
    assert 1.9 < math.log2(e[0] / e[1]) < 2.1 and 1.9 < math.log2(e[1] / e[2]) < 2.1, e
    # both steppers converge to the same solution: their difference shrinks like dt^2
    d = [np.linalg.norm(run(1, n) - run(0, n)) for n in (16, 32)]
    assert 1.8 < math.log2(d[0] / d[1]) < 2.2 and d[1] < 1e-4 * np.linalg.norm(ref)
    # two species: the second one runs with the opposite sign (conjugate propagator)
    gp = synth.random_g(nx, ny, nz, 2, seed=7, total=0.05, nperp_hi=3.0)
    gm = synth.random_g(nx, ny, nz, 2, seed=8, total=0.05, nperp_hi=3.0)
    both = Oracle(nx, ny, nz, M=2, nspecies=2, hermite_exact=1); both.set_state(z, np.concatenate([gp, gm]))
    op = Oracle(nx, ny, nz, M=2, g_sign=+1, hermite_exact=1); op.set_state(z, gp)
    om = Oracle(nx, ny, nz, M=2, g_sign=-1, hermite_exact=1); om.set_state(z, gm)
    for o in (both, op, om):
        o.step(1e-2, 3)
    assert np.array_equal(both.get_state()[1][:2], op.get_state()[1]) and np.array_equal(both.get_state()[1][2:], om.get_state()[1])


# ---- P22: truncation monitor E_M / E_total (section 3.5; Q32) -------------------------------------
def test_p22_truncation_ratio_closed_form():
    """g_m = a_m cos(x + z) for every m, xi+ = cos(x), xi- = 0: |g_hat| = a_m/2 at two modes => 1/2 sum_k |g_m|^2 = a_m^2/4;
    E_A = 1/4 k^2 |xi+|^2 summed over the two modes (+-1,0,0) with |xi_hat| = 1/2 => 1/8."""
    nx, ny, nz, M = 8, 8, 8, 4
    a = np.array([1.0, 0.5, 0.25, 0.03])
    Z, Y, X = _grid(nx, ny, nz)
    zeta = np.stack([_half(np.cos(X)), _half(0 * X)])
    g = np.stack([_half(am * np.cos(X + Z)) for am in a])
    o = Oracle(nx, ny, nz, M=M)
    o.set_state(zeta, g)
    want = (a[-1] ** 2 / 4) / (1.0 / 8 + (a ** 2).sum() / 4)
    assert abs(o.truncation_ratio() - want) <= 1e-15
    # two species: the last moment of EACH species counts
    o2 = Oracle(nx, ny, nz, M=2, nspecies=2)
    o2.set_state(zeta, g)                      # g+ = (a0, a1), g- = (a2, a3)
    want2 = ((a[1] ** 2 + a[3] ** 2) / 4) / (1.0 / 8 + (a ** 2).sum() / 4)
    assert abs(o2.truncation_ratio() - want2) <= 1e-15
