"""-m gpu: DENSE-spectrum parity on the SAME grid at the bench sizes, in the launch
configuration bench.py times: every retained mode of every field is non-zero, so the multi-CTA D layout (block index,
XOR swizzle, PD stride), the persistent item loops of P1/P3 and P4's field-fastest block order all carry real data.
Tolerances are north_star's: 1e-12 relative L2 per RHS evaluation, 1e-10 after steps, 1e-9 on energy histories.

The last test is the conditioning evidence for the input recipe (tolerance paragraph): on the rough
|n|^-1.5 spectrum at 512 points it evaluates the Elsasser RHS in extended precision from the convolution-sum definition
 and reports oracle-vs-exact and GPU-vs-exact side by side.
"""
import time

import numpy as np
import pytest

from paper_2511_21891_b200 import synth
from paper_2511_21891_b200.workloads import rel_l2

pytestmark = pytest.mark.gpu


def _pair(shape, prm):
    from oracle import Oracle
    from paper_2511_21891_b200.gandalf import Gandalf
    return Oracle(*shape, **prm), Gandalf(*shape, **prm)


def _rhs_err(o, g):
    dw_o, dg_o = o.rhs()
    dw_g, dg_g = g.rhs()
    ew = max(rel_l2(dw_g[a], dw_o[a]) for a in range(2))
    eg = rel_l2(dg_g, dg_o) if o.M else 0.0
    if o.M:
        ref = max(np.linalg.norm(dg_o[m]) for m in range(o.M))
        eg = max(eg, max(np.linalg.norm(dg_g[m] - dg_o[m]) for m in range(o.M)) / ref)
    nx, ny, nz = o.nx, o.ny, o.nz
    assert np.count_nonzero(dw_g[:, :, :, nx // 3 + 1:]) == 0
    assert np.count_nonzero(dw_g[:, :, ny // 3 + 1: ny - ny // 3, :]) == 0
    assert np.count_nonzero(dw_g[:, nz // 3 + 1: nz - nz // 3]) == 0
    return ew, eg


def _state_err(o, g):
    zo, go = o.get_state()
    zg, gg = g.get_state()
    return rel_l2(zg, zo), (rel_l2(gg, go) if o.M else 0.0)


def test_dense_same_grid_config4a_size_rhs_and_two_steps():
    """256x256x128, M = 4 moments, dense |n|^-3 spectrum on every half-plane mode: one RHS and two complete steps
    against Oracle(256, 256, 128)."""
    shape, M = (256, 256, 128), 4
    prm = dict(M=M, nu_coll=1.0, p=2.0, eta=1.0, r=2, eta_normalized=1, eta_g=1.0)        # config 4a's physics
    o, g = _pair(shape, prm)
    z = synth.dense_random(*shape, 2, seed=4400, decay=3.0)
    gm = synth.dense_random(*shape, M, seed=4401, decay=3.0)
    o.set_state(z, gm); g.set_state(z, gm)
    t0 = time.time()
    ew, eg = _rhs_err(o, g)
    print(f"dense 256x256x128 M=4: RHS rel L2 dw {ew:.2e} dg {eg:.2e} (oracle + GPU {time.time() - t0:.0f} s)")
    assert ew <= 1e-12 and eg <= 1e-12
    o.step(5e-4, 2); g.step(5e-4, 2)
    ez, egs = _state_err(o, g)
    print(f"dense 256x256x128 M=4: state after 2 steps rel L2 zeta {ez:.2e} g {egs:.2e}")
    assert ez <= 1e-10 and egs <= 1e-10
    ho, hg = o.energy_history(), g.energy_history()
    assert np.abs(hg[:, 1:] - ho[:, 1:]).max() <= 1e-9 * np.abs(ho[:, 1:]).max()


def test_dense_same_grid_config4a_size_two_species():
    shape, M = (256, 256, 128), 2
    o, g = _pair(shape, dict(M=M, nspecies=2))
    z = synth.dense_random(*shape, 2, seed=4410, decay=3.0)
    gm = synth.dense_random(*shape, 2 * M, seed=4411, decay=3.0)
    o.set_state(z, gm); g.set_state(z, gm)
    ew, eg = _rhs_err(o, g)
    print(f"dense 256x256x128 2 species x M=2: RHS rel L2 dw {ew:.2e} dg {eg:.2e}")
    assert ew <= 1e-12 and eg <= 1e-12


@pytest.mark.parametrize("M", [0, 2])
def test_dense_same_grid_512x512x8(M):
    """512-point transforms on x and y with many CTAs per pass (256 x-pass CTAs at nx = 512)."""
    shape = (512, 512, 8)
    o, g = _pair(shape, dict(M=M, eta=1e-3, r=2))
    z = synth.dense_random(*shape, 2, seed=5100 + M, decay=4.0)
    gm = synth.dense_random(*shape, M, seed=5200, decay=4.0) if M else None
    o.set_state(z, gm); g.set_state(z, gm)
    ew, eg = _rhs_err(o, g)
    print(f"dense 512x512x8 M={M}: RHS rel L2 dw {ew:.2e} dg {eg:.2e}")
    assert ew <= 1e-12 and eg <= 1e-12
    o.step(1e-3, 2); g.step(1e-3, 2)
    ez, egs = _state_err(o, g)
    assert ez <= 1e-10 and egs <= 1e-10


@pytest.mark.slow
def test_dense_same_grid_config4b_size_rhs():
    """512x512x256, zeta+- only (BASELINE config 4b's size): one RHS against Oracle(512, 512, 256) (about 20 GB of host
    memory and a minute of host time)."""
    shape = (512, 512, 256)
    o, g = _pair(shape, dict(M=0, eta=1e-3, r=2))
    z = synth.dense_random(*shape, 2, seed=4500, decay=4.0)
    o.set_state(z); g.set_state(z)
    ew, _ = _rhs_err(o, g)
    print(f"dense 512x512x256 M=0: RHS rel L2 dw {ew:.2e}")
    assert ew <= 1e-12


# ---- conditioning evidence: rough spectrum, 512 points, both sides against an extended-precision evaluation ------------
def _conv2(a, b):
    """2-D linear convolution of longdouble-complex arrays indexed [ky][kx] (small ky extent)."""
    out = np.zeros((a.shape[0] + b.shape[0] - 1, a.shape[1] + b.shape[1] - 1), dtype=np.clongdouble)
    for i in range(a.shape[0]):
        for j in range(b.shape[0]):
            out[i + j] += np.convolve(a[i], b[j])
    return out


def _exact_elsasser_rhs(wp, wm, nx, ny):
    """N+- of Eq. 1 on the kz = 0 plane from the convolution sum, in numpy.longdouble.  wp, wm: FULL spectra [ny][nx] of
    the vorticities (FFT order).  Returns [ny][nx] arrays (retained band only)."""
    hx, hy = nx // 3, ny // 3
    nxs = np.arange(-hx, hx + 1)
    nys = np.arange(-hy, hy + 1)
    PX, PY = np.meshgrid(nxs.astype(np.longdouble), nys.astype(np.longdouble))
    k2 = PX * PX + PY * PY

    def centred(a):
        return a[np.ix_(nys % ny, nxs % nx)].astype(np.clongdouble)

    w = [centred(wp), centred(wm)]
    with np.errstate(divide="ignore", invalid="ignore"):
        xi = [np.where(k2 > 0, -v / k2, 0) for v in w]

    def bracket(f, g):          # sum_{p+q=k} (p_y q_x - p_x q_y) f(p) g(q)
        full = _conv2(PY * f, PX * g) - _conv2(PX * f, PY * g)
        return full[2 * hy - hy: 2 * hy + hy + 1, 2 * hx - hx: 2 * hx + hx + 1]     # centre: k in the retained band
    A = bracket(xi[0], w[1]) + bracket(xi[1], w[0])
    B = bracket(xi[0], xi[1])
    Np = -0.5 * (A + k2 * B)            # -1/2 [A - lap B], lap -> -k2
    Nm = -0.5 * (A - k2 * B)
    out = []
    for N in (Np, Nm):
        full = np.zeros((ny, nx), dtype=np.clongdouble)
        full[np.ix_(nys % ny, nxs % nx)] = N
        out.append(full)
    return out


@pytest.mark.parametrize("shape", [(512, 8, 2), (8, 512, 2)])
def test_rough_spectrum_512_points_oracle_and_gpu_vs_extended_precision(shape):
    nx, ny, nz = shape
    o, g = _pair(shape, dict(M=0))
    z = synth.dense_random(nx, ny, nz, 2, seed=9000 + nx, decay=1.5)
    o.set_state(z); g.set_state(z)
    wp, wm = o.get_full(0)[0], o.get_full(1)[0]           # nz = 2: only the kz = 0 plane survives Eq. 20
    exact = _exact_elsasser_rhs(wp, wm, nx, ny)
    dw_o, _ = o.rhs()
    dw_g, _ = g.rhs()
    hxp = nx // 2 + 1
    errs = {}
    for name, dw in (("oracle", dw_o), ("gpu", dw_g)):
        e = 0.0
        for a in range(2):
            ref = exact[a][:, :hxp]
            d = dw[a][0].astype(np.clongdouble) - ref
            e = max(e, float(np.sqrt((np.abs(d) ** 2).sum()) / np.sqrt((np.abs(ref) ** 2).sum())))
        errs[name] = e
    between = max(rel_l2(dw_g[a], dw_o[a]) for a in range(2))
    print(f"rough |n|^-1.5 spectrum {shape}: oracle vs exact {errs['oracle']:.2e}, gpu vs exact {errs['gpu']:.2e}, "
          f"gpu vs oracle {between:.2e}")
    # both implementations are equally far from the exact value: the excess over 1e-12 on rough data is the conditioning
    # of the bracket (k_perp^2 B amplifies eps * max-amplitude), not an error of either side
    assert errs["gpu"] <= 5e-12 and errs["oracle"] <= 5e-12
    assert errs["gpu"] <= 3.0 * errs["oracle"] + 1e-13
