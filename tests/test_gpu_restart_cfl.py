"""-m gpu: exact restart through the raw-state entry points and the CFL-step guards."""
import numpy as np
import pytest

from paper_2511_21891_b200 import synth
from paper_2511_21891_b200.workloads import rel_l2

pytestmark = pytest.mark.gpu


def test_restart_is_bit_exact_with_forcing_and_matches_oracle():
    from oracle import Oracle
    from paper_2511_21891_b200.gandalf import Gandalf
    shape, M, dt = (32, 16, 8), 3, 2e-3
    kw = dict(M=M, force_eps=0.7, seed=99, force_g_amp=0.2, force_g_nz=1, nu_coll=0.3, p=2.0, eta=0.2, r=2, eta_normalized=1)
    z = synth.dense_random(*shape, 2, seed=61, decay=2.5)
    gm = synth.dense_random(*shape, M, seed=62, decay=2.5)
    a = Gandalf(*shape, **kw); a.set_state(z, gm); a.step(dt, 6)
    b = Gandalf(*shape, **kw); b.set_state(z, gm); b.step(dt, 3)
    raw = b.get_state_raw()
    t, step, _ = b.time()
    assert raw.size == b.state_raw_doubles() and step == 3
    c = Gandalf(*shape, **kw)
    c.set_state_raw(raw); c.set_time(t, step); c.step(dt, 3)
    assert np.array_equal(c.get_state_raw(), a.get_state_raw())
    assert c.time()[:2] == a.time()[:2]
    hc, ha = c.energy_history(), a.energy_history()
    assert hc.shape == (3, 7) and np.array_equal(hc, ha[3:])            # the history restarts at the resumed step
    # a resumed run without set_time replays the forcing from counter 0: different
    d = Gandalf(*shape, **kw)
    d.set_state_raw(raw); d.step(dt, 3)
    assert not np.array_equal(d.get_state_raw(), a.get_state_raw())
    # the same resumed trajectory on the oracle
    o = Oracle(*shape, **kw); o.set_state(z, gm); o.step(dt, 6)
    zo, go = o.get_state(); zc, gc = c.get_state()
    assert rel_l2(zc, zo) <= 1e-10 and rel_l2(gc, go) <= 1e-10
    # device-pointer flavour of the raw entry points
    import torch
    rd = b.get_state_raw(device=True)
    assert np.array_equal(rd.cpu().numpy(), raw)
    e = Gandalf(*shape, **kw)
    e.set_state_raw(rd); e.set_time(t, step); e.step(dt, 3)
    torch.cuda.synchronize()
    assert np.array_equal(e.get_state_raw(), a.get_state_raw())


def test_cfl_zero_flow_leaves_state_and_reports():
    from paper_2511_21891_b200.gandalf import Gandalf, GandalfError, ERR_CFL
    shape, M = (16, 16, 8), 2
    gm = synth.dense_random(*shape, M, seed=3)
    z0 = np.zeros((2, shape[2], shape[1], shape[0] // 2 + 1), dtype=np.complex128)
    g = Gandalf(*shape, M=M)
    g.set_state(z0, gm)
    before = g.get_state_raw().copy()
    g.step(0.0, 3)                                    # Eq. 16 with max|grad Phi| = 0 and no dt_max
    with pytest.raises(GandalfError) as ei:
        g.time()
    assert ei.value.code == ERR_CFL
    with pytest.raises(GandalfError):
        g.energy()
    assert np.array_equal(g.get_state_raw(), before)  # the state survived
    g.set_state(z0, gm)                               # set_state clears the flag
    g.step(1e-3, 1)
    assert g.time()[1] == 1


def test_cfl_error_is_cleared_by_a_raw_restart():
    """The sticky Eq. 16 flag belongs to the state that had no flow: loading another state the restart way
    (set_state_raw + set_time) must clear it, and the run then continues like a context that never saw the error."""
    from paper_2511_21891_b200.gandalf import Gandalf, GandalfError, ERR_CFL
    shape, M = (16, 16, 8), 2
    gm = synth.dense_random(*shape, M, seed=5, decay=2.5)
    z = synth.dense_random(*shape, 2, seed=6, decay=2.5)
    z0 = np.zeros_like(z)
    good = Gandalf(*shape, M=M)
    good.set_state(z, gm)
    good.step(-1.0, 2)
    raw, (t, step, _) = good.get_state_raw(), good.time()
    g = Gandalf(*shape, M=M)
    g.set_state(z0, gm)
    g.step(-1.0, 2)                                   # no flow, no dt_max
    with pytest.raises(GandalfError) as ei:
        g.time()
    assert ei.value.code == ERR_CFL
    g.set_state_raw(raw)
    g.set_time(t, step)
    assert g.time()[:2] == (t, step)                  # no error any more
    g.step(-1.0, 3); good.step(-1.0, 3)
    assert g.time() == good.time()
    assert np.array_equal(g.get_state_raw(), good.get_state_raw())
    # set_state_raw alone clears it too
    h = Gandalf(*shape, M=M)
    h.set_state(z0, gm)
    h.step(-1.0, 1)
    with pytest.raises(GandalfError):
        h.time()
    h.set_state_raw(raw)
    h.step(-1.0, 1)
    assert h.time()[1] == 2 and h.time()[2] > 0       # the no-op step was counted (documented), the new one took a real dt


def test_cfl_dt_max_matches_oracle():
    from oracle import Oracle
    from paper_2511_21891_b200.gandalf import Gandalf
    shape, M = (16, 16, 8), 2
    gm = synth.dense_random(*shape, M, seed=3, decay=2.5)
    z0 = np.zeros((2, shape[2], shape[1], shape[0] // 2 + 1), dtype=np.complex128)
    kw = dict(M=M, dt_max=4e-3)
    o, g = Oracle(*shape, **kw), Gandalf(*shape, **kw)
    o.set_state(z0, gm); g.set_state(z0, gm)
    o.step(0.0, 4); g.step(0.0, 4)                    # no flow: every step takes dt_max
    assert abs(g.time()[0] - 1.6e-2) <= 1e-15 and abs(o.time()[0] - g.time()[0]) <= 1e-15
    assert rel_l2(g.get_state()[1], o.get_state()[1]) <= 1e-12
    # with a flow: the cap binds only when Eq. 16 would exceed it
    z = synth.dense_random(*shape, 2, seed=4, decay=2.5)
    for cap in (1e-4, 10.0):
        kw = dict(M=M, dt_max=cap)
        o, g = Oracle(*shape, **kw), Gandalf(*shape, **kw)
        o.set_state(z, gm); g.set_state(z, gm)
        o.step(-1.0, 3); g.step(-1.0, 3)
        assert abs(g.time()[2] - o.time()[2]) <= 1e-12 * o.time()[2]
        assert (g.time()[2] == cap) == (cap < 1.0)
        assert rel_l2(g.get_state()[0], o.get_state()[0]) <= 1e-10
