"""-m gpu: the CUDA-graph launch path of gandalf_step (include/gandalf.h, gandalf_graph_mode).

A step is captured from the very launches a plain step makes and replayed; dt, time and the step number live in device memory.
The replayed path must therefore reproduce the plain path BIT FOR BIT -- state, time, energy history, forcing sequence -- and the
plain path is the one the parity tests compare with the oracle (a direct oracle check of a graph run is included)."""
import numpy as np
import pytest

from paper_2511_21891_b200 import synth
from paper_2511_21891_b200.workloads import rel_l2

pytestmark = pytest.mark.gpu

CASES = {
    "rmhd": ((32, 32, 16), dict(M=0, eta=1e-3, r=2, eta_normalized=0), 1e-3),
    "krmhd": ((32, 16, 16), dict(M=6, nu_coll=1.0, p=2.0, eta=1.0, r=2, eta_normalized=1, eta_g=1.0), 5e-4),
    "forced_cfl": ((32, 32, 8), dict(M=4, force_eps=1.0, force_nperp_min=1, force_nperp_max=2, force_nz_max=1, seed=7, cfl=0.05,
                                     force_g_amp=0.1, force_g_nz=1, eta=3.0, r=2, eta_normalized=1, nu_coll=0.5, p=2.0), 0.0),
    "exact": ((16, 16, 16), dict(M=5, hermite_exact=1, if_variant=1), 2e-3),
    "two_species": ((16, 32, 8), dict(M=3, nspecies=2, closure=1), 1e-3),
    "linear": ((16, 16, 8), dict(M=2, nonlinear=0), 1e-3),
}


def _make(shape, kw, graph):
    import torch
    from paper_2511_21891_b200.gandalf import Gandalf
    st = torch.cuda.Stream()
    g = Gandalf(*shape, stream=st.cuda_stream, **kw)
    g._keep = st
    g.graph_mode(graph)
    nf = kw.get("M", 0) * kw.get("nspecies", 1)
    z = synth.dense_random(*shape, 2, seed=11, decay=2.5)
    gm = synth.dense_random(*shape, nf, seed=12, decay=2.5) if nf else None
    g.set_state(z, gm)
    return g


@pytest.mark.parametrize("name", sorted(CASES))
def test_graph_replay_equals_plain_launches_bit_for_bit(name):
    shape, kw, dt = CASES[name]
    a, b = _make(shape, kw, True), _make(shape, kw, False)
    n0a, n0b = a.launch_count(), b.launch_count()
    for n in (7, 1, 4):                                  # capture on the first call, cached replays afterwards (also nsteps = 1)
        a.step(dt, n); b.step(dt, n)
    assert a.graph_mode() == 12 and b.graph_mode() == 0
    assert a.launch_count() - n0a == b.launch_count() - n0b
    assert np.array_equal(a.get_state_raw(), b.get_state_raw())
    assert a.time() == b.time() and a.time()[1] == 12
    ha, hb = a.energy_history(), b.energy_history()
    assert ha.shape == (12, 7) and np.array_equal(ha, hb)
    ea, eb = a.energy(), b.energy()
    assert np.array_equal(np.asarray(ea), np.asarray(eb))


def test_graph_recaptures_when_dt_or_history_buffer_changes_and_single_step_calls_are_replayed():
    shape, kw, _ = CASES["krmhd"]
    a, b = _make(shape, kw, True), _make(shape, kw, False)
    for dt, n in ((5e-4, 1), (5e-4, 1), (5e-4, 1), (1e-3, 3), (5e-4, 2)):     # second single-step call with the same dt captures
        a.step(dt, n); b.step(dt, n)
    assert a.graph_mode() == 1 + 1 + 3 + 2                # every step but the very first went through a graph
    a.step(5e-4, 4200); b.step(5e-4, 4200)               # beyond the initial 4096-record history: reallocated, graph rebuilt
    assert np.array_equal(a.get_state_raw(), b.get_state_raw())
    ha, hb = a.energy_history(), b.energy_history()
    assert ha.shape == (4208, 7) and np.array_equal(ha, hb)
    assert np.all(np.diff(ha[:, 0]) > 0)


def test_graph_run_resumed_with_set_time_continues_the_forcing_sequence():
    shape, kw, _ = CASES["forced_cfl"]
    kw = dict(kw, dt_max=1e-2)
    a = _make(shape, kw, True); a.step(0.0, 8)
    b = _make(shape, kw, True); b.step(0.0, 3)
    raw = b.get_state_raw(); t, step, _ = b.time()
    c = _make(shape, kw, True)
    c.set_state_raw(raw); c.set_time(t, step); c.step(0.0, 5)
    assert c.graph_mode() == 5
    assert np.array_equal(c.get_state_raw(), a.get_state_raw())
    assert c.time()[:2] == a.time()[:2]
    assert np.array_equal(c.energy_history(), a.energy_history()[3:])


def test_graph_run_matches_oracle():
    from oracle import Oracle
    shape, kw, _ = CASES["forced_cfl"]
    a = _make(shape, kw, True)
    a.step(0.0, 10)
    assert a.graph_mode() == 10
    o = Oracle(*shape, **kw)
    z = synth.dense_random(*shape, 2, seed=11, decay=2.5)
    gm = synth.dense_random(*shape, kw["M"], seed=12, decay=2.5)
    o.set_state(z, gm); o.step(0.0, 10)
    zo, go = o.get_state(); za, ga = a.get_state()
    assert rel_l2(za, zo) <= 1e-10 and rel_l2(ga, go) <= 1e-10
    assert abs(a.time()[0] - o.time()[0]) <= 1e-12 * abs(o.time()[0])
    assert np.allclose(a.energy_history(), o.energy_history(), rtol=1e-9, atol=0)


def test_no_graph_on_the_legacy_stream_and_with_kernel_timing():
    from paper_2511_21891_b200.gandalf import Gandalf
    shape, kw, dt = CASES["rmhd"]
    g = Gandalf(*shape, **kw)                            # stream = NULL: capture is not allowed there
    g.set_state(synth.dense_random(*shape, 2, seed=11, decay=2.5), None)
    g.step(dt, 5)
    assert g.graph_mode() == 0 and g.time()[1] == 5
    a = _make(shape, kw, True)
    a.kernel_timing(True); a.step(dt, 4)
    assert a.graph_mode() == 0
    a.kernel_timing(False); a.step(dt, 4)
    assert a.graph_mode() == 4
