"""gandalf_kperp_spectrum_noalloc: the shell spectrum (Eq. 26) for callers that cannot allocate
device memory -- an application whose own pool already holds all of the GPU's memory, or a monitoring hook that must
not cause the device-wide synchronisation of cudaMalloc / cudaFree.  It takes the caller's state and output arrays and
keeps its partial sums in a fixed 256 KB array inside the library that every call shares.

The GPU test compares it with the path that already exists (a context's gandalf_kperp_spectrum, which the parity
tests hold against the oracle) on two calls in a row.  The two calls use different states on different grids, the
larger grid first, so the second call finds the first one's partial sums still in the shared array; a third call
repeats the first.  Nothing here depends on what ran before in the process: the shared array needs no particular
contents, and the test creates its own contexts.

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here should not hide the
parity tests.
"""
import ctypes as C

import numpy as np
import pytest

from paper_2511_21891_b200 import synth

# tolerance of the existing spectrum parity test (tests/test_gpu_parity.py): 1e-10 of the largest bin
TOL_SPECTRUM = 1e-10


def _existing_path(nx, ny, nz, seed, nbins, Lx, Ly):
    """A context's own spectrum (both variants) and the raw state it was computed from, as a device tensor."""
    from paper_2511_21891_b200.gandalf import Gandalf
    g = Gandalf(nx, ny, nz, Lx=Lx, Ly=Ly)
    g.set_state(synth.dense_random(nx, ny, nz, 2, seed=seed))
    g.step(1e-3, 2)                                   # an evolved state, not just the projected input
    ref = [g.kperp_spectrum(nbins, literal) for literal in (False, True)]
    raw = g.get_state_raw(device=True)
    import torch
    torch.cuda.synchronize()                          # the context enqueued that copy on its own stream
    g.close()
    return ref, raw


@pytest.mark.gpu
def test_noalloc_spectrum_matches_the_context_path_on_consecutive_calls():
    import torch
    from paper_2511_21891_b200.gandalf import kperp_spectrum_noalloc
    cases = [dict(nx=128, ny=64, nz=16, seed=71, nbins=48, Lx=2 * np.pi, Ly=4 * np.pi),      # 43 x 43 columns, Lx != Ly
             dict(nx=32, ny=32, nz=16, seed=72, nbins=20, Lx=2 * np.pi, Ly=2 * np.pi)]       # 11 x 21 columns
    refs = [_existing_path(**c) for c in cases]
    stream = torch.cuda.Stream()
    outs = []
    with torch.cuda.stream(stream):
        for k in (0, 1, 0):                           # two calls in a row, then the first again; all on one stream
            c, (_, raw) = cases[k], refs[k]
            for literal in (False, True):
                out = torch.full((c["nbins"],), float("nan"), dtype=torch.float64, device="cuda:0")
                kperp_spectrum_noalloc(c["nx"], c["ny"], c["nz"], raw, out, literal_eq26=literal, Lx=c["Lx"], Ly=c["Ly"],
                                       device=0, stream=stream.cuda_stream)
                outs.append((k, literal, out))
    stream.synchronize()
    for k, literal, out in outs:
        ref = refs[k][0][int(literal)]
        got = out.cpu().numpy()
        assert np.isfinite(got).all() and ref.max() > 0
        assert np.abs(got - ref).max() <= TOL_SPECTRUM * ref.max(), (k, literal, np.abs(got - ref).max() / ref.max())


def test_noalloc_refuses_a_grid_beyond_its_fixed_array_before_touching_cuda():
    """512 x 512 keeps 171 x 341 = 58311 (kx, ky) columns, more than the 32768 the fixed array holds: the call must say
    so and launch nothing (the pointers below are never dereferenced; this runs on a box without a GPU)."""
    from paper_2511_21891_b200.gandalf import load_library, ERR_INVALID, NOALLOC_MAX_COLUMNS
    lib = load_library()
    msg = C.create_string_buffer(320)
    fake_in, fake_out = C.c_void_p(0x1000), C.c_void_p(0x2000)

    def call(nx, ny, nz, nbins=8, Lx=6.0, w=fake_in, o=fake_out):
        return lib.gandalf_kperp_spectrum_noalloc(0, None, nx, ny, nz, Lx, 6.0, w, nbins, 0, o, msg, len(msg))

    assert (512 // 3 + 1) * (2 * (512 // 3) + 1) > NOALLOC_MAX_COLUMNS >= (512 // 3 + 1) * (2 * (256 // 3) + 1)
    assert call(512, 512, 64) == ERR_INVALID
    assert b"58311" in msg.value and str(NOALLOC_MAX_COLUMNS).encode() in msg.value
    for bad in (dict(nx=48, ny=64, nz=16), dict(nx=64, ny=4, nz=16), dict(nx=64, ny=64, nz=1024), dict(nx=64, ny=64, nz=16, nbins=0),
                dict(nx=64, ny=64, nz=16, Lx=0.0), dict(nx=64, ny=64, nz=16, w=None), dict(nx=64, ny=64, nz=16, o=None)):
        assert call(**bad) == ERR_INVALID, bad
        assert msg.value.startswith(b"gandalf_kperp_spectrum_noalloc:")
