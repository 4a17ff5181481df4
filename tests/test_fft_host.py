"""Host-side check of the product's FFT core (csrc/fft.cuh) -- runs without a GPU.
The lane-group algorithm is emulated lane by lane and compared with numpy.fft."""
import ctypes as C
import os
import subprocess

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def lib(tmp_path_factory):
    out = tmp_path_factory.mktemp("ffth") / "libffth.so"
    subprocess.check_call(["g++", "-O1", "-std=c++17", "-fPIC", "-shared", "-o", str(out),
                           os.path.join(HERE, "fft_host_harness.cpp")])
    return C.CDLL(str(out))


ALT = 4096          # GD_FFT_ALT: plan ID of the alternative plan of a length (fft.cuh)


@pytest.mark.parametrize("n", [2, 4, 8, 16, 32, 64, 128, 256, 512, 256 + ALT])
def test_lane_group_fft_matches_numpy(lib, n):
    pid, n = n, n % ALT
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    out = np.empty_like(x)
    P = C.POINTER(C.c_double)
    for fn in (lib.host_fft, lib.host_fft_split):       # complex exchange / split (re, im) exchange
        for d, ref in ((-1, np.fft.fft(x)), (+1, np.fft.ifft(x) * n)):
            assert fn(pid, d, x.view(np.float64).ctypes.data_as(P), out.view(np.float64).ctypes.data_as(P)) == 0
            assert np.linalg.norm(out - ref) <= 1e-14 * np.sqrt(n) * np.linalg.norm(ref)


@pytest.mark.parametrize("n", [32, 64, 128, 256, 512])
def test_scatter_is_bank_conflict_free(lib, n):
    assert lib.host_fft_scatter_conflicts(n) == 1


@pytest.mark.parametrize("pid", [256, 512, 256 + ALT])
def test_split_exchange_is_bank_conflict_free_on_a_whole_warp(lib, pid):
    """8-byte exchange of the x-pass plans: 32 lanes x 8 B = 2 wavefronts at best."""
    assert lib.host_fft_split_conflicts(pid) == 2
