"""Thin Python binding over the C-ABI CUDA library (include/gandalf.h).  Argument marshalling only:
every step of the hot path runs in the library's own sm_100a kernels.  PyTorch supplies device
memory and streams when the caller wants device-resident arrays; numpy arrays go through the
host-pointer entry points.  There is no CPU fallback: a missing library is a hard error.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libgandalf.so")

OK, ERR_INVALID, ERR_CUDA, ERR_NONFINITE, ERR_UNSUPPORTED, ERR_CFL = 0, -1, -2, -3, -4, -5
KERNEL_CLASSES = ("z_inverse", "y_inverse_P1", "x_pass_P2", "y_forward_P3", "z_step_P4")


class GandalfParams(C.Structure):
    """Mirror of `gandalf_params` (include/gandalf.h)."""
    _fields_ = [
        ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("M", C.c_int),
        ("Lx", C.c_double), ("Ly", C.c_double), ("Lz", C.c_double), ("vA", C.c_double),
        ("eta", C.c_double), ("r", C.c_int), ("eta_normalized", C.c_int),
        ("eta_z", C.c_double), ("r_z", C.c_int),
        ("eta_g", C.c_double),
        ("nu_coll", C.c_double), ("p", C.c_double),
        ("closure", C.c_int), ("if_variant", C.c_int), ("g_sign", C.c_int), ("nonlinear", C.c_int),
        ("hermite_coeff", C.c_int),
        ("force_eps", C.c_double), ("force_nperp_min", C.c_int), ("force_nperp_max", C.c_int),
        ("force_nz_max", C.c_int),
        ("seed", C.c_ulonglong),
        ("cfl", C.c_double),
        ("force_g_amp", C.c_double), ("force_g_nz", C.c_int),
        ("nspecies", C.c_int),
        ("dt_max", C.c_double), ("hermite_exact", C.c_int),
        ("m_offset", C.c_int), ("M_global", C.c_int),
        ("device", C.c_int),
        ("stream", C.c_void_p),
    ]


class GandalfError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"gandalf error {code}: {msg}")
        self.code = code


_lib = None


def load_library():
    """dlopen libgandalf.so (built in-tree by csrc/build.py).  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2511_21891_b200.csrc.build` "
                          "(__graft_entry__.build()); there is no CPU fallback")
    lib = C.CDLL(LIB_PATH)
    V, D, I = C.c_void_p, C.c_double, C.c_int
    PD = C.POINTER(C.c_double)
    lib.gandalf_default_params.argtypes = [C.POINTER(GandalfParams)]
    lib.gandalf_create.argtypes = [C.POINTER(GandalfParams), C.POINTER(V)]
    lib.gandalf_destroy.argtypes = [V]
    lib.gandalf_set_state.argtypes = [V, V, V, I]
    lib.gandalf_get_state.argtypes = [V, V, V, I]
    lib.gandalf_state_raw_doubles.argtypes = [V, C.POINTER(C.c_longlong)]
    lib.gandalf_get_state_raw.argtypes = [V, V, I]
    lib.gandalf_set_state_raw.argtypes = [V, V, I]
    lib.gandalf_set_time.argtypes = [V, D, C.c_longlong]
    lib.gandalf_rhs.argtypes = [V, V, V, I]
    lib.gandalf_step.argtypes = [V, D, I]
    lib.gandalf_energy.argtypes = [V, PD]
    lib.gandalf_kperp_spectrum.argtypes = [V, I, I, PD]
    lib.gandalf_kperp_spectrum_noalloc.argtypes = [I, V, I, I, I, D, D, V, I, I, V, C.c_char_p, I]
    lib.gandalf_hermite_spectrum.argtypes = [V, PD]
    lib.gandalf_kpar_spectrum.argtypes = [V, I, PD]
    lib.gandalf_truncation_ratio.argtypes = [V, PD]
    lib.gandalf_step_stage.argtypes = [V, D, I]
    lib.gandalf_field_ptr.argtypes = [V, I, I, C.POINTER(V), C.POINTER(C.c_longlong)]
    lib.gandalf_halo_refresh.argtypes = [V, I]
    lib.gandalf_energy_history.argtypes = [V, I, PD, C.POINTER(I)]
    lib.gandalf_get_time.argtypes = [V, PD, C.POINTER(C.c_longlong), PD]
    lib.gandalf_transfer_bytes.argtypes = [V, C.POINTER(C.c_longlong), C.POINTER(C.c_longlong)]
    lib.gandalf_launch_count.argtypes = [V]
    lib.gandalf_launch_count.restype = C.c_longlong
    lib.gandalf_graph_mode.argtypes = [V, I, C.POINTER(C.c_longlong)]
    lib.gandalf_kernel_timing.argtypes = [V, I]
    lib.gandalf_kernel_time_ms.argtypes = [V, I, PD, C.POINTER(C.c_longlong)]
    lib.gandalf_microbench.argtypes = [I, I, PD, I]
    lib.gandalf_last_error.argtypes = [V]
    lib.gandalf_last_error.restype = C.c_char_p
    _lib = lib
    return lib


MICROBENCHES = ("fp64_fma", "fft256_lane_group", "tmem_load", "smem_load")


def microbench(which, device=0):
    """gandalf_microbench(which): four doubles (see include/gandalf.h)."""
    lib = load_library()
    out = np.zeros(4)
    rc = lib.gandalf_microbench(int(which), int(device), out.ctypes.data_as(C.POINTER(C.c_double)), 4)
    if rc != OK:
        raise GandalfError(rc, "gandalf_microbench failed")
    return out


NOALLOC_MAX_COLUMNS = 32768      # GANDALF_NOALLOC_MAX_COLUMNS of include/gandalf.h


def kperp_spectrum_noalloc(nx, ny, nz, w_raw, out, literal_eq26=False, Lx=2.0 * np.pi, Ly=2.0 * np.pi, device=0, stream=None):
    """gandalf_kperp_spectrum_noalloc: the shell spectrum of Eq. 26 without a context and without any device allocation, for
    callers that cannot allocate (all GPU memory already in their own pool, or no device-wide synchronisation allowed).
    `w_raw` (float64 CUDA tensor: w+ then w- in the get_state_raw layout; more fields may follow) and `out` (float64 CUDA
    tensor, one entry per bin, overwritten) are the caller's; the partial sums use a fixed 256 KB array inside the library that
    all calls share, so do not let two calls overlap on the GPU.  Enqueues on `stream` (a cudaStream_t value; None = legacy
    default stream) and does not synchronise.  Grids with more than NOALLOC_MAX_COLUMNS retained (kx, ky) columns raise
    GandalfError(ERR_INVALID).  Make the first call on a device at start-up, outside any stream capture."""
    import torch
    lib = load_library()
    need = 2 * 2 * (2 * (nz // 3) + 1) * (2 * (ny // 3) + 1) * (nx // 3 + 1)
    for t in (w_raw, out):
        assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and t.device.index == device
    assert w_raw.numel() >= need, (w_raw.numel(), need)
    msg = C.create_string_buffer(320)
    rc = lib.gandalf_kperp_spectrum_noalloc(int(device), C.c_void_p(int(stream) if stream else None), nx, ny, nz, float(Lx), float(Ly),
                                            C.c_void_p(w_raw.data_ptr()), int(out.numel()), int(bool(literal_eq26)),
                                            C.c_void_p(out.data_ptr()), msg, len(msg))
    if rc != OK:
        raise GandalfError(rc, msg.value.decode())
    return out


def _is_torch(x):
    return type(x).__module__.startswith("torch")


class Gandalf:
    """One solver context.  Boundary arrays: complex128, shape (fields, nz, ny, nx//2+1); zeta = the
    Elsasser potentials xi^+, xi^- (2 fields), g = Hermite moments g_0..g_{M-1}.
    numpy arrays use the host entry points; torch CUDA tensors are passed as device pointers."""

    def __init__(self, nx, ny, nz, M=0, device=0, stream=None, **kw):
        self._h = None
        lib = load_library()
        p = GandalfParams()
        lib.gandalf_default_params(C.byref(p))
        p.nx, p.ny, p.nz, p.M, p.device = nx, ny, nz, M, device
        names = {f[0] for f in GandalfParams._fields_}
        for k, v in kw.items():
            if k not in names:
                raise TypeError(f"unknown gandalf parameter {k!r}")
            setattr(p, k, v)
        if stream is not None:
            p.stream = int(stream)
        self.params = p
        # self.M = number of moment FIELDS at the boundary (2M with both species: g^+ then g^-)
        self.nx, self.ny, self.nz, self.M, self.hx = nx, ny, nz, M * max(int(p.nspecies), 1), nx // 2 + 1
        h = C.c_void_p()
        rc = lib.gandalf_create(C.byref(p), C.byref(h))
        if rc != OK:
            raise GandalfError(rc, "gandalf_create failed (invalid parameters, unsupported combination or CUDA error)")
        self._h, self._lib = h, lib

    # -- plumbing -------------------------------------------------------------------------------
    def close(self):
        if getattr(self, "_h", None):
            self._lib.gandalf_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ck(self, rc):
        if rc != OK:
            raise GandalfError(rc, self._lib.gandalf_last_error(self._h).decode())

    def _shape(self, nf):
        return (nf, self.nz, self.ny, self.hx)

    def _in_ptr(self, a, nf):
        """(pointer, on_device, keepalive) for an input array."""
        if a is None:
            return None, None, None
        if _is_torch(a):
            import torch
            assert a.is_cuda and a.dtype == torch.complex128 and a.is_contiguous() and tuple(a.shape) == self._shape(nf)
            return C.c_void_p(a.data_ptr()), 1, a
        arr = np.ascontiguousarray(a, dtype=np.complex128)
        assert arr.shape == self._shape(nf), (arr.shape, self._shape(nf))
        return C.c_void_p(arr.ctypes.data), 0, arr

    # -- API ------------------------------------------------------------------------------------
    def set_state(self, zeta_hat, g_hat=None):
        zp, dev, k1 = self._in_ptr(zeta_hat, 2)
        gp, dev2, k2 = self._in_ptr(g_hat, self.M) if self.M > 0 else (None, dev, None)
        assert dev == dev2, "zeta and g must both be host or both be device arrays"
        self._ck(self._lib.gandalf_set_state(self._h, zp, gp, dev))

    def _out(self, like_torch, nf):
        if like_torch:
            import torch
            t = torch.empty(self._shape(max(nf, 1)), dtype=torch.complex128, device=f"cuda:{self.params.device}")
            return t, C.c_void_p(t.data_ptr())
        a = np.empty(self._shape(max(nf, 1)), dtype=np.complex128)
        return a, C.c_void_p(a.ctypes.data)

    def get_state(self, device=False):
        z, zp = self._out(device, 2)
        g, gp = self._out(device, self.M)
        self._ck(self._lib.gandalf_get_state(self._h, zp, gp, int(bool(device))))
        return z, g[: self.M]

    def state_raw_doubles(self):
        n = C.c_longlong(0)
        self._ck(self._lib.gandalf_state_raw_doubles(self._h, C.byref(n)))
        return n.value

    def get_state_raw(self, device=False, out=None):
        """The evolved variables w+-, g_m on the retained modes (exact checkpoint), a flat float64 array.
        `out`: a contiguous float64 numpy array of state_raw_doubles() entries to fill instead (e.g. a view of pinned memory)."""
        n = self.state_raw_doubles()
        if out is not None:
            assert not device and isinstance(out, np.ndarray) and out.dtype == np.float64 and out.flags.c_contiguous and out.size == n
            self._ck(self._lib.gandalf_get_state_raw(self._h, C.c_void_p(out.ctypes.data), 0))
            return out
        if device:
            import torch
            t = torch.empty(n, dtype=torch.float64, device=f"cuda:{self.params.device}")
            self._ck(self._lib.gandalf_get_state_raw(self._h, C.c_void_p(t.data_ptr()), 1))
            return t
        a = np.empty(n, dtype=np.float64)
        self._ck(self._lib.gandalf_get_state_raw(self._h, C.c_void_p(a.ctypes.data), 0))
        return a

    def set_state_raw(self, raw):
        n = self.state_raw_doubles()
        if _is_torch(raw):
            import torch
            assert raw.is_cuda and raw.dtype == torch.float64 and raw.is_contiguous() and raw.numel() == n
            self._ck(self._lib.gandalf_set_state_raw(self._h, C.c_void_p(raw.data_ptr()), 1))
        else:
            a = np.ascontiguousarray(raw, dtype=np.float64)
            assert a.size == n
            self._ck(self._lib.gandalf_set_state_raw(self._h, C.c_void_p(a.ctypes.data), 0))

    def set_time(self, t, step):
        self._ck(self._lib.gandalf_set_time(self._h, float(t), int(step)))

    def rhs(self, device=False):
        dw, wp = self._out(device, 2)
        dg, gp = self._out(device, self.M)
        self._ck(self._lib.gandalf_rhs(self._h, wp, gp, int(bool(device))))
        return dw, dg[: self.M]

    def step(self, dt, nsteps=1):
        self._ck(self._lib.gandalf_step(self._h, float(dt), int(nsteps)))

    def step_stage(self, dt, stage):
        """gandalf_step_stage: stage 0 = RHS + predictor, stage 1 = midpoint RHS + corrector + ... (moment-sharded runs
        refresh their halo moments in between)."""
        self._ck(self._lib.gandalf_step_stage(self._h, float(dt), int(stage)))

    def field_tensor(self, state, field):
        """Zero-copy torch view (float64, 2 * ncomplex entries) of one field of the raw retained-mode array
        (gandalf_field_ptr): state 0 = the state, 1 = the half-step stage state; field 0, 1 = w+-, 2+j = local moment j."""
        import torch
        ptr, n = C.c_void_p(), C.c_longlong()
        self._ck(self._lib.gandalf_field_ptr(self._h, int(state), int(field), C.byref(ptr), C.byref(n)))

        class _View:       # the CUDA array interface lets torch wrap a raw device pointer without copying
            __cuda_array_interface__ = {"shape": (2 * n.value,), "typestr": "<f8", "data": (ptr.value, False), "version": 2}
        return torch.as_tensor(_View(), device=f"cuda:{self.params.device}")

    def halo_refresh(self, state):
        self._ck(self._lib.gandalf_halo_refresh(self._h, int(state)))

    def transfer_bytes(self):
        """(host -> device, device -> host) bytes moved by the host-pointer entry points so far."""
        a, b = C.c_longlong(), C.c_longlong()
        self._ck(self._lib.gandalf_transfer_bytes(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def energy(self):
        out = np.zeros(6)
        self._ck(self._lib.gandalf_energy(self._h, out.ctypes.data_as(C.POINTER(C.c_double))))
        return out

    def kperp_spectrum(self, nbins, literal_eq26=False):
        out = np.zeros(nbins)
        self._ck(self._lib.gandalf_kperp_spectrum(self._h, nbins, int(literal_eq26), out.ctypes.data_as(C.POINTER(C.c_double))))
        return out

    def hermite_spectrum(self):
        out = np.zeros(max(self.M, 1))
        self._ck(self._lib.gandalf_hermite_spectrum(self._h, out.ctypes.data_as(C.POINTER(C.c_double))))
        return out[: self.M]

    def truncation_ratio(self):
        """E_M / E_total of PAPER.md:269 (gandalf_truncation_ratio)."""
        out = C.c_double()
        self._ck(self._lib.gandalf_truncation_ratio(self._h, C.byref(out)))
        return out.value

    def kpar_spectrum(self, nbins):
        out = np.zeros(nbins)
        self._ck(self._lib.gandalf_kpar_spectrum(self._h, nbins, out.ctypes.data_as(C.POINTER(C.c_double))))
        return out

    def energy_history(self, max_records=None):
        _, nstep, _ = self.time()
        k = nstep if max_records is None else min(nstep, max_records)
        buf = np.zeros((max(k, 1), 7))
        n = C.c_int(0)
        self._ck(self._lib.gandalf_energy_history(self._h, k, buf.ctypes.data_as(C.POINTER(C.c_double)), C.byref(n)))
        return buf[: n.value].copy()

    def time(self):
        t, s, d = C.c_double(0), C.c_longlong(0), C.c_double(0)
        self._ck(self._lib.gandalf_get_time(self._h, C.byref(t), C.byref(s), C.byref(d)))
        return t.value, s.value, d.value

    def launch_count(self):
        return int(self._lib.gandalf_launch_count(self._h))

    def graph_mode(self, enable=None):
        """gandalf_graph_mode: switch the CUDA-graph launch path of step() on/off (None: query); returns the graph replays so far."""
        n = C.c_longlong(0)
        self._ck(self._lib.gandalf_graph_mode(self._h, -1 if enable is None else int(bool(enable)), C.byref(n)))
        return n.value

    def kernel_timing(self, enable=True):
        self._ck(self._lib.gandalf_kernel_timing(self._h, int(bool(enable))))

    def kernel_times(self):
        """{class name: (average ms per launch, launches)} since timing was enabled."""
        out = {}
        for i, name in enumerate(KERNEL_CLASSES):
            ms, n = C.c_double(0), C.c_longlong(0)
            self._ck(self._lib.gandalf_kernel_time_ms(self._h, i, C.byref(ms), C.byref(n)))
            out[name] = (ms.value, n.value)
        return out
