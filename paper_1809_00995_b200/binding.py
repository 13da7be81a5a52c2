"""Thin ctypes binding of libahs (include/ahs.h): same names, argument marshalling only.

Every step of the hot path runs inside the CUDA kernels of csrc/; this module never computes anything of the
method.  There is no CPU fallback: if libahs.so cannot be loaded, or no CUDA device is present, the calls
raise.  PyTorch, when available, supplies the device buffer and the CUDA stream (so that torch.cuda.Event
timings see the kernels); without torch the library allocates with cudaMalloc on the default stream.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

AHS_OK, AHS_ERR_INVALID_ARG, AHS_ERR_OOM, AHS_ERR_CUDA, AHS_ERR_NONFINITE, AHS_ERR_STATE = 0, -1, -2, -3, -4, -5
AHS_F32, AHS_F64 = 0, 1
AHS_IC_RANDOM_PHASE, AHS_IC_GAUSSIAN, AHS_IC_NONE = 0, 1, 2
AHS_KERNEL_AUTO, AHS_KERNEL_GENERIC, AHS_KERNEL_MARCH = 0, 1, 2
AHS_OPT_STAGING, AHS_OPT_STEP_CHUNKS, AHS_OPT_DIAG_CHUNKS, AHS_OPT_DIAG_TRIG, AHS_OPT_STEP_PDL = 0, 1, 2, 3, 4
AHS_STAGING_TENSOR, AHS_STAGING_ROWS = 0, 1
AHS_TRIG_HARDWARE, AHS_TRIG_POLYNOMIAL = 0, 1
AHS_EXCHANGE_STORES, AHS_EXCHANGE_COPIES = 0, 1

FIELD_NAMES = ("phi_re", "phi_im", "pi_re", "pi_im", "theta_0", "theta_1", "theta_2", "eps_0", "eps_1", "eps_2")

# every symbol include/ahs.h declares (tests/test_abi.py checks the header against this list and the .so)
SYMBOLS = (
    "ahs_required_bytes", "ahs_create", "ahs_create_ex", "ahs_step", "ahs_diagnostics", "ahs_diagnostics_ex",
    "ahs_diagnostics_launch", "ahs_diagnostics_fetch", "ahs_get_fields", "ahs_set_fields", "ahs_get_fields_native",
    "ahs_set_fields_native", "ahs_set_fields_native_async", "ahs_field_device_ptr", "ahs_get_state", "ahs_kernel_kind", "ahs_set_option", "ahs_set_s_schedule", "ahs_coefficients",
    "ahs_synchronize", "ahs_destroy", "ahs_last_error", "ahs_version",
    "ahs_group_create", "ahs_group_step", "ahs_group_diagnostics", "ahs_group_get_fields_native", "ahs_group_set_fields_native",
    "ahs_group_synchronize", "ahs_group_slab_count", "ahs_group_slab", "ahs_group_destroy",
    "ahs_diagnostics_static", "ahs_slab_layout", "ahs_group_set_exchange", "ahs_group_exchange_faces",
)
AHS_STATIC_MAX_RECORDS, AHS_STATIC_MAX_N, AHS_STATIC_SCRATCH_BYTES = 4736, 2048, 96 * (4736 + 1) + 160


class ahs_params(C.Structure):
    _fields_ = [("N", C.c_int32), ("precision", C.c_int32), ("ic_kind", C.c_int32), ("kernel", C.c_int32),
                ("dx", C.c_double), ("dt", C.c_double), ("lambda_", C.c_double), ("e", C.c_double),
                ("sigma", C.c_double), ("m", C.c_double), ("s", C.c_double), ("tau0", C.c_double),
                ("tau_ref", C.c_double), ("seed", C.c_uint64), ("device_buffer", C.c_void_p),
                ("device_buffer_bytes", C.c_size_t), ("stream", C.c_void_p), ("c_B", C.c_double), ("c_E", C.c_double)]


class ahs_diag(C.Structure):
    _fields_ = [("step", C.c_int64), ("tau", C.c_double), ("n_pierced", C.c_uint64), ("sum_abs_w", C.c_uint64),
                ("L", C.c_double), ("xi", C.c_double), ("v2_num", C.c_double), ("v2_den", C.c_double),
                ("v2", C.c_double), ("mean_lagrangian", C.c_double), ("gauss_max", C.c_double),
                ("gauss_rhs_rms", C.c_double), ("nonfinite", C.c_int32), ("reserved", C.c_int32),
                ("v2v_num", C.c_double), ("v2v_den", C.c_double), ("v2_V", C.c_double), ("xi_L", C.c_double),
                ("eos_num", C.c_double), ("eos_den", C.c_double), ("v2_omega", C.c_double)]


class AhsError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libahs error %d: %s" % (code, msg))
        self.code = code


_lib = None


def load(path: str | None = None):
    """dlopen libahs.so (building it in-tree with nvcc if it is missing or stale) and declare the prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    path = path or os.environ.get("AHS_LIBRARY") or _build.build_library()   # AHS_LIBRARY: an already built libahs.so
    lib = C.CDLL(path)
    vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    lib.ahs_required_bytes.argtypes = [i32, i32]; lib.ahs_required_bytes.restype = C.c_size_t
    lib.ahs_create.argtypes = [i32] + [dbl] * 8 + [C.c_uint64]; lib.ahs_create.restype = vp
    lib.ahs_create_ex.argtypes = [C.POINTER(ahs_params)]; lib.ahs_create_ex.restype = vp
    lib.ahs_step.argtypes = [vp, i32]; lib.ahs_step.restype = i32
    lib.ahs_diagnostics.argtypes = [vp] + [C.POINTER(dbl)] * 3; lib.ahs_diagnostics.restype = i32
    lib.ahs_diagnostics_ex.argtypes = [vp, C.POINTER(ahs_diag)]; lib.ahs_diagnostics_ex.restype = i32
    lib.ahs_diagnostics_launch.argtypes = [vp]; lib.ahs_diagnostics_launch.restype = i32
    lib.ahs_diagnostics_fetch.argtypes = [vp, C.POINTER(ahs_diag)]; lib.ahs_diagnostics_fetch.restype = i32
    lib.ahs_get_fields.argtypes = [vp, vp]; lib.ahs_get_fields.restype = i32
    lib.ahs_set_fields.argtypes = [vp, vp, i64]; lib.ahs_set_fields.restype = i32
    lib.ahs_get_fields_native.argtypes = [vp, vp]; lib.ahs_get_fields_native.restype = i32
    lib.ahs_set_fields_native.argtypes = [vp, vp, i64]; lib.ahs_set_fields_native.restype = i32
    lib.ahs_set_fields_native_async.argtypes = [vp, vp, i64]; lib.ahs_set_fields_native_async.restype = i32
    lib.ahs_field_device_ptr.argtypes = [vp, i32, C.POINTER(vp)]; lib.ahs_field_device_ptr.restype = i32
    lib.ahs_get_state.argtypes = [vp, C.POINTER(i64), C.POINTER(dbl), C.POINTER(i64)]; lib.ahs_get_state.restype = i32
    lib.ahs_kernel_kind.argtypes = [vp]; lib.ahs_kernel_kind.restype = i32
    lib.ahs_set_option.argtypes = [vp, i32, i32]; lib.ahs_set_option.restype = i32
    lib.ahs_set_s_schedule.argtypes = [vp, i32, C.POINTER(dbl), C.POINTER(dbl)]; lib.ahs_set_s_schedule.restype = i32
    lib.ahs_coefficients.argtypes = [vp, i64, C.POINTER(dbl)]; lib.ahs_coefficients.restype = i32
    lib.ahs_synchronize.argtypes = [vp]; lib.ahs_synchronize.restype = i32
    lib.ahs_destroy.argtypes = [vp]; lib.ahs_destroy.restype = i32
    lib.ahs_last_error.argtypes = []; lib.ahs_last_error.restype = C.c_char_p
    lib.ahs_version.argtypes = []; lib.ahs_version.restype = C.c_char_p
    lib.ahs_group_create.argtypes = [C.POINTER(ahs_params), i32, C.POINTER(i32)]; lib.ahs_group_create.restype = vp
    lib.ahs_group_step.argtypes = [vp, i32]; lib.ahs_group_step.restype = i32
    lib.ahs_group_diagnostics.argtypes = [vp, C.POINTER(ahs_diag)]; lib.ahs_group_diagnostics.restype = i32
    lib.ahs_group_get_fields_native.argtypes = [vp, vp]; lib.ahs_group_get_fields_native.restype = i32
    lib.ahs_group_set_fields_native.argtypes = [vp, vp, i64]; lib.ahs_group_set_fields_native.restype = i32
    lib.ahs_group_synchronize.argtypes = [vp]; lib.ahs_group_synchronize.restype = i32
    lib.ahs_group_slab_count.argtypes = [vp]; lib.ahs_group_slab_count.restype = i32
    lib.ahs_group_slab.argtypes = [vp, i32]; lib.ahs_group_slab.restype = vp
    lib.ahs_group_destroy.argtypes = [vp]; lib.ahs_group_destroy.restype = i32
    lib.ahs_group_set_exchange.argtypes = [vp, i32]; lib.ahs_group_set_exchange.restype = i32
    lib.ahs_group_exchange_faces.argtypes = [vp, C.POINTER(i32)]; lib.ahs_group_exchange_faces.restype = i32
    lib.ahs_slab_layout.argtypes = [i32, i32, i32, C.POINTER(i32)]; lib.ahs_slab_layout.restype = i32
    lib.ahs_diagnostics_static.argtypes = [C.POINTER(ahs_params), C.POINTER(vp), i64, C.POINTER(ahs_diag)]; lib.ahs_diagnostics_static.restype = i32
    _lib = lib
    return lib


def last_error() -> str:
    return load().ahs_last_error().decode()


def _check(code: int, allow=()):
    if code != AHS_OK and code not in allow:
        raise AhsError(code, last_error())
    return code


def required_bytes(N: int, precision: str | int) -> int:
    return int(load().ahs_required_bytes(N, _prec(precision)))


def _prec(precision) -> int:
    if precision in (AHS_F32, "f32", "float32", np.float32):
        return AHS_F32
    if precision in (AHS_F64, "f64", "float64", np.float64):
        return AHS_F64
    raise ValueError("precision must be 'f32' or 'f64'")


_KERNELS = {"auto": AHS_KERNEL_AUTO, "generic": AHS_KERNEL_GENERIC, "march": AHS_KERNEL_MARCH}
_ICS = {"random_phase": AHS_IC_RANDOM_PHASE, "gaussian": AHS_IC_GAUSSIAN, "none": AHS_IC_NONE}


class Simulation:
    """One ahs_sim handle.  Methods mirror the C functions one to one."""

    def __init__(self, N, dx=0.5, dt=0.1, lambda0=2.0, e0=1.0, sigma=1.0, m=1.0, s=0.0, tau0=1.0, seed=0,
                 precision="f32", ic="random_phase", tau_ref=0.0, kernel="auto", use_torch=True, c_B=0.0, c_E=0.0):
        self._h = None
        lib = load()
        self.N = int(N)
        self.precision = _prec(precision)
        self.dtype = np.float32 if self.precision == AHS_F32 else np.float64
        self.params = dict(N=self.N, dx=dx, dt=dt, lambda0=lambda0, e0=e0, sigma=sigma, m=m, s=s, tau0=tau0,
                           tau_ref=tau_ref, seed=seed)
        p = ahs_params()
        p.N, p.precision, p.ic_kind, p.kernel = self.N, self.precision, _ICS[ic], _KERNELS[kernel]
        p.dx, p.dt, p.lambda_, p.e, p.sigma, p.m, p.s, p.tau0, p.tau_ref = dx, dt, lambda0, e0, sigma, m, s, tau0, tau_ref
        p.seed = seed
        p.c_B = c_B
        p.c_E = c_E
        self._buffer = None
        self.stream_handle = 0
        if use_torch:
            import torch
            if not torch.cuda.is_available():
                raise AhsError(AHS_ERR_CUDA, "no CUDA device (libahs has no CPU fallback)")
            need = int(lib.ahs_required_bytes(self.N, self.precision))
            if need == 0:
                raise AhsError(AHS_ERR_INVALID_ARG, "invalid N or precision")
            # device memory and stream come from PyTorch: plumbing only
            self._buffer = torch.empty(need, dtype=torch.uint8, device="cuda")
            self.stream_handle = int(torch.cuda.current_stream().cuda_stream)
            p.device_buffer = self._buffer.data_ptr()
            p.device_buffer_bytes = need
            p.stream = self.stream_handle
        h = lib.ahs_create_ex(C.byref(p))
        if not h:
            self._buffer = None
            msg = last_error()
            code = AHS_ERR_CUDA if "CUDA" in msg else (AHS_ERR_OOM if "bytes of device memory" in msg else AHS_ERR_INVALID_ARG)
            raise AhsError(code, msg)
        self._h = C.c_void_p(h)

    # -- context manager / lifetime ---------------------------------------------------------------------------------
    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()

    def destroy(self):
        if self._h is not None:
            load().ahs_destroy(self._h)
            self._h = None
            self._buffer = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    # -- the hot path ---------------------------------------------------------------------------------------------------
    def step(self, n=1):
        _check(load().ahs_step(self._h, int(n)))

    def diagnostics(self, allow_nonfinite=True) -> dict:
        d = ahs_diag()
        _check(load().ahs_diagnostics_ex(self._h, C.byref(d)), allow=(AHS_ERR_NONFINITE,) if allow_nonfinite else ())
        return {k: getattr(d, k) for k, _ in ahs_diag._fields_ if k != "reserved"}

    def diagnostics3(self):
        """The north_star call ahs_diagnostics(&L, &v2, &gauss)."""
        L, v2, g = C.c_double(), C.c_double(), C.c_double()
        _check(load().ahs_diagnostics(self._h, C.byref(L), C.byref(v2), C.byref(g)), allow=(AHS_ERR_NONFINITE,))
        return L.value, v2.value, g.value

    def diagnostics_launch(self):
        _check(load().ahs_diagnostics_launch(self._h))

    def diagnostics_fetch(self) -> dict:
        d = ahs_diag()
        _check(load().ahs_diagnostics_fetch(self._h, C.byref(d)), allow=(AHS_ERR_NONFINITE,))
        return {k: getattr(d, k) for k, _ in ahs_diag._fields_ if k != "reserved"}

    # -- state transfer ---------------------------------------------------------------------------------------------------
    def get_fields(self) -> np.ndarray:
        """Snapshot as float64 array of shape (10, N, N, N), index [field, z, y, x]."""
        out = np.empty((10, self.N, self.N, self.N), dtype=np.float64)
        _check(load().ahs_get_fields(self._h, out.ctypes.data))
        return out

    def set_fields(self, f10: np.ndarray, step: int = 0):
        f10 = np.ascontiguousarray(f10, dtype=np.float64)
        assert f10.shape == (10, self.N, self.N, self.N)
        _check(load().ahs_set_fields(self._h, f10.ctypes.data, int(step)))

    def get_fields_native(self, out=None):
        """Snapshot in the storage type into `out` (numpy array or an integer host address, e.g. pinned memory)."""
        if out is None:
            out = np.empty((10, self.N, self.N, self.N), dtype=self.dtype)
        ptr = out if isinstance(out, int) else out.ctypes.data
        _check(load().ahs_get_fields_native(self._h, ptr))
        return out

    def set_fields_native(self, src, step: int = 0, wait: bool = True):
        """Upload a snapshot in the storage type.  wait=False: ahs_set_fields_native_async (the caller keeps `src` alive and
        unchanged until a synchronising call of this handle has returned)."""
        ptr = src if isinstance(src, int) else src.ctypes.data
        lib = load()
        _check((lib.ahs_set_fields_native if wait else lib.ahs_set_fields_native_async)(self._h, ptr, int(step)))

    def field_device_ptr(self, k: int) -> int:
        p = C.c_void_p()
        _check(load().ahs_field_device_ptr(self._h, k, C.byref(p)))
        return int(p.value)

    # -- bookkeeping ---------------------------------------------------------------------------------------------------------
    def state(self):
        st, tau, nl = C.c_int64(), C.c_double(), C.c_int64()
        _check(load().ahs_get_state(self._h, C.byref(st), C.byref(tau), C.byref(nl)))
        return st.value, tau.value, nl.value

    @property
    def step_count(self):
        return self.state()[0]

    @property
    def tau(self):
        return self.state()[1]

    @property
    def kernel_launches(self):
        return self.state()[2]

    @property
    def kernel_kind(self) -> str:
        return {AHS_KERNEL_GENERIC: "generic", AHS_KERNEL_MARCH: "march"}[load().ahs_kernel_kind(self._h)]

    def set_option(self, option: int, value: int):
        _check(load().ahs_set_option(self._h, int(option), int(value)))

    def set_s_schedule(self, knots):
        """ahs_set_s_schedule: knots = ((tau_0, s_0), (tau_1, s_1), ...); () restores the constant s."""
        _check(_set_s_schedule(self._h, knots))

    def coefficients(self, n: int) -> np.ndarray:
        out = (C.c_double * 6)()
        _check(load().ahs_coefficients(self._h, int(n), out))
        return np.array(out[:], dtype=np.float64)

    def synchronize(self):
        _check(load().ahs_synchronize(self._h))


def _set_s_schedule(handle, knots):
    k = len(knots)
    t = (C.c_double * max(k, 1))(*[float(a) for a, _ in knots])
    v = (C.c_double * max(k, 1))(*[float(b) for _, b in knots])
    return load().ahs_set_s_schedule(handle, k, t, v)


class Group:
    """One lattice cut into z-slabs (ahs_group): one handle per slab on `devices` (CUDA ordinals, may repeat; None = the current
    device for all).  Methods mirror the C functions one to one."""

    def __init__(self, N, nslabs, devices=None, dx=0.5, dt=0.1, lambda0=2.0, e0=1.0, sigma=1.0, m=1.0, s=0.0, tau0=1.0, seed=0,
                 precision="f32", ic="random_phase", tau_ref=0.0, c_B=0.0, c_E=0.0):
        self._g = None
        lib = load()
        self.N, self.nslabs = int(N), int(nslabs)
        self.precision = _prec(precision)
        self.dtype = np.float32 if self.precision == AHS_F32 else np.float64
        p = ahs_params()
        p.N, p.precision, p.ic_kind, p.kernel = self.N, self.precision, _ICS[ic], AHS_KERNEL_AUTO
        p.dx, p.dt, p.lambda_, p.e, p.sigma, p.m, p.s, p.tau0, p.tau_ref = dx, dt, lambda0, e0, sigma, m, s, tau0, tau_ref
        p.seed, p.c_B, p.c_E = seed, c_B, c_E
        dev = (C.c_int32 * self.nslabs)(*[int(d) for d in devices]) if devices is not None else None
        g = lib.ahs_group_create(C.byref(p), self.nslabs, dev)
        if not g:
            msg = last_error()
            raise AhsError(AHS_ERR_CUDA if "CUDA" in msg or "device" in msg else AHS_ERR_INVALID_ARG, msg)
        self._g = C.c_void_p(g)

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()

    def destroy(self):
        if self._g is not None:
            load().ahs_group_destroy(self._g)
            self._g = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def step(self, n=1):
        _check(load().ahs_group_step(self._g, int(n)))

    def diagnostics(self, allow_nonfinite=True) -> dict:
        d = ahs_diag()
        _check(load().ahs_group_diagnostics(self._g, C.byref(d)), allow=(AHS_ERR_NONFINITE,) if allow_nonfinite else ())
        return {k: getattr(d, k) for k, _ in ahs_diag._fields_ if k != "reserved"}

    def get_fields_native(self, out=None):
        if out is None:
            out = np.empty((10, self.N, self.N, self.N), dtype=self.dtype)
        _check(load().ahs_group_get_fields_native(self._g, out if isinstance(out, int) else out.ctypes.data))
        return out

    def set_fields_native(self, src, step: int = 0):
        _check(load().ahs_group_set_fields_native(self._g, src if isinstance(src, int) else src.ctypes.data, int(step)))

    def synchronize(self):
        _check(load().ahs_group_synchronize(self._g))

    def set_exchange(self, mode: int):
        """ahs_group_set_exchange: AHS_EXCHANGE_STORES (the step kernel's stores where the GPUs have peer access) or AHS_EXCHANGE_COPIES."""
        _check(load().ahs_group_set_exchange(self._g, int(mode)))

    @property
    def copied_faces(self) -> int:
        n = C.c_int32()
        _check(load().ahs_group_exchange_faces(self._g, C.byref(n)))
        return n.value

    def launches_per_slab(self) -> list:
        lib, out = load(), []
        for r in range(lib.ahs_group_slab_count(self._g)):
            nl = C.c_int64()
            _check(lib.ahs_get_state(C.c_void_p(lib.ahs_group_slab(self._g, r)), None, None, C.byref(nl)))
            out.append(nl.value)
        return out

    @property
    def layout(self):
        """The slabs' extents and neighbours (slabs.Slab records)."""
        from . import slabs
        return slabs.layout(self.N, self.nslabs)

    def set_s_schedule(self, knots):
        """ahs_set_s_schedule on every slab."""
        lib = load()
        for r in range(lib.ahs_group_slab_count(self._g)):
            _check(_set_s_schedule(C.c_void_p(lib.ahs_group_slab(self._g, r)), knots))

    def set_option(self, option: int, value: int):
        """ahs_set_option on every slab."""
        lib = load()
        for r in range(lib.ahs_group_slab_count(self._g)):
            _check(lib.ahs_set_option(C.c_void_p(lib.ahs_group_slab(self._g, r)), int(option), int(value)))

    @property
    def kernel_launches(self):
        lib, tot = load(), 0
        for r in range(lib.ahs_group_slab_count(self._g)):
            nl = C.c_int64()
            _check(lib.ahs_get_state(C.c_void_p(lib.ahs_group_slab(self._g, r)), None, None, C.byref(nl)))
            tot += nl.value
        return tot


def slab_layout(N: int, nslabs: int, r: int) -> tuple:
    """ahs_slab_layout: (z_offset, nz, lo, hi, nz_alloc) of slab r -- the library's own slab rules; needs no GPU."""
    out = (C.c_int32 * 5)()
    _check(load().ahs_slab_layout(int(N), int(nslabs), int(r), out))
    return tuple(out)


def diagnostics_static(fields10, N, step, precision="f32", dx=0.5, dt=0.1, lambda0=2.0, e0=1.0, sigma=1.0, m=1.0, s=0.0, tau0=1.0,
                       tau_ref=0.0, c_B=0.0, c_E=0.0, stream=0, allow_nonfinite=True) -> dict:
    """ahs_diagnostics_static: the diagnostics of ten field arrays the caller already holds on the current device, for callers that
    cannot allocate (a run that has filled the GPU's memory, a hook inside another framework's loop where cudaMalloc would fail or
    stall the device).  The library allocates nothing: its reduction scratch is a fixed 444 KiB array inside libahs.so, one per GPU,
    shared by all calls -- so do not overlap two calls on one GPU, and make the first call on each GPU during set-up.
    fields10: ten device addresses (ints) or objects with .data_ptr() (torch tensors), order FIELD_NAMES, N^3 values each of the
    storage type.  `stream` is a cudaStream_t as an integer (0 = the default stream).  Returns the same dict as
    Simulation.diagnostics()."""
    if len(fields10) != 10:
        raise ValueError("fields10 must hold ten device pointers")
    p = ahs_params()
    p.N, p.precision = int(N), _prec(precision)
    p.dx, p.dt, p.lambda_, p.e, p.sigma, p.m, p.s, p.tau0, p.tau_ref = dx, dt, lambda0, e0, sigma, m, s, tau0, tau_ref
    p.c_B, p.c_E, p.stream = c_B, c_E, int(stream)
    ptrs = (C.c_void_p * 10)(*[int(f.data_ptr()) if hasattr(f, "data_ptr") else int(f) for f in fields10])
    d = ahs_diag()
    _check(load().ahs_diagnostics_static(C.byref(p), ptrs, int(step), C.byref(d)), allow=(AHS_ERR_NONFINITE,) if allow_nonfinite else ())
    return {k: getattr(d, k) for k, _ in ahs_diag._fields_ if k != "reserved"}


def create(N, dx, dt, lambda0, e0, sigma, m, s, tau0, seed):
    """The north_star call ahs_create(N, dx, dt, lambda, e, sigma, m, s, tau0, seed): fp32, random-phase IC,
    library-owned memory on the default stream.  Returns a raw handle (int); pair with destroy_raw()."""
    h = load().ahs_create(N, dx, dt, lambda0, e0, sigma, m, s, tau0, seed)
    if not h:
        raise AhsError(AHS_ERR_INVALID_ARG, last_error())
    return h


def destroy_raw(h):
    load().ahs_destroy(C.c_void_p(h))
