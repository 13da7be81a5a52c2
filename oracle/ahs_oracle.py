"""ctypes wrapper of oracle/ahs_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It imports nothing from paper_1809_00995_b200 and the CUDA path imports nothing from
here.  All arithmetic of the method lives in ahs_oracle.c (fp64; one thread unless set_threads); this file only
builds the shared object with gcc, marshals numpy arrays and mirrors the two C structs.

Field container ("f10"): float64 array of shape (10, N, N, N), C-contiguous, index [field, z, y, x]
in the order phi_re, phi_im, Pi_re, Pi_im, theta_0..2, eps_0..2 (theta = e0*dx*A, eps = d theta/d eta,
PAPER.md L44, L62).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, asdict

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ahs_oracle.c")
_LIB = os.path.join(_HERE, "libahs_oracle.so")

FIELD_NAMES = ("phi_re", "phi_im", "pi_re", "pi_im", "theta_0", "theta_1", "theta_2", "eps_0", "eps_1", "eps_2")
IC_RANDOM_PHASE, IC_GAUSSIAN = 0, 1


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no fast-math, no FMA contraction).  -fopenmp only marks the independent site loops
    parallel (results do not depend on the thread count); without libgomp the pragmas are ignored: one thread.
    AHS_ORACLE_SANITIZE=1 builds a second library with -fsanitize=address,undefined next to the plain one (same source, same
    arithmetic flags) and loads that instead; the process then needs the sanitizer runtimes preloaded (profiles/r7_sanitizers.md has
    the command)."""
    san = os.environ.get("AHS_ORACLE_SANITIZE", "") not in ("", "0")
    out = _LIB[:-3] + "_san.so" if san else _LIB
    if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(_SRC):
        tmp = out + ".tmp.%d" % os.getpid()
        extra = ["-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer", "-g"] if san else []
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-std=c11", "-D_GNU_SOURCE"] + extra + ["-o", tmp, _SRC, "-lm"]
        if subprocess.call(cmd[:1] + ["-fopenmp"] + cmd[1:], stderr=subprocess.DEVNULL) != 0:
            subprocess.check_call(cmd)
        os.replace(tmp, out)
    return out


class _Params(C.Structure):
    _fields_ = [("N", C.c_int32), ("q", C.c_int32), ("dx", C.c_double), ("dt", C.c_double),
                ("lambda0", C.c_double), ("e0", C.c_double), ("sigma", C.c_double), ("m", C.c_double),
                ("s", C.c_double), ("tau0", C.c_double), ("tau_ref", C.c_double), ("c_B", C.c_double), ("c_E", C.c_double),
                ("ns", C.c_int32), ("pad_", C.c_int32), ("sched_tau", C.POINTER(C.c_double)), ("sched_s", C.POINTER(C.c_double))]


class _Diag(C.Structure):
    _fields_ = [("n_pierced", C.c_uint64), ("sum_abs_w", C.c_uint64), ("L", C.c_double), ("xi", C.c_double),
                ("v2_num", C.c_double), ("v2_den", C.c_double), ("v2", C.c_double),
                ("mean_lagrangian", C.c_double), ("gauss_max", C.c_double), ("gauss_rhs_rms", C.c_double),
                ("nonfinite", C.c_int32), ("pad_", C.c_int32),
                ("v2v_num", C.c_double), ("v2v_den", C.c_double), ("v2_V", C.c_double), ("xi_L", C.c_double),
                ("eos_num", C.c_double), ("eos_den", C.c_double), ("v2_omega", C.c_double)]


@dataclass
class Params:
    """Physical and lattice parameters (PAPER.md L36 lambda,e,sigma; L51 dx,dt; L68-70 s; L224 m)."""
    N: int
    dx: float = 0.5
    dt: float = 0.1
    lambda0: float = 2.0
    e0: float = 1.0
    sigma: float = 1.0
    m: float = 1.0
    s: float = 1.0
    tau0: float = 1.0
    tau_ref: float = 0.0   # 0 => tau0
    q: int = 1
    c_B: float = 1.0
    c_E: float = 1.0      # factor on the electric term in the weight; (dt/dx)^2 = L44's "E -> e dt E" read literally (R21)
    s_schedule: tuple = ()   # ((tau_0, s_0), (tau_1, s_1), ...): piecewise-linear s(tau) (R23); empty = the constant s

    def _c(self) -> _Params:
        tref = self.tau_ref if self.tau_ref != 0.0 else self.tau0
        c = _Params(self.N, self.q, self.dx, self.dt, self.lambda0, self.e0, self.sigma, self.m,
                    self.s, self.tau0, tref, self.c_B, self.c_E)
        if self.s_schedule:
            k = len(self.s_schedule)
            c._keep = ((C.c_double * k)(*[float(t) for t, _ in self.s_schedule]), (C.c_double * k)(*[float(v) for _, v in self.s_schedule]))
            c.ns = k
            c.sched_tau = C.cast(c._keep[0], C.POINTER(C.c_double))
            c.sched_s = C.cast(c._keep[1], C.POINTER(C.c_double))
        return c


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        _lib.aho_philox4x32_10.argtypes = [C.POINTER(C.c_uint32), C.POINTER(C.c_uint32), C.POINTER(C.c_uint32)]
        _lib.aho_ic.argtypes = [C.POINTER(_Params), C.c_uint64, C.c_int32, dp]
        _lib.aho_ic_window.argtypes = [C.POINTER(_Params), C.c_uint64, C.c_int32, C.c_int64, C.c_int64, C.c_int64, C.c_int64, dp]
        _lib.aho_coeffs.argtypes = [C.POINTER(_Params), C.c_int64, dp]
        _lib.aho_step.argtypes = [C.POINTER(_Params), dp, C.c_int64, C.c_int32]
        _lib.aho_winding.argtypes = [C.POINTER(_Params), dp, C.POINTER(C.c_int32),
                                     C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
        _lib.aho_diag_compute.argtypes = [C.POINTER(_Params), dp, C.c_int64, C.POINTER(_Diag)]
        _lib.aho_site_fields.argtypes = [C.POINTER(_Params), dp, C.c_int64, dp, dp, dp]
        _lib.aho_site_fields4.argtypes = [C.POINTER(_Params), dp, C.c_int64, dp, dp, dp, dp]
        _lib.aho_site_fields6.argtypes = [C.POINTER(_Params), dp, C.c_int64, dp, dp, dp, dp, dp, dp]
        for f in ("aho_philox4x32_10", "aho_ic", "aho_ic_window", "aho_coeffs", "aho_step", "aho_winding",
                  "aho_diag_compute", "aho_site_fields", "aho_site_fields4", "aho_site_fields6"):
            getattr(_lib, f).restype = None
        _lib.aho_set_threads.argtypes = [C.c_int32]
        _lib.aho_set_threads.restype = C.c_int32
        assert _lib.aho_sizeof_params() == C.sizeof(_Params)
        assert _lib.aho_sizeof_diag() == C.sizeof(_Diag)
    return _lib


def set_threads(n: int = 0) -> int:
    """Threads for the site loops (0 = all cores online; default at load time: 1).  Results do not depend on it.
    Returns the count in effect (1 if the library was built without OpenMP)."""
    return int(lib().aho_set_threads(int(n)))


def _dptr(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _check_f10(p: Params, f10: np.ndarray):
    assert f10.shape == (10, p.N, p.N, p.N) and f10.dtype == np.float64 and f10.flags["C_CONTIGUOUS"]


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(v) & 0xFFFFFFFF for v in ctr])
    k = (C.c_uint32 * 2)(*[int(v) & 0xFFFFFFFF for v in key])
    o = (C.c_uint32 * 4)()
    lib().aho_philox4x32_10(c, k, o)
    return tuple(int(v) for v in o)


def initial_condition(p: Params, seed: int, kind: int = IC_RANDOM_PHASE) -> np.ndarray:
    f10 = np.empty((10, p.N, p.N, p.N), dtype=np.float64)
    lib().aho_ic(C.byref(p._c()), C.c_uint64(seed), kind, _dptr(f10))
    return f10


def initial_condition_window(p: Params, seed: int, n_full: int, origin, kind: int = IC_RANDOM_PHASE) -> np.ndarray:
    """IC of the p.N^3 window at `origin` = (x0, y0, z0) (periodic) of an n_full^3 lattice, as a p.N^3 container."""
    f10 = np.empty((10, p.N, p.N, p.N), dtype=np.float64)
    x0, y0, z0 = (int(v) for v in origin)
    lib().aho_ic_window(C.byref(p._c()), C.c_uint64(seed), kind, n_full, x0, y0, z0, _dptr(f10))
    return f10


def coeffs(p: Params, n: int) -> np.ndarray:
    """(c1, c2, c3, d1, d2, d3) of Eqs. 4-5 for the step n -> n+1."""
    c = np.empty(6, dtype=np.float64)
    lib().aho_coeffs(C.byref(p._c()), n, _dptr(c))
    return c


def step(p: Params, f10: np.ndarray, n0: int, nsteps: int = 1) -> np.ndarray:
    """nsteps leapfrog steps in place, starting from the snapshot after n0 steps. Returns f10."""
    _check_f10(p, f10)
    lib().aho_step(C.byref(p._c()), _dptr(f10), n0, nsteps)
    return f10


def winding(p: Params, f10: np.ndarray, want_w: bool = False):
    """(n_pierced, sum_abs_w[, W]) with W int32 of shape (3, N, N, N) for planes (0,1),(0,2),(1,2)."""
    _check_f10(p, f10)
    cnt, tot = C.c_uint64(), C.c_uint64()
    W = np.empty((3, p.N, p.N, p.N), dtype=np.int32) if want_w else None
    wp = W.ctypes.data_as(C.POINTER(C.c_int32)) if want_w else None
    lib().aho_winding(C.byref(p._c()), _dptr(f10), wp, C.byref(cnt), C.byref(tot))
    return (cnt.value, tot.value, W) if want_w else (cnt.value, tot.value)


def diagnostics(p: Params, f10: np.ndarray, n: int) -> dict:
    _check_f10(p, f10)
    d = _Diag()
    lib().aho_diag_compute(C.byref(p._c()), _dptr(f10), n, C.byref(d))
    return {k: getattr(d, k) for k, _ in _Diag._fields_ if k != "pad_"}


def site_fields(p: Params, f10: np.ndarray, n: int):
    """Per-site K = |Pi|^2, G = |D phi|^2, Lag = Eq. 2, each of shape (N, N, N)."""
    _check_f10(p, f10)
    K = np.empty((p.N,) * 3); G = np.empty((p.N,) * 3); L = np.empty((p.N,) * 3)
    lib().aho_site_fields(C.byref(p._c()), _dptr(f10), n, _dptr(K), _dptr(G), _dptr(L))
    return K, G, L


def site_fields4(p: Params, f10: np.ndarray, n: int):
    """Per-site K, G, Lag and the potential term Vp = (a^2 lambda(a)/4)(|phi|^2 - sigma^2)^2, each of shape (N, N, N)."""
    _check_f10(p, f10)
    K = np.empty((p.N,) * 3); G = np.empty((p.N,) * 3); L = np.empty((p.N,) * 3); Vp = np.empty((p.N,) * 3)
    lib().aho_site_fields4(C.byref(p._c()), _dptr(f10), n, _dptr(K), _dptr(G), _dptr(L), _dptr(Vp))
    return K, G, L, Vp


def site_fields6(p: Params, f10: np.ndarray, n: int):
    """Per-site K, G, Lag, Vp and the electric / magnetic energy densities El, Bm (unit factors), each of shape (N, N, N)."""
    _check_f10(p, f10)
    out = [np.empty((p.N,) * 3) for _ in range(6)]
    lib().aho_site_fields6(C.byref(p._c()), _dptr(f10), n, *[_dptr(a) for a in out])
    return tuple(out)


def params_dict(p: Params) -> dict:
    return asdict(p)
