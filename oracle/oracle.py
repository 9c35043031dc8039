"""ctypes front end of the CPU oracle (oracle/wave2d_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It never touches the CUDA path and the CUDA path never touches it.

The arithmetic lives in the C file; this wrapper only marshals numpy arrays (fp64, C-contiguous,
interior points, shape (n2, n1) with x fastest -- SURVEY.md 8b) and builds the shared object with
gcc when it is missing or older than its source.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "wave2d_oracle.c")
# WAVE2D_ORACLE_SANITIZE=1: a separate ASan + UBSan build (run python with LD_PRELOAD=$(gcc -print-file-name=libasan.so))
_SANITIZE = os.environ.get("WAVE2D_ORACLE_SANITIZE") == "1"
_LIB = os.path.join(_HERE, "liboracle_wave2d_san.so" if _SANITIZE else "liboracle_wave2d.so")
_lock = threading.Lock()
_lib = None

_dp = C.POINTER(C.c_double)


def build(force: bool = False) -> str:
    """Compile oracle/wave2d_oracle.c -> oracle/liboracle_wave2d.so (gcc -O2 -fopenmp)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        flags = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-omit-frame-pointer"] if _SANITIZE else ["-O2"]
        subprocess.check_call(
            ["gcc"] + flags + ["-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def lib() -> C.CDLL:
    global _lib
    with _lock:
        if _lib is None:
            L = C.CDLL(build())
            L.oracle_thomas.argtypes = [C.c_int, _dp, _dp, _dp, _dp, _dp, _dp, _dp]
            L.oracle_thomas.restype = None
            L.oracle_half_step.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                           C.c_double, _dp, _dp, _dp, _dp]
            L.oracle_half_step.restype = None
            L.oracle_factored_step.argtypes = [C.c_int, C.c_int] + [C.c_double] * 5 + [_dp, _dp, _dp, _dp]
            L.oracle_factored_step.restype = None
            L.oracle_wave2d_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_double,
                                               C.c_double, C.c_int]
            L.oracle_wave2d_destroy.argtypes = [C.c_void_p]
            L.oracle_wave2d_destroy.restype = None
            L.oracle_wave2d_set_option.argtypes = [C.c_void_p, C.c_char_p, C.c_double]
            L.oracle_wave2d_set_initial.argtypes = [C.c_void_p, _dp, _dp, C.c_long]
            L.oracle_wave2d_set_speed.argtypes = [C.c_void_p, _dp, C.c_int]
            L.oracle_wave2d_set_source.argtypes = [C.c_void_p, _dp, C.c_long, _dp, C.c_int]
            L.oracle_wave2d_set_speed_field.argtypes = [C.c_void_p, _dp, C.c_long]
            L.oracle_half_step_var.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                               C.c_double, _dp, _dp, _dp, _dp, _dp]
            L.oracle_half_step_var.restype = None
            L.oracle_wave2d_run.argtypes = [C.c_void_p, C.c_int]
            L.oracle_wave2d_get.argtypes = [C.c_void_p, _dp, C.c_long]
            L.oracle_wave2d_get_prev.argtypes = [C.c_void_p, _dp, C.c_long]
            L.oracle_wave2d_steps_done.argtypes = [C.c_void_p, C.POINTER(C.c_int)]
            L.oracle_num_threads.restype = C.c_int
            _lib = L
    return _lib


def _f64(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None and a.shape != tuple(shape):
        raise ValueError(f"expected shape {tuple(shape)}, got {a.shape}")
    return a


def _p(a):
    return a.ctypes.data_as(_dp) if a is not None else None


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def thomas(a, b, c, f) -> np.ndarray:
    """Solve a[p] x[p-1] + b[p] x[p] + c[p] x[p+1] = f[p] (oracle_thomas)."""
    a, b, c, f = (_f64(v) for v in (a, b, c, f))
    n = f.shape[0]
    x = np.empty(n)
    cp = np.empty(n)
    fp = np.empty(n)
    lib().oracle_thomas(n, _p(a), _p(b), _p(c), _p(f), _p(x), _p(cp), _p(fp))
    return x


def half_step(direction: int, ap: float, am: float, gamma: float, q: float, w_prev, w_cur, s=None) -> np.ndarray:
    """One half-step (eq (2.11) for direction 0, (2.12) for direction 1); arrays of shape (n2, n1)."""
    w_prev = _f64(w_prev)
    w_cur = _f64(w_cur, w_prev.shape)
    s = _f64(s, w_prev.shape) if s is not None else None
    n2, n1 = w_prev.shape
    out = np.empty_like(w_prev)
    lib().oracle_half_step(n1, n2, int(direction), ap, am, gamma, q, _p(w_prev), _p(w_cur), _p(s), _p(out))
    return out


def half_step_var(direction: int, ap: float, am: float, gamma: float, q: float, cs, w_prev, w_cur, s=None) -> np.ndarray:
    """One half-step with the spatial speed factor cs (oracle_half_step_var); arrays of shape (n2, n1)."""
    w_prev = _f64(w_prev)
    w_cur = _f64(w_cur, w_prev.shape)
    cs = _f64(cs, w_prev.shape)
    s = _f64(s, w_prev.shape) if s is not None else None
    n2, n1 = w_prev.shape
    out = np.empty_like(w_prev)
    lib().oracle_half_step_var(n1, n2, int(direction), ap, am, gamma, q, _p(cs), _p(w_prev), _p(w_cur), _p(s), _p(out))
    return out


def factored_step(axp, axm, ayp, aym, q, u_prev, u_cur, s=None) -> np.ndarray:
    """One step k -> k+1 of the factorised unsplit scheme (2.8) (oracle_factored_step); arrays (n2, n1)."""
    u_prev = _f64(u_prev)
    u_cur = _f64(u_cur, u_prev.shape)
    s = _f64(s, u_prev.shape) if s is not None else None
    n2, n1 = u_prev.shape
    out = np.empty_like(u_prev)
    lib().oracle_factored_step(n1, n2, axp, axm, ayp, aym, q, _p(u_prev), _p(u_cur), _p(s), _p(out))
    return out


class OracleError(RuntimeError):
    pass


def _check(st: int, what: str):
    if st != 0:
        raise OracleError(f"{what} failed with status {st}")


class Wave2DOracle:
    """Handle API mirroring paper_2006_10142_b200.Wave2D (host, fp64)."""

    def __init__(self, N1: int, N2: int, l: float, tau: float, M: int):
        self._h = C.c_void_p()
        _check(lib().oracle_wave2d_create(C.byref(self._h), N1, N2, l, tau, M), "oracle_wave2d_create")
        self.N1, self.N2, self.n1, self.n2, self.M = N1, N2, N1 - 1, N2 - 1, M
        self.l, self.tau = l, tau

    def close(self):
        if self._h:
            lib().oracle_wave2d_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_option(self, name: str, value: float):
        _check(lib().oracle_wave2d_set_option(self._h, name.encode(), float(value)), "set_option")

    def set_initial(self, phi, psi=None):
        phi = _f64(phi, (self.n2, self.n1))
        psi = _f64(psi, (self.n2, self.n1)) if psi is not None else None
        _check(lib().oracle_wave2d_set_initial(self._h, _p(phi), _p(psi), self.n1), "set_initial")

    def set_speed(self, c_half):
        c_half = _f64(np.atleast_1d(c_half))
        _check(lib().oracle_wave2d_set_speed(self._h, _p(c_half), c_half.shape[0]), "set_speed")

    def set_speed_field(self, cs):
        if cs is None:
            _check(lib().oracle_wave2d_set_speed_field(self._h, None, 0), "set_speed_field")
            return
        cs = _f64(cs, (self.n2, self.n1))
        _check(lib().oracle_wave2d_set_speed_field(self._h, _p(cs), self.n1), "set_speed_field")

    def set_source(self, s, g_half=None):
        if s is None:
            _check(lib().oracle_wave2d_set_source(self._h, None, 0, None, 0), "set_source")
            return
        s = _f64(s, (self.n2, self.n1))
        g = _f64(g_half) if g_half is not None else None
        _check(lib().oracle_wave2d_set_source(self._h, _p(s), self.n1, _p(g), 0 if g is None else g.shape[0]),
               "set_source")

    def run(self, steps: int):
        _check(lib().oracle_wave2d_run(self._h, int(steps)), "run")

    def get(self) -> np.ndarray:
        out = np.empty((self.n2, self.n1))
        _check(lib().oracle_wave2d_get(self._h, _p(out), self.n1), "get")
        return out

    def get_prev(self) -> np.ndarray:
        out = np.empty((self.n2, self.n1))
        _check(lib().oracle_wave2d_get_prev(self._h, _p(out), self.n1), "get_prev")
        return out

    def steps_done(self) -> int:
        k = C.c_int()
        _check(lib().oracle_wave2d_steps_done(self._h, C.byref(k)), "steps_done")
        return k.value


def solve(N1, N2, l, tau, M, phi, psi=None, c_half=None, s=None, g_half=None, steps=None,
          gamma=None, kappa=None, scheme=0, cs=None, sigma=None, start=None) -> np.ndarray:
    """Convenience: advance to time level `steps` (default M) and return u^steps.
    scheme 1 (factorised (2.8)): set_initial already stands at level 1, so steps - 1 solves are run."""
    o = Wave2DOracle(N1, N2, l, tau, M)
    try:
        if scheme:
            o.set_option("scheme", scheme)
        if gamma is not None:
            o.set_option("gamma", gamma)
        if kappa is not None:
            o.set_option("kappa", kappa)
        if sigma is not None:
            o.set_option("sigma", sigma)
        if start is not None:
            o.set_option("start", start)
        if c_half is not None:
            o.set_speed(c_half)
        if cs is not None:
            o.set_speed_field(cs)
        if s is not None:
            o.set_source(s, g_half)
        o.set_initial(phi, psi)
        o.run((M if steps is None else steps) - o.steps_done())
        return o.get()
    finally:
        o.close()
