"""ctypes binding over include/wave2d.h -- argument marshalling only.

Every step of the hot path runs inside libwave2d.so's CUDA kernels.  If the library cannot be loaded
this module raises; it never falls back to a CPU implementation.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBNAME = "libwave2d.so"
_lib = None

F64, F32 = 0, 1
SOLVER_AUTO, SOLVER_EXACT, SOLVER_STREAM, SOLVER_LINE = 0, 1, 2, 3

EXPORTS = [
    "wave2d_create", "wave2d_destroy", "wave2d_set_stream", "wave2d_set_option", "wave2d_set_initial",
    "wave2d_set_state",
    "wave2d_set_speed", "wave2d_set_speed_field", "wave2d_set_source", "wave2d_run", "wave2d_get", "wave2d_get_prev",
    "wave2d_get_rows", "wave2d_set_rows", "wave2d_steps_done", "wave2d_sync", "wave2d_get_info", "wave2d_profile_sweeps", "wave2d_get_trace",
    "wave2d_host_scalars", "wave2d_host_plan", "wave2d_strerror", "wave2d_last_error",
    "wave2d_small_steps_static", "wave2d_host_decay", "wave2d_workspace_bytes", "wave2d_set_workspace",
]


class Wave2DError(RuntimeError):
    def __init__(self, status: int, what: str, detail: str = ""):
        self.status = status
        super().__init__(f"{what}: status {status}" + (f" ({detail})" if detail else ""))


def library_path() -> str:
    return os.path.join(_HERE, _LIBNAME)


def load_library() -> C.CDLL:
    """dlopen paper_2006_10142_b200/libwave2d.so (built by __graft_entry__.build() / build.py)."""
    global _lib
    if _lib is not None:
        return _lib
    path = library_path()
    if not os.path.exists(path):
        raise ImportError(f"{path} is missing: build it with `python -m paper_2006_10142_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(path)
    vp, dp, ip = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int)
    L.wave2d_create.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_double, C.c_double, C.c_int, C.c_int]
    L.wave2d_destroy.argtypes = [vp]
    L.wave2d_destroy.restype = None
    L.wave2d_set_stream.argtypes = [vp, vp]
    L.wave2d_set_option.argtypes = [vp, C.c_char_p, C.c_double]
    L.wave2d_set_initial.argtypes = [vp, vp, vp, C.c_long]
    L.wave2d_set_state.argtypes = [vp, C.c_int, vp, vp, C.c_long]
    L.wave2d_set_speed.argtypes = [vp, dp, C.c_int]
    L.wave2d_set_source.argtypes = [vp, vp, C.c_long, dp, C.c_int]
    L.wave2d_set_speed_field.argtypes = [vp, vp, C.c_long]
    L.wave2d_run.argtypes = [vp, C.c_int]
    L.wave2d_get.argtypes = [vp, vp, C.c_long]
    L.wave2d_get_prev.argtypes = [vp, vp, C.c_long]
    L.wave2d_get_rows.argtypes = [vp, C.c_int, C.c_int, C.c_int, vp, C.c_long]
    L.wave2d_set_rows.argtypes = [vp, C.c_int, C.c_int, C.c_int, vp, C.c_long]
    L.wave2d_steps_done.argtypes = [vp, ip]
    L.wave2d_sync.argtypes = [vp]
    L.wave2d_get_info.argtypes = [vp, C.c_char_p, dp]
    L.wave2d_profile_sweeps.argtypes = [vp, C.c_int, dp, dp]
    L.wave2d_get_trace.argtypes = [vp, C.c_int, vp, C.c_int, C.POINTER(C.c_int)]
    ip = C.POINTER(C.c_int)
    L.wave2d_host_scalars.argtypes = [C.c_double, C.c_double, C.c_double, C.c_double, dp, C.c_int, ip]
    L.wave2d_workspace_bytes.argtypes = [vp, C.POINTER(C.c_ulonglong)]
    L.wave2d_set_workspace.argtypes = [vp, vp, C.c_ulonglong]
    L.wave2d_host_decay.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, C.c_double, C.c_double, dp]
    L.wave2d_host_plan.argtypes = [C.c_int] * 8 + [C.c_double, ip, C.c_int, ip, ip, ip]
    L.wave2d_strerror.argtypes = [C.c_int]
    L.wave2d_strerror.restype = C.c_char_p
    L.wave2d_last_error.argtypes = [vp]
    L.wave2d_last_error.restype = C.c_char_p
    L.wave2d_small_steps_static.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int, C.c_int,
                                            vp, vp, vp, vp, C.c_long, vp, C.c_char_p, C.c_int]
    _lib = L
    return L


def _is_torch(a) -> bool:
    return type(a).__module__.startswith("torch")


class Wave2D:
    """One simulation handle (include/wave2d.h).  Arrays: numpy (host) or torch tensors (host or cuda),
    shape (n2, n1) = (N2-1, N1-1), dtype matching the handle's; a last-dimension-contiguous 2-D view
    with row stride ld >= n1 is accepted as is."""

    def __init__(self, N1: int, N2: int, l: float, tau: float, M: int, dtype: str = "f64"):
        self._L = load_library()
        self._h = C.c_void_p()
        self.dtype = dtype
        self._code = {"f64": F64, "f32": F32}[dtype]
        self._np = np.float64 if dtype == "f64" else np.float32
        self.N1, self.N2, self.n1, self.n2, self.M = N1, N2, N1 - 1, N2 - 1, M
        st = self._L.wave2d_create(C.byref(self._h), N1, N2, l, tau, M, self._code)
        if st != 0:
            raise Wave2DError(st, "wave2d_create", self._L.wave2d_strerror(st).decode())

    # -- plumbing -------------------------------------------------------------------------------
    def _check(self, st: int, what: str):
        if st != 0:
            detail = self._L.wave2d_strerror(st).decode()
            more = self._L.wave2d_last_error(self._h)
            if more:
                detail += "; " + more.decode()
            raise Wave2DError(st, what, detail)

    def _field(self, a, keep: list):
        """-> (pointer, ld) for a host/device array of shape (n2, n1)."""
        if a is None:
            return None, 0
        if _is_torch(a):
            import torch
            want = torch.float64 if self.dtype == "f64" else torch.float32
            if a.dtype != want or a.dim() != 2 or tuple(a.shape) != (self.n2, self.n1):
                raise ValueError(f"expected torch {want} tensor of shape {(self.n2, self.n1)}")
            if a.stride(1) != 1:
                a = a.contiguous()
            keep.append(a)
            return C.c_void_p(a.data_ptr()), int(a.stride(0)) if self.n2 > 1 else self.n1
        a = np.asarray(a)
        if a.shape != (self.n2, self.n1):
            raise ValueError(f"expected shape {(self.n2, self.n1)}, got {a.shape}")
        if a.dtype != self._np or a.strides[1] != a.itemsize or a.strides[0] % a.itemsize:
            a = np.ascontiguousarray(a, dtype=self._np)
        keep.append(a)
        ld = a.strides[0] // a.itemsize if self.n2 > 1 else self.n1
        return C.c_void_p(a.ctypes.data), int(ld)

    def close(self):
        if getattr(self, "_h", None):
            self._L.wave2d_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # -- the C ABI, one method per entry point -----------------------------------------------------
    def set_stream(self, stream):
        ptr = getattr(stream, "cuda_stream", stream)
        self._check(self._L.wave2d_set_stream(self._h, C.c_void_p(ptr or 0)), "wave2d_set_stream")

    def set_option(self, name: str, value: float):
        self._check(self._L.wave2d_set_option(self._h, name.encode(), float(value)), "wave2d_set_option")

    def workspace_bytes(self) -> int:
        n = C.c_ulonglong()
        self._check(self._L.wave2d_workspace_bytes(self._h, C.byref(n)), "wave2d_workspace_bytes")
        return int(n.value)

    def set_workspace(self, block):
        """Keep the time levels in `block` (a torch CUDA tensor of at least workspace_bytes() bytes, or None to return
        to handle-owned memory).  The handle holds a reference, so the block outlives it."""
        if block is None:
            self._check(self._L.wave2d_set_workspace(self._h, None, 0), "wave2d_set_workspace")
            self._workspace = None
            return
        nbytes = block.numel() * block.element_size()
        self._check(self._L.wave2d_set_workspace(self._h, C.c_void_p(block.data_ptr()), nbytes), "wave2d_set_workspace")
        self._workspace = block

    def set_initial(self, phi, psi=None):
        keep = []
        p, ld = self._field(phi, keep)
        q, ld2 = self._field(psi, keep)
        if psi is not None and ld2 != ld:
            raise ValueError("phi and psi must share one row stride")
        self._check(self._L.wave2d_set_initial(self._h, p, q, ld), "wave2d_set_initial")

    def set_state(self, k: int, u_prev_half, u):
        keep = []
        p, ld = self._field(u_prev_half, keep)
        q, ld2 = self._field(u, keep)
        if ld2 != ld:
            raise ValueError("both fields must share one row stride")
        self._check(self._L.wave2d_set_state(self._h, int(k), p, q, ld), "wave2d_set_state")

    def set_speed(self, c_half):
        c = np.ascontiguousarray(np.atleast_1d(c_half), dtype=np.float64)
        self._check(self._L.wave2d_set_speed(self._h, c.ctypes.data_as(C.POINTER(C.c_double)), c.shape[0]),
                    "wave2d_set_speed")

    def set_speed_field(self, cs):
        keep = []
        p, ld = self._field(cs, keep)
        self._check(self._L.wave2d_set_speed_field(self._h, p, ld), "wave2d_set_speed_field")

    def set_source(self, s, g_half=None):
        keep = []
        p, ld = self._field(s, keep)
        g = None if g_half is None else np.ascontiguousarray(g_half, dtype=np.float64)
        gp = None if g is None else g.ctypes.data_as(C.POINTER(C.c_double))
        self._check(self._L.wave2d_set_source(self._h, p, ld, gp, 0 if g is None else g.shape[0]),
                    "wave2d_set_source")

    def run(self, steps: int):
        self._check(self._L.wave2d_run(self._h, int(steps)), "wave2d_run")

    def _out(self, fn, what, out):
        if out is None:
            out = np.empty((self.n2, self.n1), dtype=self._np)
        keep = []
        p, ld = self._field(out, keep)
        if keep[0] is not out:
            raise ValueError("output array must have the handle's dtype and unit inner stride")
        self._check(fn(self._h, p, ld), what)
        return out

    def get(self, out=None):
        return self._out(self._L.wave2d_get, "wave2d_get", out)

    def get_prev(self, out=None):
        return self._out(self._L.wave2d_get_prev, "wave2d_get_prev", out)

    def _rows(self, a, count: int):
        """-> (pointer, ld, array) for a host/device array of `count` rows of n1 values."""
        if _is_torch(a):
            if a.dim() != 2 or tuple(a.shape) != (count, self.n1) or a.stride(1) != 1:
                raise ValueError(f"expected a torch tensor of shape {(count, self.n1)} with unit inner stride")
            return C.c_void_p(a.data_ptr()), int(a.stride(0)) if count > 1 else self.n1, a
        if a.shape != (count, self.n1) or a.dtype != self._np or a.strides[1] != a.itemsize:
            raise ValueError(f"expected a {self._np.__name__} array of shape {(count, self.n1)} with unit inner stride")
        return C.c_void_p(a.ctypes.data), int(a.strides[0] // a.itemsize) if count > 1 else self.n1, a

    def get_rows(self, level: int, j0: int, count: int, out=None):
        if out is None:
            out = np.empty((count, self.n1), dtype=self._np)
        p, ld, _ = self._rows(out, count)
        self._check(self._L.wave2d_get_rows(self._h, int(level), int(j0), int(count), p, ld), "wave2d_get_rows")
        return out

    def set_rows(self, level: int, j0: int, rows):
        if not _is_torch(rows):
            rows = np.ascontiguousarray(rows, dtype=self._np)
        count = int(rows.shape[0])
        p, ld, keep = self._rows(rows, count)
        self._check(self._L.wave2d_set_rows(self._h, int(level), int(j0), count, p, ld), "wave2d_set_rows")

    def steps_done(self) -> int:
        k = C.c_int()
        self._check(self._L.wave2d_steps_done(self._h, C.byref(k)), "wave2d_steps_done")
        return k.value

    def sync(self):
        self._check(self._L.wave2d_sync(self._h), "wave2d_sync")

    def info(self, name: str) -> float:
        v = C.c_double()
        self._check(self._L.wave2d_get_info(self._h, name.encode(), C.byref(v)), "wave2d_get_info")
        return v.value

    def trace(self, direction: int) -> np.ndarray:
        """Per-CTA records of the last launch of a direction: 16 uint64 per CTA (include/wave2d.h)."""
        cap = 4096
        buf = np.zeros((cap, 16), dtype=np.uint64)
        cnt = C.c_int()
        self._check(self._L.wave2d_get_trace(self._h, int(direction), buf.ctypes.data_as(C.c_void_p), cap,
                                             C.byref(cnt)), "wave2d_get_trace")
        return buf[:cnt.value]

    def profile_sweeps(self, steps: int):
        a, b = C.c_double(), C.c_double()
        self._check(self._L.wave2d_profile_sweeps(self._h, int(steps), C.byref(a), C.byref(b)),
                    "wave2d_profile_sweeps")
        return a.value, b.value


def from_workload(w, dtype=None, solver=None, graph=None) -> "Wave2D":
    """Create a handle and feed it a workloads.Workload (inputs converted to the handle's dtype)."""
    dt = dtype or w.dtype
    h = Wave2D(w.N1, w.N2, w.l, w.tau, w.M, dt)
    npdt = np.float64 if dt == "f64" else np.float32
    if solver is not None:
        h.set_option("solver", solver)
    if graph is not None:
        h.set_option("graph", graph)
    h.set_speed(w.c_half)
    if w.s is not None:
        h.set_source(w.s.astype(npdt, copy=False), w.g_half)
    h.set_initial(w.phi.astype(npdt, copy=False), None if w.psi is None else w.psi.astype(npdt, copy=False))
    return h


def small_steps_static(N1: int, N2: int, l: float, tau: float, c: float, steps: int, u_prev_half, u, u_out,
                       u_prev_out=None, stream=None):
    """wave2d_small_steps_static: `steps` time steps on a small grid (N1, N2 <= 257) with no allocation anywhere in
    the library -- for callers that cannot cudaMalloc (a framework's allocator owns the GPU's memory, a fixed memory
    budget, or other streams that a device-wide synchronisation would stall); the kernel's working memory is a 1.5 MiB
    array inside libwave2d.so, shared by all calls in the process (see include/wave2d.h for what that implies).

    u_prev_half, u (inputs: u^{k-1/2}, u^k) and u_out, u_prev_out (outputs: u^{k+steps}, u^{k+steps-1/2}; the second is
    optional) are torch CUDA tensors of shape (N2-1, N1-1), float64 or float32, unit inner stride and one common row
    stride; the caller creates them, this function only passes their pointers on.  Asynchronous on `stream` (default:
    torch's current stream).  Nothing is returned: the result is in u_out / u_prev_out."""
    import torch
    L = load_library()
    n1, n2 = N1 - 1, N2 - 1
    fields = [u_prev_half, u, u_out] + ([] if u_prev_out is None else [u_prev_out])
    for t in fields:
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dim() == 2 and tuple(t.shape) == (n2, n1) and
                t.stride(1) == 1 and t.dtype == u.dtype and t.stride(0) == u.stride(0)):
            raise ValueError(f"expected CUDA tensors of shape {(n2, n1)}, one dtype, unit inner stride, one row stride")
    if u.dtype not in (torch.float64, torch.float32):
        raise ValueError("dtype must be float64 or float32")
    ld = int(u.stride(0)) if n2 > 1 else n1
    if stream is None:
        stream = torch.cuda.current_stream(u.device)
    sp = getattr(stream, "cuda_stream", stream)
    err = C.create_string_buffer(512)
    with torch.cuda.device(u.device):
        st = L.wave2d_small_steps_static(int(N1), int(N2), float(l), float(tau), float(c), int(steps),
                                         F64 if u.dtype == torch.float64 else F32,
                                         C.c_void_p(u_prev_half.data_ptr()), C.c_void_p(u.data_ptr()),
                                         C.c_void_p(u_out.data_ptr()),
                                         C.c_void_p(0 if u_prev_out is None else u_prev_out.data_ptr()), ld,
                                         C.c_void_p(sp or 0), err, len(err))
    if st != 0:
        detail = L.wave2d_strerror(st).decode()
        if err.value:
            detail += "; " + err.value.decode()
        raise Wave2DError(st, "wave2d_small_steps_static", detail)


def host_scalars(gamma: float, alpha_plus: float, alpha_minus: float, q: float = 0.0) -> np.ndarray:
    """wave2d_host_scalars: the scalar row of one half-step (host only, no device)."""
    L = load_library()
    out = np.zeros(4096, dtype=np.float64)
    cnt = C.c_int()
    st = L.wave2d_host_scalars(gamma, alpha_plus, alpha_minus, q, out.ctypes.data_as(C.POINTER(C.c_double)),
                               out.size, C.byref(cnt))
    if st != 0:
        raise Wave2DError(st, "wave2d_host_scalars", L.wave2d_strerror(st).decode())
    return out[:cnt.value].copy()


def host_decay(N: int, extent: float, tau: float, c: float, gamma: float = 2.0, sigma: float = 0.5) -> float:
    """wave2d_host_decay: rho of a sweep over lines of mesh width extent / N at speed c (host only, no device)."""
    L = load_library()
    rho = C.c_double()
    st = L.wave2d_host_decay(int(N), float(extent), float(tau), float(c), float(gamma), float(sigma), C.byref(rho))
    if st != 0:
        raise Wave2DError(st, "wave2d_host_decay", L.wave2d_strerror(st).decode())
    return rho.value


def host_plan(n: int, nlines: int, unit: int, units_per_stage: int, units_per_tile: int, nbk: int, slots: int,
              fixed_stages: int = 0, static_frac: float = 0.75):
    """wave2d_host_plan: (pieces[npieces, 4], nstatic, cta_off[slots + 1]) (host only, no device)."""
    L = load_library()
    cap = 1 << 20
    pieces = np.zeros((cap, 4), dtype=np.int32)
    cta_off = np.zeros(slots + 1, dtype=np.int32)
    npieces, nstatic = C.c_int(), C.c_int()
    ip = C.POINTER(C.c_int)
    st = L.wave2d_host_plan(n, nlines, unit, units_per_stage, units_per_tile, nbk, slots, fixed_stages,
                            float(static_frac), pieces.ctypes.data_as(ip), cap, C.byref(npieces), C.byref(nstatic),
                            cta_off.ctypes.data_as(ip))
    if st != 0:
        raise Wave2DError(st, "wave2d_host_plan", L.wave2d_strerror(st).decode())
    return pieces[:npieces.value].copy(), nstatic.value, cta_off
