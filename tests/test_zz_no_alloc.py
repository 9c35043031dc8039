"""wave2d_small_steps_static, the entry point for callers that cannot allocate device memory -- collected last on purpose.

Why the entry point exists: every other call of include/wave2d.h works on a handle, and a handle cudaMallocs its time
levels and tables.  A caller living inside a framework whose allocator already owns the GPU's memory, a service with a
fixed device-memory budget, or a loop sharing the GPU with other streams (cudaMalloc / cudaFree stall the whole device)
cannot do that.  For them the small-grid kernel's working memory is a fixed 1.5 MiB array inside libwave2d.so; the limit
is 256 unknowns per line in each direction (N1, N2 <= 257).

What is checked: the new path against the existing handle path (the library's own small-grid kernels, which allocate),
at the tolerance every parity test here uses (1e-10 relative in fp64, 1e-4 in fp32), on TWO CALLS IN A ROW -- the second
continues from the first one's outputs, and in the second test it has another size and dtype, so anything the first call
left behind in the shared array would show.  The oracle is the second witness.  The array is shared by the whole process:
these tests pass alone in a fresh process (the first call does the per-device set-up) and after the rest of the suite.

This file sorts after every other test file: `pytest -x` stops at the first failure, and a failure here must not hide
the parity tests.
"""
import numpy as np
import pytest

from oracle import oracle
from paper_2006_10142_b200 import binding as B
from paper_2006_10142_b200 import workloads as W

TOL = {"f64": 1e-10, "f32": 1e-4}
SEED = 20061016


def relerr(u, r):
    return float(np.abs(np.asarray(u, dtype=np.float64) - r).max() / max(np.abs(r).max(), 1e-300))


def seeded_phi(N1, N2, seed):
    """config 4's recipe: uniform [-1, 1], five Jacobi passes, rounded to fp32 so both dtypes get the same bytes"""
    rng = np.random.default_rng(seed)
    phi = rng.uniform(-1.0, 1.0, size=(N2 - 1, N1 - 1))
    return W.jacobi_smooth(phi, 5).astype(np.float32).astype(np.float64)


def handle_path(N1, N2, l, tau, c, dtype, phi, steps_a, steps_b, **opts):
    """existing path: (u^{a}, u^{a-1/2}, u^{a+b}) from a wave2d_create handle (psi = 0)"""
    npdt = np.float64 if dtype == "f64" else np.float32
    h = B.Wave2D(N1, N2, l, tau, steps_a + steps_b, dtype)
    try:
        for k, v in opts.items():
            h.set_option(k, v)
        h.set_speed([c])
        h.set_initial(phi.astype(npdt))
        h.run(steps_a)
        ua, pa = h.get(), h.get_prev()
        h.run(steps_b)
        ub = h.get()
        assert h.info("solver_x") == B.SOLVER_LINE
    finally:
        h.close()
    return ua, pa, ub


def static_path(N1, N2, l, tau, c, dtype, phi, steps_a, steps_b, pad=0, in_place=False):
    """new path, two calls in a row on torch's current stream; every tensor is made here, by the caller"""
    import torch
    tdt = torch.float64 if dtype == "f64" else torch.float32
    n1, n2 = N1 - 1, N2 - 1

    def field(fill=None):   # rows `pad` elements apart more than needed: ld > n1 is part of the interface
        t = torch.full((n2, n1 + pad), float("nan"), dtype=tdt, device="cuda")[:, :n1]
        if fill is not None:
            t.copy_(torch.from_numpy(fill).to(tdt))
        return t

    u0 = field(phi)
    p0 = field(phi)                      # psi = 0: u^{-1/2} = phi
    u1, p1 = (u0, p0) if in_place else (field(), field())
    B.small_steps_static(N1, N2, l, tau, c, steps_a, p0, u0, u1, p1)
    ua, pa = u1.cpu().numpy().copy(), p1.cpu().numpy().copy()
    u2 = field()
    B.small_steps_static(N1, N2, l, tau, c, steps_b, p1, u1, u2)        # u_prev_out left out
    return ua, pa, u2.cpu().numpy()


CASES = [
    # N1, N2, tau / h, c, steps of call 1, steps of call 2, row padding, outputs over the inputs
    (128, 128, 0.5, 1.0, 7, 5, 0, False),      # config 1's grid: 4 points per lane
    (257, 200, 1.0, 1.3, 4, 3, 3, False),      # the largest line in x, ragged in y, ld > n1
    (51, 257, 2.5, 0.7, 3, 6, 0, True),        # the largest line in y, tau > h, call 1 in place
    (2, 3, 1.0, 1.0, 2, 2, 0, False),          # one unknown per x line
]


@pytest.mark.gpu
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("case", CASES, ids=lambda c: f"{c[0]}x{c[1]}")
def test_two_calls_in_a_row_match_the_handle_path(case, dtype):
    N1, N2, tau_h, c, sa, sb, pad, in_place = case
    l = 1.0
    tau = tau_h * min(l / N1, l / N2)
    phi = seeded_phi(N1, N2, SEED + N1)
    ua, pa, ub = static_path(N1, N2, l, tau, c, dtype, phi, sa, sb, pad, in_place)
    for opts in ({"resident": 0}, {}):   # the kernel this one is a variant of; the library's default for the size
        ha, hp, hb = handle_path(N1, N2, l, tau, c, dtype, phi, sa, sb, **opts)
        assert relerr(ua, ha.astype(np.float64)) <= TOL[dtype]
        assert relerr(pa, hp.astype(np.float64)) <= TOL[dtype]
        assert relerr(ub, hb.astype(np.float64)) <= TOL[dtype]
    cs = np.full(2 * (sa + sb) + 1, c)
    assert relerr(ua, oracle.solve(N1, N2, l, tau, sa + sb, phi, None, c_half=cs, steps=sa)) <= TOL[dtype]
    assert relerr(ub, oracle.solve(N1, N2, l, tau, sa + sb, phi, None, c_half=cs)) <= TOL[dtype]


@pytest.mark.gpu
def test_a_call_does_not_see_what_the_previous_one_left_in_the_array():
    """a 257 x 257 fp64 call with huge values fills the whole array; the 100 x 90 fp32 call right after it, and the one after
    that, must still match the handle path (its pad columns have to be zero, not the neighbour's leftovers)"""
    import torch
    big = torch.full((256, 256), 1e30, dtype=torch.float64, device="cuda")
    out = torch.empty_like(big)
    B.small_steps_static(257, 257, 1.0, 1.0 / 257, 1.0, 1, big, big, out, None)
    N1, N2, l, c = 100, 90, 1.0, 1.0
    tau = 1.0 / 100
    phi = seeded_phi(N1, N2, SEED)
    ua, pa, ub = static_path(N1, N2, l, tau, c, "f32", phi, 5, 4)
    ha, hp, hb = handle_path(N1, N2, l, tau, c, "f32", phi, 5, 4, resident=0)
    assert relerr(ua, ha.astype(np.float64)) <= TOL["f32"]
    assert relerr(pa, hp.astype(np.float64)) <= TOL["f32"]
    assert relerr(ub, hb.astype(np.float64)) <= TOL["f32"]


@pytest.mark.gpu
def test_refusals_on_the_device():
    import torch
    t = torch.zeros((9, 9), dtype=torch.float64, device="cuda")
    host = torch.zeros((9, 9), dtype=torch.float64)
    L = B.load_library()
    import ctypes as C
    err = C.create_string_buffer(256)
    st = L.wave2d_small_steps_static(10, 10, 1.0, 0.1, 1.0, 1, B.F64, C.c_void_p(host.data_ptr()), C.c_void_p(t.data_ptr()),
                                     C.c_void_p(t.data_ptr()), None, 9, None, err, len(err))
    assert st == -1 and b"DEVICE memory" in err.value            # a host array is refused, not staged
    with pytest.raises(B.Wave2DError) as e:
        B.small_steps_static(10, 10, 1.0, 0.1, -1.0, 1, t, t, t)  # c <= 0
    assert e.value.status == -1


def test_sizes_beyond_the_array_are_refused_before_any_cuda_call():
    """no GPU needed: the size check comes first.  258 intervals = 257 unknowns per line > 256."""
    import ctypes as C
    L = B.load_library()
    err = C.create_string_buffer(256)
    dummy = C.c_void_p(16)   # never dereferenced
    for N1, N2 in ((258, 10), (10, 258), (4096, 4096)):
        st = L.wave2d_small_steps_static(N1, N2, 1.0, 0.01, 1.0, 1, B.F64, dummy, dummy, dummy, None, N1 - 1, None, err, len(err))
        assert st == -5, (N1, N2, st)
        assert b"at most 256 unknowns" in err.value and b"wave2d_create" in err.value
    st = L.wave2d_small_steps_static(257, 257, 1.0, 0.01, 1.0, 0, B.F64, dummy, dummy, dummy, None, 256, None, err, len(err))
    assert st == -1 and err.value                                 # steps < 1
    st = L.wave2d_small_steps_static(257, 257, 1.0, 0.01, 1.0, 1, B.F64, dummy, dummy, dummy, None, 255, None, None, 0)
    assert st == -1                                               # ld < n1; no error buffer is fine
