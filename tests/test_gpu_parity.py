"""Parity of the CUDA path (through the C ABI, include/wave2d.h) against the CPU oracle -- `-m gpu`.

Tolerances are BASELINE.json's north_star: max|u_gpu - u_oracle| <= 1e-10 * max|u_oracle| after all M
steps in fp64, 1e-4 in the fp32 variant.  Every input is seeded and synthetic
(paper_2006_10142_b200/workloads.py); the same bytes go to both sides.  Nothing here reads /root/reference.
"""
import numpy as np
import pytest

from oracle import oracle
from paper_2006_10142_b200 import binding as B
from paper_2006_10142_b200 import workloads as W
from tests.modal import modal_amplitudes

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-10, "f32": 1e-4}


def ref(w, steps=None, gamma=None, kappa=None):
    return oracle.solve(w.N1, w.N2, w.l, w.tau, w.M, w.phi, w.psi, c_half=w.c_half, s=w.s, g_half=w.g_half,
                        steps=steps, gamma=gamma, kappa=kappa)


def gpu(w, steps=None, **opts):
    return gpu_info(w, (), steps, **opts)


def gpu_info(w, keys, steps=None, **opts):
    h = B.Wave2D(w.N1, w.N2, w.l, w.tau, w.M, w.dtype)
    try:
        for k, v in opts.items():
            h.set_option(k, v)
        npdt = np.float64 if w.dtype == "f64" else np.float32
        h.set_speed(w.c_half)
        if w.s is not None:
            h.set_source(w.s.astype(npdt), w.g_half)
        h.set_initial(w.phi.astype(npdt), None if w.psi is None else w.psi.astype(npdt))
        h.run(w.M if steps is None else steps)
        u = h.get()
        info = {k: h.info(k) for k in ("solver_x", "solver_y", "launches", "chunks_x", "chunks_y") + tuple(keys)}
    finally:
        h.close()
    return u, info


def relerr(u, r):
    return float(np.abs(u.astype(np.float64) - r).max() / max(np.abs(r).max(), 1e-300))


def small_cases():
    return [
        ("cfg1", W.cfg1()),
        ("cfg2_N96", W.cfg2(N=96, M=40)),
        ("cfg2_N700", W.cfg2(N=700, M=50)),            # several line tiles, ragged tail in both directions
        ("cfg3_N128", W.cfg3(N=128, M=60)),
        ("cfg3_N1000", W.cfg3(N=1000, M=260)),         # source switched on (Ricker centre at step ~245)
        ("cfg4_160x40", W.cfg4(N1=160, N2=40, M=30)),
        ("cfg4_1030x270", W.cfg4(N1=1030, N2=270, M=24)),
        ("cfg4_160x40_f32", W.cfg4(N1=160, N2=40, M=30, dtype="f32")),
        ("cfg4_1030x270_f32", W.cfg4(N1=1030, N2=270, M=200, dtype="f32")),
        ("cfg5_N192", W.cfg5(N=192, M=20)),
    ]


_ST = {"solver": B.SOLVER_STREAM}


@pytest.mark.parametrize("name,w", small_cases(), ids=[c[0] for c in small_cases()])
@pytest.mark.parametrize("opts", [{}, _ST, {"solver": B.SOLVER_EXACT}, {"graph": 0, **_ST},
                                  {"quota_x": 3, "quota_y": 3, **_ST},
                                  {"shape_x": 1, "shape_y": 1, "quota_x": 4, "quota_y": 5, **_ST},
                                  {"shape_x": 2, "shape_y": 3, **_ST}, {"shape_x": 3, "shape_y": 2, **_ST}],
                         ids=["default", "stream", "exact", "nograph", "quota3", "shapes1_cut", "shapes23", "shapes32"])
def test_small_workloads_match_oracle(name, w, opts):
    r = ref(w)
    u, info = gpu(w, **opts)
    assert np.isfinite(u).all()
    assert relerr(u, r) <= TOL[w.dtype]
    want = opts.get("solver", B.SOLVER_LINE if max(w.n1, w.n2) <= 256 else B.SOLVER_STREAM)   # AUTO: small grids -> LINE
    assert info["solver_x"] == want and info["solver_y"] == want
    if want == B.SOLVER_LINE:
        assert info["launches"] == 1            # Algorithm 1's whole loop in one launch
    else:
        assert info["launches"] >= 2 * w.M      # the CUDA kernels ran: >= 2 sweeps per step


@pytest.mark.parametrize("N1,N2", [(2, 2), (2, 9), (9, 2), (3, 3), (4, 5), (16, 17), (17, 16), (18, 33), (33, 18),
                                   (127, 129), (129, 127), (128, 128), (130, 66), (257, 40)])
def test_tiny_and_ragged_sizes(N1, N2):
    """n = 1, 2, 3 unknowns per line, sizes straddling one 16-point unit / one 32-line tile."""
    rng = np.random.default_rng(1000 * N1 + N2)
    M = 7
    tau = 0.9 / max(N1, N2)
    phi = rng.uniform(-1, 1, (N2 - 1, N1 - 1))
    psi = rng.uniform(-1, 1, (N2 - 1, N1 - 1))
    s = rng.uniform(-1, 1, (N2 - 1, N1 - 1))
    c = rng.uniform(0.5, 1.5, 2 * M + 1)
    g = rng.uniform(-1, 1, 2 * M)
    w = W.Workload("rand", N1, N2, 1.0, tau, M, "f64", phi, psi, c, s=s, g_half=g)
    r = ref(w)
    for opts in ({}, {"solver": B.SOLVER_STREAM}, {"solver": B.SOLVER_EXACT}):   # {}: the small-grid kernel (LINE)
        u, _ = gpu(w, **opts)
        assert relerr(u, r) <= 1e-12, (opts, relerr(u, r))


def test_literal_constants_gamma1_kappa1():
    """The scheme exactly as printed: gamma = kappa = 1 (reading A2)."""
    w = W.cfg3(N=200, M=30)
    w.phi = W.cfg2(N=200, M=30).phi
    w.g_half = np.cos(np.arange(2 * w.M) * 0.3)
    r = ref(w, gamma=1.0, kappa=1.0)
    u, _ = gpu(w, gamma=1.0, kappa=1.0)
    assert relerr(u, r) <= 1e-10
    assert relerr(u, ref(w)) > 1e-3   # and it differs from the default reading


@pytest.mark.parametrize("N", [160, 300])
def test_large_tau_falls_back_to_exact_solver(N):
    """tau = 16 h: rho = 0.88, the decay bound needs ~300 points of look-ahead: the streamed kernels refuse, AUTO
    picks the small-grid kernel (exact for any tau) at N = 160 and the EXACT path at N = 300."""
    M = 12
    w = W.cfg2(N=N, M=M)
    w.tau = 16.0 / N
    r = ref(w)
    u, info = gpu(w)
    want = B.SOLVER_LINE if N <= 257 else B.SOLVER_EXACT
    assert info["solver_x"] == want and info["solver_y"] == want
    assert relerr(u, r) <= 1e-10
    with pytest.raises(B.Wave2DError) as e:
        gpu(w, solver=B.SOLVER_STREAM)
    assert e.value.status == -5
    u, info = gpu(w, solver=B.SOLVER_EXACT)
    assert info["solver_x"] == B.SOLVER_EXACT and relerr(u, r) <= 1e-10


@pytest.mark.parametrize("ratio,H", [(2.3, 47), (3.0, 60)])
def test_moderate_tau_uses_longer_carry_series(ratio, H):
    """tau = 2.3 h / 3 h (alpha = 2.6 / 4.5, rho = 0.43 / 0.52): rho^H <= 1e-17 needs H = 47 / 60 points in
    fp64, i.e. a carry series of 6 / 8 units of 8 points (the kernels carry up to 8 units); the boundary pivots
    still converge inside the 128-row table.  Cut lines (quota) exercise the carry warm-up."""
    N, M = 600, 8
    w = W.cfg2(N=N, M=M)
    w.tau = ratio / N
    w.c_half = np.ones(2 * M + 1)
    r = ref(w)
    for opts in ({}, {"quota_x": 4, "quota_y": 4}):
        u, info = gpu_info(w, ("nbk_x", "nbk_y", "unit_x", "unit_y"), **opts)
        assert info["solver_x"] == B.SOLVER_STREAM and info["solver_y"] == B.SOLVER_STREAM
        assert info["nbk_x"] == -(-H // info["unit_x"]) and info["nbk_y"] == -(-H // info["unit_y"])
        assert relerr(u, r) <= 1e-10


def test_run_in_pieces_equals_one_run_and_reset_is_reproducible():
    w = W.cfg2(N=260, M=40)
    h = B.from_workload(w)
    try:
        h.run(w.M)
        a = h.get()
        h.set_initial(w.phi)            # resets k to 0
        assert h.steps_done() == 0
        for part in (1, 12, 2, 24, 1):   # plain launches, graph replays, tails
            h.run(part)
        assert h.steps_done() == w.M
        b = h.get()
        prev = h.get_prev()
    finally:
        h.close()
    assert np.array_equal(a, b)         # bit-reproducible regardless of how the steps are batched
    o = oracle.Wave2DOracle(w.N1, w.N2, w.l, w.tau, w.M)
    o.set_speed(w.c_half)
    o.set_initial(w.phi)
    o.run(w.M)
    assert relerr(prev, o.get_prev()) <= 1e-10
    o.close()


@pytest.mark.parametrize("scheme", [0, 1])
def test_every_run_call_replays_graphs_at_any_ring_phase(scheme):
    """A7: the graphs are built with the plan, the kernels take the buffer roles from the device step counter, so
    run(5); run(20) (the driver's bench pattern: warm-up 5, then 20 timed steps at ring phase 5 mod 3) issues graph
    replays only -- no sweep kernel outside a graph, no capture inside a run call -- and is bit-identical to run(25)
    and to plain launches (graph = 0)."""
    w = W.cfg2(N=700, M=60)
    src = W.cfg3(N=700, M=60)
    w.s, w.g_half = src.s, W.ricker(W.half_times(w.tau, 2 * w.M) + 0.058)

    def handle(**opts):
        h = B.Wave2D(w.N1, w.N2, w.l, w.tau, w.M, "f64")
        if scheme:
            h.set_option("scheme", 1)
        for k, v in opts.items():
            h.set_option(k, v)
        h.set_speed(w.c_half)
        h.set_source(w.s, w.g_half)
        h.set_initial(w.phi)
        return h

    h = handle()
    try:
        h.run(0)                                     # plans, captures, instantiates, uploads
        assert h.info("launches") == 0 and h.info("graph_launches") == 0
        h.run(5)                                     # 4 + 1
        assert h.info("graph_launches") == 2
        h.run(20)                                    # 16 + 4
        assert h.info("graph_launches") == 4 and h.info("plain_sweeps") == 0
        assert h.info("launches") == 2 * 25 + 4 + (2 if scheme else 0)   # two sweeps per step, one counter kernel per chunk
                                                                          # (scheme 1: + the two start kernels)
        a = h.get()
        for part in (1, 1, 1, 2, 3, 7, 13):          # every phase of the ring, every chunk length below 16
            h.run(part)
        assert h.info("plain_sweeps") == 0
        a2 = h.get()
    finally:
        h.close()
    K2 = 25 + 28
    for opts, K, want in (({}, 25, a), ({"graph": 0}, 25, a), ({"graph_steps": 4}, 25, a), ({}, K2, a2),
                          ({"graph": 0, "pdl": 0}, K2, a2)):
        h = handle(**opts)
        try:
            h.run(K)                                 # K solves in one call
            u = h.get()
            if opts.get("graph") == 0:
                assert h.info("graph_launches") == 0 and h.info("plain_sweeps") > 0
        finally:
            h.close()
        assert np.array_equal(u, want), (opts, K)
    if scheme == 0:
        assert relerr(a2, ref(w, steps=K2)) <= 1e-10
    else:
        assert relerr(a2, ref1(w, K=K2 + 1)) <= 1e-10          # set_initial stands at level 1: K2 solves reach K2 + 1


def test_device_pointers_strided_inputs_and_user_stream():
    import torch
    w = W.cfg4(N1=200, N2=120, M=15)
    r = ref(w)
    dev = torch.device("cuda:0")
    ld = w.n1 + 5
    big = torch.zeros((w.n2, ld), dtype=torch.float64, device=dev)
    big[:, :w.n1] = torch.from_numpy(w.phi).to(dev)
    st = torch.cuda.Stream()
    h = B.Wave2D(w.N1, w.N2, w.l, w.tau, w.M, "f64")
    try:
        h.set_stream(st)
        h.set_speed(w.c_half)
        h.set_initial(big[:, :w.n1])     # device pointer, ld > n1
        h.run(w.M)
        out = torch.full((w.n2, ld), 7.0, dtype=torch.float64, device=dev)
        h.get(out[:, :w.n1])
    finally:
        h.close()
    assert relerr(out[:, :w.n1].cpu().numpy(), r) <= 1e-10
    assert bool((out[:, w.n1:] == 7.0).all())   # padding columns of the caller's buffer untouched


def test_state_machine_and_argument_errors():
    with pytest.raises(B.Wave2DError) as e:
        B.Wave2D(1, 8, 1.0, 0.1, 4)
    assert e.value.status == -1
    h = B.Wave2D(32, 32, 1.0, 0.01, 4)
    try:
        with pytest.raises(B.Wave2DError) as e:
            h.run(1)
        assert e.value.status == -2                       # run before set_initial
        with pytest.raises(B.Wave2DError) as e:
            h.set_speed(np.array([1.0, -1.0, 1.0, 1.0, 1.0, 1.0, 1.0, 1.0, 1.0]))
        assert e.value.status == -1                       # c must be positive
        with pytest.raises(B.Wave2DError) as e:
            h.set_speed(np.ones(5))
        assert e.value.status == -1                       # count must be 1 or 2M+1
        h.set_initial(np.zeros((31, 31)))
        h.run(3)
        with pytest.raises(B.Wave2DError) as e:
            h.set_speed(np.ones(1))
        assert e.value.status == -2                       # set_* after the first run
        with pytest.raises(B.Wave2DError) as e:
            h.run(2)
        assert e.value.status == -6                       # more than M steps
        assert np.array_equal(h.get(), np.zeros((31, 31)))   # zero in, exactly zero out
    finally:
        h.close()


# ---- full-size grids in the launch configuration bench.py times --------------------------------------------
def test_cfg1_full_modal_closed_form():
    w = W.cfg1()
    u, _ = gpu(w)
    a = modal_amplitudes(w.N1, w.N2, w.l, w.tau, 1, 1, 1.0, 0.0, w.c_half, 2 * w.M)[-1]
    # rounding noise eps per half-step enters the marginally stable three-term recurrence and grows like
    # n per injection, so ~ n^2 eps / 2 = 200^2 * 1.1e-16 / 2 = 2e-12 in the worst case (the oracle itself sits
    # 1.3e-12 from the closed form, tests/test_oracle_pins.py): 1e-11 absolute on an O(0.17) field.
    assert np.abs(u - a * w.phi).max() <= 1e-11
    assert relerr(u, ref(w)) <= 1e-10


def test_cfg2_full_size_full_M():
    w = W.cfg2()
    r = ref(w)
    u, info = gpu(w)
    assert relerr(u, r) <= 1e-10
    assert np.abs(u - u[::-1, :]).max() <= 1e-12 and np.abs(u - u[:, ::-1]).max() <= 1e-12   # quadrant symmetry


def test_cfg3_full_grid_source_on():
    """4095^2 grid in bench.py's launch configuration; 24 steps with the Ricker wavelet shifted so that the
    source is at its peak inside the window (the full M = 1000 oracle run is opt-in, see below)."""
    M = 24
    w = W.cfg3(N=4096, M=M)
    w.g_half = W.ricker(W.half_times(w.tau, 2 * M) + 0.058)
    r = ref(w)
    u, info = gpu(w)
    assert info["solver_x"] == B.SOLVER_STREAM and info["solver_y"] == B.SOLVER_STREAM
    assert np.abs(r).max() > 1e-6
    assert relerr(u, r) <= 1e-10


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_cfg4_full_grid(dtype):
    w = W.cfg4(M=16, dtype=dtype)
    r = ref(w)
    u, info = gpu(w)
    assert info["solver_x"] == B.SOLVER_STREAM and info["solver_y"] == B.SOLVER_STREAM
    assert relerr(u, r) <= TOL[dtype]


def test_cfg5_full_size_full_M_against_modal_closed_form():
    """16383^2, M = 200: every mode's amplitude follows the exact scalar recurrence (tests/modal.py), so the
    result is known at every point without running the oracle at this size.  Compared on 64 sampled rows."""
    w = W.cfg5()
    u, info = gpu(w)
    assert info["solver_x"] == B.SOLVER_STREAM and info["solver_y"] == B.SOLVER_STREAM
    x, y = W.grid(w.N1, w.N2)
    rows = np.unique(np.r_[0, 1, w.n2 - 1, np.random.default_rng(5).integers(0, w.n2, 61)])
    expect = np.zeros((rows.size, w.n1))
    for m, n, A in w.modes:
        a = modal_amplitudes(w.N1, w.N2, w.l, w.tau, m, n, A, 0.0, w.c_half, 2 * w.M)[-1]
        expect += a * np.outer(np.sin(n * np.pi * y[rows]), np.sin(m * np.pi * x))
    scale = max(abs(A) for _, _, A in w.modes)
    assert np.abs(u[rows] - expect).max() <= 1e-10 * scale
    assert np.isfinite(u).all()


def test_results_do_not_depend_on_which_cta_runs_a_piece():
    """The pieces of the dynamic tail are drawn by whichever CTA is free, and every stage goes through two CTA
    barriers, an mbarrier ring and double-buffered store tiles: any race or order dependence would show up as
    run-to-run differences.  Three runs of a 2047^2 grid (several pieces per CTA) must agree bit for bit, and so
    must runs under different work distributions (what a thread computes never depends on the cut positions of
    other pieces)."""
    w = W.cfg3(N=2048, M=30)
    w.g_half = W.ricker(W.half_times(w.tau, 2 * w.M) + 0.058)
    runs = [gpu(w)[0] for _ in range(3)]
    assert np.array_equal(runs[0], runs[1]) and np.array_equal(runs[0], runs[2])
    assert relerr(runs[0], ref(w)) <= 1e-10
    other, info = gpu(w, static_frac=0.3, shape_y=3)
    assert relerr(other, runs[0]) <= 1e-13      # different cuts: same to rounding of the carry truncation


def test_trace_records_every_cta():
    w = W.cfg2(N=700, M=6)
    h = B.from_workload(w)
    try:
        h.set_option("trace", 1)
        h.run(w.M)
        for d in (0, 1):
            t = h.trace(d).astype(np.int64)
            assert len(t) == int(h.info("grid_x" if d == 0 else "grid_y"))
            assert np.all(t[:, 1] > t[:, 0]) and np.all(t[:, 2] < 160)      # end after start; SM ids
            assert t[:, 3].sum() == int(h.info("chunks_x" if d == 0 else "chunks_y"))   # every piece ran exactly once
        u = h.get()
    finally:
        h.close()
    assert relerr(u, ref(w)) <= 1e-10


def test_zero_steps_and_M_zero():
    w = W.cfg2(N=64, M=4)
    h = B.from_workload(w)
    try:
        h.run(0)
        assert h.steps_done() == 0
        assert np.array_equal(h.get(), w.phi)           # u^0 = phi, untouched
    finally:
        h.close()
    h = B.Wave2D(16, 16, 1.0, 0.01, 0)                   # M = 0: nothing can be run, nothing breaks
    try:
        h.set_initial(np.ones((15, 15)))
        h.run(0)
        with pytest.raises(B.Wave2DError):
            h.run(1)
        assert np.array_equal(h.get(), np.ones((15, 15)))
    finally:
        h.close()


# ---- scheme 1: the factorised form of the unsplit scheme (2.8) -------------
def ref1(w, K=None):
    npdt = np.float64 if w.dtype == "f64" else np.float32
    cast = lambda a: None if a is None else a.astype(npdt).astype(np.float64)
    return oracle.solve(w.N1, w.N2, w.l, w.tau, w.M, cast(w.phi), cast(w.psi), c_half=w.c_half, s=cast(w.s),
                        g_half=w.g_half, steps=K, scheme=1)


def gpu1(w, K=None, **opts):
    h = B.Wave2D(w.N1, w.N2, w.l, w.tau, w.M, w.dtype)
    try:
        h.set_option("scheme", 1)
        for k, v in opts.items():
            h.set_option(k, v)
        npdt = np.float64 if w.dtype == "f64" else np.float32
        h.set_speed(w.c_half)
        if w.s is not None:
            h.set_source(w.s.astype(npdt), w.g_half)
        h.set_initial(w.phi.astype(npdt), None if w.psi is None else w.psi.astype(npdt))
        assert h.steps_done() == 1                      # (2.9): set_initial stands at time level 1
        h.run((w.M if K is None else K) - 1)
        u = h.get()
        info = {k: h.info(k) for k in ("solver_x", "solver_y", "launches")}
    finally:
        h.close()
    return u, info


def factored_cases():
    rng = np.random.default_rng(77)
    a = W.cfg2(N=300, M=30)
    a.psi = 0.3 * a.phi
    b = W.cfg3(N=260, M=40)
    b.g_half = W.ricker(W.half_times(b.tau, 2 * b.M) + 0.058)
    c = W.cfg4(N1=330, N2=140, M=25)
    c.psi = rng.uniform(-1, 1, c.phi.shape)
    d = W.cfg4(N1=330, N2=140, M=25, dtype="f32")
    e = W.cfg5(N=200, M=26)
    f = W.cfg3(N=261, M=40)                          # fp32 with a source: the x sweep adds it, the y sweep has none
    f.dtype = "f32"
    f.g_half = W.ricker(W.half_times(f.tau, 2 * f.M) + 0.058)
    return [("cfg2_N300_psi", a), ("cfg3_N260_source", b), ("cfg4_330x140_psi", c), ("cfg4_330x140_f32", d),
            ("cfg5_N200", e), ("cfg3_N261_source_f32", f)]


@pytest.mark.parametrize("name,w", factored_cases(), ids=[c[0] for c in factored_cases()])
@pytest.mark.parametrize("opts", [{}, _ST, {"solver": B.SOLVER_EXACT}, {"graph": 0, **_ST},
                                  {"quota_x": 3, "quota_y": 3, **_ST}],
                         ids=["default", "stream", "exact", "nograph", "quota3"])
def test_factored_scheme_matches_oracle(name, w, opts):
    r = ref1(w)
    u, info = gpu1(w, **opts)
    assert np.isfinite(u).all()
    assert relerr(u, r) <= TOL[w.dtype]
    if info["solver_x"] == B.SOLVER_LINE:
        assert info["launches"] == 3            # the two start kernels + one launch for every step
    else:
        assert info["launches"] >= 2 * (w.M - 1)


def test_factored_scheme_levels_one_by_one_and_modal():
    """Every time level of a single mode against the scalar recurrence of tests/modal.py (c(t), psi != 0)."""
    from tests.modal import modal_amplitudes_factored
    N1, N2, M = 96, 80, 23
    tau = 1.1 / 96
    x, y = W.grid(N1, N2)
    shape = np.outer(np.sin(2 * np.pi * y), np.sin(3 * np.pi * x))
    c_half = 1.0 + 0.4 * np.sin(np.arange(2 * M + 1) * 0.3)
    amps = modal_amplitudes_factored(N1, N2, 1.0, tau, 3, 2, 0.8, -0.5, c_half, M)
    h = B.Wave2D(N1, N2, 1.0, tau, M, "f64")
    try:
        h.set_option("scheme", 1)
        h.set_speed(c_half)
        h.set_initial(0.8 * shape, -0.5 * shape)
        assert np.abs(h.get_prev() - 0.8 * shape).max() == 0.0          # U^0 until the first solve
        for K in range(1, M + 1):
            assert h.steps_done() == K
            assert np.abs(h.get() - amps[K] * shape).max() <= 1e-12
            if K < M:
                h.run(1)
        with pytest.raises(B.Wave2DError):
            h.run(1)                                                      # past M
        with pytest.raises(B.Wave2DError):
            h.get_prev()                                                  # the ring carries V^{k-1}, not U^{k-1}
    finally:
        h.close()


def test_factored_scheme_full_grid_4095():
    w = W.cfg3(N=4096, M=26)
    w.g_half = W.ricker(W.half_times(w.tau, 2 * w.M) + 0.058)
    w.phi = W.cfg2(N=4096, M=1).phi
    r = ref1(w)
    u, info = gpu1(w)
    assert info["solver_x"] == B.SOLVER_STREAM and info["solver_y"] == B.SOLVER_STREAM
    assert relerr(u, r) <= 1e-10


def test_factored_scheme_state_machine():
    h = B.Wave2D(32, 32, 1.0, 0.01, 4)
    try:
        h.set_initial(np.zeros((31, 31)))
        with pytest.raises(B.Wave2DError) as e:
            h.set_option("scheme", 1)                   # must precede set_initial
        assert e.value.status == -1
    finally:
        h.close()
    h = B.Wave2D(32, 32, 1.0, 0.01, 0)
    try:
        h.set_option("scheme", 1)
        with pytest.raises(B.Wave2DError) as e:
            h.set_initial(np.zeros((31, 31)))           # (2.9) needs level 1 to exist: M >= 1
        assert e.value.status == -6
    finally:
        h.close()
    h = B.Wave2D(32, 32, 1.0, 0.01, 3)
    try:
        h.set_option("scheme", 1)
        phi = np.ones((31, 31))
        h.set_initial(phi, 2.0 * phi)
        assert h.steps_done() == 1 and np.allclose(h.get(), 1.0 + 0.02)   # u^1 = phi + tau psi
        h.run(0)
        h.run(2)
        assert h.steps_done() == 3
        with pytest.raises(B.Wave2DError) as e:
            h.run(1)
        assert e.value.status == -6
        h.set_initial(phi)                               # reset: back to level 1
        assert h.steps_done() == 1 and np.array_equal(h.get(), phi)
    finally:
        h.close()


def test_checkpoint_resume_is_bit_identical():
    """State of Algorithm 1 = (u^{k-1/2}, u^k): get_prev/get at k = 17, a fresh handle put there
    with wave2d_set_state, and the continuation equals the uninterrupted run bit for bit."""
    w = W.cfg3(N=300, M=40)
    w.g_half = W.ricker(W.half_times(w.tau, 2 * w.M) + 0.058)
    w.phi = W.cfg2(N=300, M=1).phi
    h = B.from_workload(w)
    try:
        h.run(17)
        prev, cur = h.get_prev(), h.get()
        h.run(w.M - 17)
        full = h.get()
    finally:
        h.close()
    h = B.Wave2D(w.N1, w.N2, w.l, w.tau, w.M, w.dtype)
    try:
        h.set_speed(w.c_half)
        h.set_source(w.s, w.g_half)
        h.set_state(17, prev, cur)
        assert h.steps_done() == 17
        h.run(w.M - 17)
        assert np.array_equal(h.get(), full)
        with pytest.raises(B.Wave2DError):
            h.set_state(w.M + 1, prev, cur)
    finally:
        h.close()
    assert relerr(full, ref(w)) <= 1e-10
    h = B.Wave2D(w.N1, w.N2, w.l, w.tau, w.M, w.dtype)
    try:
        h.set_option("scheme", 1)
        with pytest.raises(B.Wave2DError) as e:
            h.set_state(3, prev, cur)
        assert e.value.status == -5
    finally:
        h.close()


@pytest.mark.parametrize("scheme", [0, 1])
def test_constant_speed_needs_no_per_step_table(scheme):
    """c = const, g = const (the paper's own runs): two table rows serve every step, so M = 600 000
    (a 1.3 GB table otherwise: ERR_UNSUPPORTED) runs; the first 26 levels are compared with the oracle."""
    N, M, K = 200, 600_000, 26
    w = W.cfg2(N=N, M=K)
    tau = w.tau
    s = W.cfg3(N=N, M=K).s
    def run_gpu(c_half):
        h = B.Wave2D(N, N, 1.0, tau, M, "f64")
        try:
            if scheme:
                h.set_option("scheme", 1)
            h.set_speed(c_half)
            h.set_source(s, None)                       # g == 1: the time-independent "full grid" source (R11)
            h.set_initial(w.phi)
            h.run(K - h.steps_done())
            return h.get()
        finally:
            h.close()
    u = run_gpu(np.array([1.3]))
    r = oracle.solve(N, N, 1.0, tau, K, w.phi, None, c_half=np.full(2 * K + 1, 1.3), s=s, g_half=None, scheme=scheme)
    assert relerr(u, r) <= 1e-10
    varying = np.full(2 * M + 1, 1.3)
    varying[7] = 1.31                                   # not constant: needs 2M rows of 2 KB -> refused, not truncated
    with pytest.raises(B.Wave2DError) as e:
        run_gpu(varying)
    assert e.value.status == -5


@pytest.mark.parametrize("N1,N2", [(2, 2), (2, 9), (9, 2), (3, 3), (4, 5), (17, 16), (18, 33), (33, 18), (34, 34),
                                   (65, 66), (66, 65), (127, 129), (129, 127), (130, 66), (257, 40), (40, 257)])
@pytest.mark.parametrize("dtype,scheme", [("f32", 0), ("f64", 1), ("f32", 1)])
def test_tiny_and_ragged_sizes_fp32_and_scheme1(N1, N2, dtype, scheme):
    """Sizes straddling one unit / one 32-line (fp32 y sweep: 64-column) panel, odd and even n1 (the vec2f y sweep
    pairs columns; an odd n1 leaves a zero pad column in the last pair), for fp32 and for scheme 1."""
    rng = np.random.default_rng(7000 * N1 + 13 * N2 + scheme)
    M = 7
    tau = 0.9 / max(N1, N2)
    shape = (N2 - 1, N1 - 1)
    phi, psi, s = (rng.uniform(-1, 1, shape) for _ in range(3))
    c = rng.uniform(0.5, 1.5, 2 * M + 1)
    g = rng.uniform(-1, 1, 2 * M)
    w = W.Workload("rand", N1, N2, 1.0, tau, M, dtype, phi, psi, c, s=s, g_half=g)
    tol = 1e-12 if dtype == "f64" else 2e-5
    for opts in ({}, {"solver": B.SOLVER_STREAM}, {"solver": B.SOLVER_EXACT}):
        if scheme:
            u, _ = gpu1(w, **opts)
            r = ref1(w)
        else:
            u, _ = gpu(w, **opts)
            npdt = np.float32
            r = oracle.solve(N1, N2, 1.0, tau, M, phi.astype(npdt).astype(float), psi.astype(npdt).astype(float),
                             c_half=c, s=s.astype(npdt).astype(float), g_half=g)
        assert relerr(u, r) <= tol, (opts, relerr(u, r))


def test_early_start_engages_and_changes_no_bit():
    """At 3000^2 both sweeps deal out a static share AND draw a tail, so the planner marks safe pieces (at
    2048^2 and below it marks none and the early-start protocol was never exercised bitwise).  Early start on / off
    and programmatic launch on / off must agree bit for bit, repeatedly, for both schemes."""
    w = W.cfg2(N=3000, M=14)
    src = W.cfg3(N=3000, M=14)
    w.s, w.g_half = src.s, W.ricker(W.half_times(w.tau, 2 * w.M) + 0.058)
    base, info = gpu_info(w, ("safe_x", "safe_y", "static_x", "static_y", "chunks_x", "chunks_y"), early=0, pdl=0)
    assert relerr(base, ref(w)) <= 1e-10
    _, info = gpu_info(w, ("safe_x", "safe_y", "static_x", "static_y"), early=1)
    assert info["safe_x"] > 0 and info["safe_y"] > 0, info
    assert info["static_x"] < info["chunks_x"] and info["static_y"] < info["chunks_y"]   # a drawn tail exists
    for opts in ({"early": 1}, {"early": 0}, {"early": 1, "graph": 0}, {"early": 1}, {"early": 1, "graph_steps": 2},
                 {"early": 1}):
        u, _ = gpu(w, **opts)
        assert np.array_equal(u, base), opts
    base1, _ = gpu1(w, early=0, pdl=0)
    assert relerr(base1, ref1(w)) <= 1e-10
    for opts in ({"early": 1}, {"early": 1, "graph": 0}, {"early": 1}):
        u, _ = gpu1(w, **opts)
        assert np.array_equal(u, base1), opts


def test_early_start_and_pdl_do_not_change_a_single_bit():
    """Early start only changes WHEN a piece runs (and the order of a CTA's share), programmatic launch only how
    kernels are chained: with both off, one off, both on, three runs each way must agree bit for bit on a grid with
    several pieces per CTA, a source and time-varying c (split scheme) -- and the same for scheme 1."""
    w = W.cfg2(N=2048, M=26)
    src = W.cfg3(N=2048, M=26)
    w.s, w.g_half = src.s, W.ricker(W.half_times(w.tau, 2 * w.M) + 0.058)
    base, _ = gpu(w, early=0, pdl=0)
    assert relerr(base, ref(w)) <= 1e-10
    for opts in ({"early": 1}, {"early": 0}, {"early": 1, "graph": 0}, {"early": 1}, {"early": 1}):
        u, _ = gpu(w, **opts)
        assert np.array_equal(u, base), opts
    base1, _ = gpu1(w, early=0, pdl=0)
    assert relerr(base1, ref1(w)) <= 1e-10
    for opts in ({"early": 1}, {"early": 1, "graph": 0}, {"early": 1}):
        u, _ = gpu1(w, **opts)
        assert np.array_equal(u, base1), opts


@pytest.mark.parametrize("N", [160, 300])
def test_factored_scheme_large_tau_falls_back_to_exact_solver(N):
    M = 10
    w = W.cfg2(N=N, M=M)
    w.tau = 16.0 / N
    w.psi = 0.2 * w.phi
    r = ref1(w)
    u, info = gpu1(w)
    want = B.SOLVER_LINE if N <= 257 else B.SOLVER_EXACT
    assert info["solver_x"] == want and info["solver_y"] == want
    assert relerr(u, r) <= 1e-10


def test_two_handles_on_two_streams_run_concurrently():
    """Two independent simulations, each with persistent one-CTA-per-SM kernels, early start and its own graph, queued
    on two streams at once: no deadlock, and each result equals its solo run bit for bit."""
    import torch
    wa = W.cfg2(N=2700, M=36)                   # static share + drawn tail: early start engaged (safe pieces > 0)
    wb = W.cfg4(N1=1800, N2=900, M=36)
    solo_a, ia = gpu_info(wa, ("safe_x", "safe_y"))
    solo_b, _ = gpu(wb)
    assert ia["safe_x"] > 0 and ia["safe_y"] > 0
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    for it in range(40):   # sharing the SMs shifts every timing inside a CTA: this loop exposed a shared-memory race
        ha, hb = B.from_workload(wa), B.from_workload(wb)   # (7 % of iterations) that no single-handle run ever showed
        try:
            ha.set_stream(sa)
            hb.set_stream(sb)
            for _ in range(3):                 # interleave the submissions
                ha.run(12)
                hb.run(12)
            ua, ub = ha.get(), hb.get()
        finally:
            ha.close()
            hb.close()
        assert np.array_equal(ua, solo_a) and np.array_equal(ub, solo_b), it


# ---- the small-grid kernel (solver LINE): one cluster, one launch for the whole step loop, exact warp-scan solves ----
@pytest.mark.parametrize("n", [1, 2, 3, 5, 31, 32, 33, 126, 127, 128, 129, 200, 255, 256])
@pytest.mark.parametrize("alpha", [0.5, 50.0, 128.0])
def test_line_kernel_sizes_and_any_tau(n, alpha):
    """SURVEY.md 8c pin 7: n in {1, 2, 3, 126..129, ...} and alpha = tau^2 c / (2 h^2) in {0.5, 50, 128} (tau up to 16 h,
    rho = 0.88, where a truncated solver fails: tiny n with large alpha gave 1.7e-1 in the survey's probe).  The warp
    scan truncates nothing, so every case matches the Thomas oracle to rounding.  Asymmetric grid: n x (n + 3)."""
    N1, N2 = n + 1, min(n + 4, 257)
    M = 6
    rng = np.random.default_rng(31 * n + int(alpha))
    tau = np.sqrt(2.0 * alpha) / N1                      # alpha_x = tau^2 / (2 h1^2) with c = 1
    shape = (N2 - 1, N1 - 1)
    phi, psi, s = (rng.uniform(-1, 1, shape) for _ in range(3))
    c = rng.uniform(0.8, 1.0, 2 * M + 1)
    g = rng.uniform(-1, 1, 2 * M)
    # fp32 away from the configs' alpha <= 1: the systems' condition number (gamma + 4 alpha) / gamma bounds the rounding
    # of each solve, ~ cond * 6e-8 per half-step
    tol32 = max(1e-4, 12 * (2.0 + 4.0 * alpha * (N2 / N1) ** 2) / 2.0 * 6e-8 * 4)
    for dtype, tol in (("f64", 1e-11), ("f32", tol32)):
        w = W.Workload("rand", N1, N2, 1.0, tau, M, dtype, phi, psi, c, s=s, g_half=g)
        npdt = np.float64 if dtype == "f64" else np.float32
        cast = lambda a: a.astype(npdt).astype(np.float64)
        r = oracle.solve(N1, N2, 1.0, tau, M, cast(phi), cast(psi), c_half=c, s=cast(s), g_half=g)
        u, info = gpu(w)
        assert info["solver_x"] == B.SOLVER_LINE and info["solver_y"] == B.SOLVER_LINE and info["launches"] == 1
        assert relerr(u, r) <= tol, (dtype, relerr(u, r))
        r1 = oracle.solve(N1, N2, 1.0, tau, M, cast(phi), cast(psi), c_half=c, s=cast(s), g_half=g, scheme=1)
        u1, info = gpu1(w)
        assert info["solver_x"] == B.SOLVER_LINE
        assert relerr(u1, r1) <= tol, (dtype, "scheme 1", relerr(u1, r1))


def test_line_kernel_run_in_pieces_checkpoint_and_limits():
    w = W.cfg2(N=256, M=40)
    src = W.cfg3(N=256, M=40)
    w.s, w.g_half = src.s, W.ricker(W.half_times(w.tau, 2 * w.M) + 0.058)
    h = B.from_workload(w)
    try:
        h.run(w.M)
        a = h.get()
        assert h.info("line_launches") == 1 and h.info("graph_launches") == 0 and h.info("plain_sweeps") == 0
        h.set_initial(w.phi)
        for part in (1, 2, 0, 7, 13, 17):
            h.run(part)
        assert h.steps_done() == w.M
        b = h.get()
        h.set_initial(w.phi)
        h.run(11)
        prev, cur = h.get_prev(), h.get()
    finally:
        h.close()
    assert np.array_equal(a, b)                     # one launch of 40 steps == six launches
    assert relerr(a, ref(w)) <= 1e-10
    h = B.Wave2D(w.N1, w.N2, w.l, w.tau, w.M, w.dtype)
    try:
        h.set_speed(w.c_half)
        h.set_source(w.s, w.g_half)
        h.set_state(11, prev, cur)
        h.run(w.M - 11)
        assert np.array_equal(h.get(), a)           # resume from a checkpoint: the device step counter follows set_state
    finally:
        h.close()
    u, info = gpu(w, solver=B.SOLVER_STREAM)         # the streamed kernels on the same grid agree to rounding
    assert info["solver_x"] == B.SOLVER_STREAM and relerr(u, a) <= 1e-12
    big = W.cfg2(N=258, M=2)
    with pytest.raises(B.Wave2DError) as e:
        gpu(big, solver=B.SOLVER_LINE)
    assert e.value.status == -5


# ---- the exact whole-line solvers (solver EXACT, exact.cuh): block-wide scan, any tau / h, lines up to 16384 ----------
@pytest.mark.parametrize("N1,N2", [(4096, 24), (24, 4096), (16384, 20), (20, 16384), (1024, 520), (520, 1024),
                                   (4097, 37), (37, 4097), (8200, 18), (18, 8200)])
@pytest.mark.parametrize("alpha", [0.5, 50.0, 128.0])
def test_exact_solver_long_lines_any_tau(N1, N2, alpha):
    """parity of the whole-line solver at n in {4095, 16383, ...} and alpha in {0.5, 50, 128}
    (alpha = 128 is tau = 16 h, rho = 0.88: the streamed kernels refuse).  One segment per line (n <= 4096), several
    segments with y parked in shared memory (n = 8199, 16383), several rows per CTA (n = 1023: 4 warps per line),
    strips of 16 .. 1 columns in y.  Both dtypes, both schemes."""
    M = 3
    rng = np.random.default_rng(N1 * 7 + N2 + int(alpha))
    tau = np.sqrt(2.0 * alpha) / max(N1, N2)             # alpha along the long direction (c = 1)
    shape = (N2 - 1, N1 - 1)
    phi, psi, s = (rng.uniform(-1, 1, shape) for _ in range(3))
    c = rng.uniform(0.8, 1.0, 2 * M + 1)
    g = rng.uniform(-1, 1, 2 * M)
    for dtype, tol in (("f64", 1e-11), ("f32", max(1e-4, 12 * (1.0 + 2.0 * alpha) * 6e-8 * 4))):
        w = W.Workload("rand", N1, N2, 1.0, tau, M, dtype, phi, psi, c, s=s, g_half=g)
        npdt = np.float64 if dtype == "f64" else np.float32
        cast = lambda a: a.astype(npdt).astype(np.float64)
        r = oracle.solve(N1, N2, 1.0, tau, M, cast(phi), cast(psi), c_half=c, s=cast(s), g_half=g)
        u, info = gpu(w, solver=B.SOLVER_EXACT)
        assert info["solver_x"] == B.SOLVER_EXACT and info["solver_y"] == B.SOLVER_EXACT
        assert info["launches"] == 2 * M + 2             # one kernel per sweep; M = 3 steps = chunks of 2 + 1
        assert relerr(u, r) <= tol, (dtype, relerr(u, r))
        r1 = oracle.solve(N1, N2, 1.0, tau, M, cast(phi), cast(psi), c_half=c, s=cast(s), g_half=g, scheme=1)
        u1, _ = gpu1(w, solver=B.SOLVER_EXACT)
        assert relerr(u1, r1) <= tol, (dtype, "scheme 1", relerr(u1, r1))


@pytest.mark.parametrize("N1,N2", [(2, 2), (3, 9), (9, 8), (33, 18), (257, 40), (40, 257), (513, 24), (300, 1025),
                                   (4097, 12), (12, 4098)])
@pytest.mark.parametrize("alpha", [1e-6, 0.5, 5000.0])
def test_exact_solver_both_ends_repaired_at_extreme_alpha(N1, N2, alpha):
    """The Toeplitz lines of solver EXACT run the stationary recurrences on the padded line and repair both ends with
    A rho^(p+1) + B rho^(n-p) (exact.cuh, Ends).  rho = 5e-7 (alpha = 1e-6: the repair vanishes after one point) up to
    rho = 0.986 (alpha = 5000, tau = 100 h: both modes span the whole line, and rho^(n+1) couples the two ends on the
    short lines); lines that end exactly on the padded length (n = 256, 512, 4096: no x''_n) and one point beyond it."""
    M = 3
    rng = np.random.default_rng(N1 * 11 + N2)
    tau = np.sqrt(2.0 * alpha) / max(N1, N2)
    shape = (N2 - 1, N1 - 1)
    phi, psi, s = (rng.uniform(-1, 1, shape) for _ in range(3))
    c = rng.uniform(0.8, 1.2, 2 * M + 1)
    g = rng.uniform(-1, 1, 2 * M)
    w = W.Workload("rand", N1, N2, 1.0, tau, M, "f64", phi, psi, c, s=s, g_half=g)
    u, info = gpu(w, solver=B.SOLVER_EXACT)
    assert info["solver_x"] == B.SOLVER_EXACT and info["solver_y"] == B.SOLVER_EXACT
    assert relerr(u, ref(w)) <= 1e-11


def test_exact_solver_full_grid_tau_16h():
    """tau = 16 h on the 4095^2 grid (alpha = 128): AUTO picks the exact solvers; a few steps against the oracle."""
    M = 6
    w = W.cfg3(N=4096, M=M)
    w.tau = 16.0 / 4096
    w.phi = W.cfg2(N=4096, M=1).phi
    w.g_half = W.ricker(W.half_times(w.tau, 2 * M) + 0.058)
    r = ref(w)
    u, info = gpu_info(w, ("strip_y", "grid_x", "grid_y"))
    assert info["solver_x"] == B.SOLVER_EXACT and info["solver_y"] == B.SOLVER_EXACT
    assert info["strip_y"] == 4                           # 4 columns x 4095 rows x (9/8) x 8 B = 147 KB on chip
    assert relerr(u, r) <= 1e-10


# ---- variable speed c(t) cs(x,y): per-line pivots by a scan of linear-fractional maps -------------
def _speed_field(rng, shape, lo=0.4, hi=2.2):
    """Smooth + rough positive field: a few random Fourier modes plus point noise."""
    n2, n1 = shape
    y = np.linspace(0, 1, n2)[:, None]
    x = np.linspace(0, 1, n1)[None, :]
    f = 1.0 + 0.4 * np.sin(2 * np.pi * x * rng.integers(1, 4)) * np.cos(np.pi * y * rng.integers(1, 4)) + 0.3 * x - 0.2 * y
    f = f + 0.15 * rng.uniform(-1, 1, shape)
    return np.clip(f, lo, hi)


def gpu_var(w, cs, **opts):
    h = B.Wave2D(w.N1, w.N2, w.l, w.tau, w.M, w.dtype)
    try:
        for k, v in opts.items():
            h.set_option(k, v)
        npdt = np.float64 if w.dtype == "f64" else np.float32
        h.set_speed(w.c_half)
        h.set_speed_field(cs.astype(npdt))
        if w.s is not None:
            h.set_source(w.s.astype(npdt), w.g_half)
        h.set_initial(w.phi.astype(npdt), None if w.psi is None else w.psi.astype(npdt))
        h.run(w.M)
        u = h.get()
        info = {k: h.info(k) for k in ("solver_x", "solver_y", "launches", "strip_y")}
    finally:
        h.close()
    return u, info


@pytest.mark.parametrize("N1,N2", [(2, 2), (3, 9), (9, 3), (17, 16), (33, 34), (130, 66), (257, 40), (40, 257), (300, 260),
                                   (1030, 270), (270, 1030), (4096, 24), (24, 4096), (2050, 2050)])
@pytest.mark.parametrize("ratio", [0.9, 3.0, 16.0])
def test_variable_speed_matches_oracle(N1, N2, ratio):
    """Random positive speed field, time-varying c(t), source, psi != 0; tau = 0.9 h, 3 h and 16 h (the pivot scan is exact
    for any tau).  Element by element against the oracle's variable-speed mode; fp64 and fp32."""
    M = 5 if max(N1, N2) < 2000 else 3
    rng = np.random.default_rng(N1 * 13 + N2 + int(ratio))
    tau = ratio / max(N1, N2)
    shape = (N2 - 1, N1 - 1)
    phi, psi, s = (rng.uniform(-1, 1, shape) for _ in range(3))
    c = rng.uniform(0.7, 1.3, 2 * M + 1)
    g = rng.uniform(-1, 1, 2 * M)
    cs = _speed_field(rng, shape)
    alpha = 0.5 * ratio ** 2 * 1.3 * 2.2 * (max(N1, N2) / min(N1, N2)) ** 0       # along the long direction
    for dtype, tol in (("f64", 1e-10), ("f32", max(1e-4, 12 * (1.0 + 2.0 * alpha) * 6e-8 * 4))):
        w = W.Workload("var", N1, N2, 1.0, tau, M, dtype, phi, psi, c, s=s, g_half=g)
        npdt = np.float64 if dtype == "f64" else np.float32
        cast = lambda a: a.astype(npdt).astype(np.float64)
        r = oracle.solve(N1, N2, 1.0, tau, M, cast(phi), cast(psi), c_half=c, s=cast(s), g_half=g, cs=cast(cs))
        u, info = gpu_var(w, cs)
        assert info["solver_x"] == B.SOLVER_EXACT and info["solver_y"] == B.SOLVER_EXACT
        assert info["launches"] == 2 * M + 2      # one kernel per sweep; two chunks (2 + 1 or 4 + 1 steps)
        assert relerr(u, r) <= tol, (dtype, relerr(u, r))


def test_variable_speed_constant_field_and_state_machine():
    w = W.cfg2(N=300, M=12)
    ones = np.full(w.phi.shape, 1.25)
    u, _ = gpu_var(w, ones)
    w2 = W.cfg2(N=300, M=12)
    w2.c_half = 1.25 * w.c_half
    v, info = gpu(w2, solver=B.SOLVER_EXACT)
    assert relerr(u, v) <= 1e-12                       # cs == const is the Toeplitz problem with c scaled
    h = B.Wave2D(32, 32, 1.0, 0.01, 4)
    try:
        with pytest.raises(B.Wave2DError) as e:
            h.set_speed_field(np.zeros((31, 31)))      # must be positive
        assert e.value.status == -1
        h.set_speed_field(np.ones((31, 31)))
        with pytest.raises(B.Wave2DError) as e:
            h.set_option("scheme", 1)                  # split scheme only
        assert e.value.status == -5
        h.set_option("solver", B.SOLVER_STREAM)
        h.set_initial(np.ones((31, 31)))
        with pytest.raises(B.Wave2DError) as e:
            h.run(1)                                   # the streamed kernels assume Toeplitz systems
        assert e.value.status == -5
        h.set_speed_field(None)                        # back to c = c(t)
        h.run(1)
        with pytest.raises(B.Wave2DError) as e:
            h.set_speed_field(np.ones((31, 31)))       # not after the first run
        assert e.value.status == -2
    finally:
        h.close()
    big = B.Wave2D(4200, 16, 1.0, 0.01, 2)
    try:
        big.set_speed_field(np.ones((15, 4199)))
        big.set_initial(np.ones((15, 4199)))
        with pytest.raises(B.Wave2DError) as e:
            big.run(1)                                 # lines of more than 4096 unknowns: not yet
        assert e.value.status == -5
    finally:
        big.close()


def test_variable_speed_full_grid_4095():
    M = 4
    w = W.cfg3(N=4096, M=M)
    w.phi = W.cfg2(N=4096, M=1).phi
    w.g_half = W.ricker(W.half_times(w.tau, 2 * M) + 0.058)
    cs = _speed_field(np.random.default_rng(5), w.phi.shape)
    r = oracle.solve(w.N1, w.N2, w.l, w.tau, M, w.phi, None, c_half=w.c_half, s=w.s, g_half=w.g_half, cs=cs)
    u, info = gpu_var(w, cs)
    assert info["strip_y"] == 2                          # r and a_p of 2 columns x 4095 rows on chip
    assert relerr(u, r) <= 1e-10


# ---- SURVEY.md 8f NEXT-4, the rest: the weight sigma (Listing 1: sigma = 1) and the second-order start of (2.8) ----------
@pytest.mark.parametrize("sigma,gamma", [(1.0, 1.0), (1.0, 2.0), (0.75, 2.0)])
@pytest.mark.parametrize("name,w", [("cfg1", W.cfg1()), ("cfg2_N700", W.cfg2(N=700, M=30)),
                                    ("cfg3_N1000", W.cfg3(N=1000, M=250)), ("cfg4_1030x270", W.cfg4(N1=1030, N2=270, M=24))],
                         ids=["cfg1", "cfg2_N700", "cfg3_N1000", "cfg4_1030x270"])
def test_sigma_weight_matches_oracle_on_every_solver_path(name, w, sigma, gamma):
    """Option "sigma": sigma = 1, gamma = 1 is the system Listing 1 prints.  The weights enter through
    the per-half-step scalars only, so every kernel family must agree with the oracle's sigma mode."""
    r = oracle.solve(w.N1, w.N2, w.l, w.tau, w.M, w.phi, w.psi, c_half=w.c_half, s=w.s, g_half=w.g_half, gamma=gamma,
                     sigma=sigma)
    for opts in ({}, {"solver": B.SOLVER_STREAM}, {"solver": B.SOLVER_EXACT}):
        u, info = gpu(w, gamma=gamma, sigma=sigma, **opts)
        assert relerr(u, r) <= 1e-10, (opts, relerr(u, r))
    assert relerr(r, ref(w)) > 1e-4      # and sigma changes the answer


def test_sigma_with_variable_speed_and_fp32():
    w = W.cfg4(N1=300, N2=200, M=20, dtype="f32")
    rng = np.random.default_rng(5)
    cs = rng.uniform(0.5, 1.5, (w.n2, w.n1)).astype(np.float32)
    r = oracle.solve(w.N1, w.N2, w.l, w.tau, w.M, w.phi, w.psi, c_half=w.c_half, cs=cs.astype(np.float64), sigma=1.0)
    h = B.Wave2D(w.N1, w.N2, w.l, w.tau, w.M, "f32")
    try:
        h.set_option("sigma", 1.0)
        h.set_speed(w.c_half)
        h.set_speed_field(cs)
        h.set_initial(w.phi.astype(np.float32))
        h.run(w.M)
        u = h.get()
    finally:
        h.close()
    assert relerr(u, r) <= 1e-4


@pytest.mark.parametrize("N1,N2", [(96, 80), (700, 300), (1500, 1200)])
def test_second_order_start_of_the_factored_scheme(N1, N2):
    """Option "start" = 2 (scheme 1): u^1 = phi + tau psi + tau^2/2 (c^0 Lap_h phi + g^0 s); small-grid kernel, streamed
    kernels and exact solvers; the term is added at the first run."""
    M = 12
    rng = np.random.default_rng(N1 + N2)
    w = W.cfg2(N=N1, M=M)
    shape = (N2 - 1, N1 - 1)
    yy, xx = np.meshgrid(np.arange(1, N2) / N2, np.arange(1, N1) / N1, indexing="ij")
    phi = np.exp(-((xx - 0.4) ** 2 + (yy - 0.55) ** 2) / 0.02)
    psi = np.sin(3 * np.pi * xx) * np.sin(2 * np.pi * yy)
    s = np.zeros(shape)
    s[N2 // 3:N2 // 3 + 20, N1 // 4:N1 // 4 + 30] = rng.uniform(-1, 1, (20, 30))
    g = np.cos(np.arange(2 * M) * 0.2) + 0.5
    tau = 1.0 / max(N1, N2)
    c = w.c_half
    r = oracle.solve(N1, N2, 1.0, tau, M, phi, psi, c_half=c, s=s, g_half=g, scheme=1, start=2)
    r1 = oracle.solve(N1, N2, 1.0, tau, M, phi, psi, c_half=c, s=s, g_half=g, scheme=1)
    assert relerr(r1, r) > 1e-6
    for opts in ({}, {"solver": B.SOLVER_EXACT}):
        h = B.Wave2D(N1, N2, 1.0, tau, M, "f64")
        try:
            h.set_option("scheme", 1)
            h.set_option("start", 2)
            for k, v in opts.items():
                h.set_option(k, v)
            h.set_initial(phi, psi)                      # before the speed and the source: the term waits for the run
            h.set_speed(c)
            h.set_source(s, g)
            np.testing.assert_allclose(h.get(), phi + tau * psi, rtol=0, atol=1e-15)
            h.run(M - 1)
            u = h.get()
        finally:
            h.close()
        assert relerr(u, r) <= 1e-10, (opts, relerr(u, r))


def test_sigma_and_start_are_refused_where_they_do_not_apply():
    h = B.Wave2D(64, 64, 1.0, 0.01, 4, "f64")
    try:
        h.set_option("start", 2)
        h.set_initial(np.ones((63, 63)))
        with pytest.raises(B.Wave2DError) as e:
            h.run(1)
        assert e.value.status == -5
    finally:
        h.close()
    h = B.Wave2D(64, 64, 1.0, 0.01, 4, "f64")
    try:
        h.set_option("scheme", 1)
        with pytest.raises(B.Wave2DError) as e:
            h.set_option("sigma", 1.0)
        assert e.value.status == -5
        with pytest.raises(B.Wave2DError):
            h.set_option("sigma", 0.0)
    finally:
        h.close()


# ---- header = code: what a failed call leaves behind, the limits the error texts quote, start = 2 at M = 1 ----
def test_a_rejected_speed_field_leaves_the_accepted_one_in_force():
    """wave2d_set_speed_field checks the new field before it touches the handle: after ERR_ARG the run still uses the
    field that was accepted before (it used to fall back to c = c(t) silently)."""
    w = W.cfg2(N=200, M=6)
    cs = _speed_field(np.random.default_rng(77), w.phi.shape)
    r = oracle.solve(w.N1, w.N2, w.l, w.tau, w.M, w.phi, None, c_half=w.c_half, cs=cs)
    h = B.from_workload(w)
    try:
        h.set_speed_field(cs)
        bad = cs.copy()
        bad[17, 23] = 0.0
        with pytest.raises(B.Wave2DError) as e:
            h.set_speed_field(bad)
        assert e.value.status == -1
        h.run(w.M)
        u = h.get()
        assert h.info("solver_x") == B.SOLVER_EXACT      # the variable-speed path, not the Toeplitz one
    finally:
        h.close()
    assert relerr(u, r) <= 1e-10
    assert relerr(u, ref(w)) > 1e-3                      # and it differs from c = c(t)


@pytest.mark.parametrize("dtype,N1,N2,text", [("f64", 24578, 3, "24576 fp64"), ("f32", 49154, 3, "49152 fp32"),
                                              ("f64", 3, 22754, "22752 fp64"), ("f32", 3, 45506, "45504 fp32")])
def test_exact_solver_limits_are_the_ones_the_header_states(dtype, N1, N2, text):
    """One unknown more than include/wave2d.h's limit for WAVE2D_SOLVER_EXACT is refused at the first plan, with the limit
    of THIS dtype in the message; the limit itself is accepted."""
    for extra, ok in ((0, False), (-1, True)):
        n1, n2 = (N1 + extra, N2) if N1 > N2 else (N1, N2 + extra)
        h = B.Wave2D(n1, n2, 1.0, 1e-3, 2, dtype)
        try:
            h.set_option("solver", B.SOLVER_EXACT)
            h.set_initial(np.ones((n2 - 1, n1 - 1), dtype=np.float64 if dtype == "f64" else np.float32))
            if ok:
                h.run(1)
                assert np.isfinite(h.get()).all()
            else:
                with pytest.raises(B.Wave2DError) as e:
                    h.run(0)
                assert e.value.status == -5 and text in str(e.value), str(e.value)
        finally:
            h.close()


def test_second_order_start_is_not_applied_before_a_step_is_run():
    """include/wave2d.h, option "start": the tau^2/2 term is added by the first wave2d_run with steps > 0.  With M = 1 no
    step can be run, so wave2d_get is the first-order phi + tau psi -- on both sides (the oracle adds it at the same place)."""
    N, tau = 48, 0.02
    rng = np.random.default_rng(5)
    phi, psi = rng.uniform(-1, 1, (N - 1, N - 1)), rng.uniform(-1, 1, (N - 1, N - 1))
    r = oracle.solve(N, N, 1.0, tau, 1, phi, psi, scheme=1, start=2)
    np.testing.assert_allclose(r, phi + tau * psi, rtol=0, atol=1e-15)
    h = B.Wave2D(N, N, 1.0, tau, 1, "f64")
    try:
        h.set_option("scheme", 1)
        h.set_option("start", 2)
        h.set_initial(phi, psi)
        h.run(0)
        assert h.steps_done() == 1
        np.testing.assert_allclose(h.get(), r, rtol=0, atol=1e-15)
        with pytest.raises(B.Wave2DError) as e:
            h.run(1)
        assert e.value.status == -6
    finally:
        h.close()


# ---- SURVEY.md 8b "Memory": the ring of time levels in a block the caller allocated (wave2d_set_workspace) ---------------------
@pytest.mark.parametrize("name,w,scheme", [("cfg2_N700", W.cfg2(N=700, M=20), 0), ("cfg3_N300", W.cfg3(N=300, M=30), 0),
                                           ("cfg1", W.cfg1(), 0), ("cfg2_N700_scheme1", W.cfg2(N=700, M=20), 1),
                                           ("cfg4_f32", W.cfg4(N1=1030, N2=270, M=12, dtype="f32"), 0)],
                         ids=["cfg2_N700", "cfg3_N300", "cfg1", "cfg2_N700_scheme1", "cfg4_f32"])
def test_workspace_owned_by_the_caller(name, w, scheme):
    """A torch allocation backs the time levels: same result, bit for bit, as the handle that allocates its own; the
    handle then owns less than one field of device memory; the block can be dropped only after the handle."""
    import torch
    npdt = np.float64 if w.dtype == "f64" else np.float32

    def run(with_block):
        h = B.Wave2D(w.N1, w.N2, w.l, w.tau, w.M, w.dtype)
        try:
            if scheme:
                h.set_option("scheme", 1)
            own = h.info("device_bytes")
            if with_block:
                need = h.workspace_bytes()
                field = h.info("pitch") * w.n2 * (8 if w.dtype == "f64" else 4)
                assert (4 if scheme else 3) * field <= need <= (4 if scheme else 3) * (field + 255)
                block = torch.full((need,), 0x7f, dtype=torch.uint8, device="cuda")     # garbage: the library clears it
                h.set_workspace(block)
                assert h.info("device_bytes") < min(field, own - 2 * field)
            h.set_speed(w.c_half)
            if w.s is not None:
                h.set_source(w.s.astype(npdt), w.g_half)
            h.set_initial(w.phi.astype(npdt), None if w.psi is None else w.psi.astype(npdt))
            h.run(w.M - h.steps_done())
            return h.get()
        finally:
            h.close()

    u_own, u_ws = run(False), run(True)
    assert np.array_equal(u_own, u_ws)
    r = oracle.solve(w.N1, w.N2, w.l, w.tau, w.M, w.phi, w.psi, c_half=w.c_half, s=w.s, g_half=w.g_half, scheme=scheme)
    assert relerr(u_ws, r) <= TOL[w.dtype]


def test_workspace_state_machine():
    import torch
    h = B.Wave2D(200, 120, 1.0, 0.004, 6)
    try:
        need = h.workspace_bytes()
        block = torch.empty((need + 256,), dtype=torch.uint8, device="cuda")
        for bad in (block[:need - 1], block[1:need + 1], torch.empty((need,), dtype=torch.uint8)):
            with pytest.raises(B.Wave2DError) as e:      # too small; not 256-byte aligned; host memory
                h.set_workspace(bad)
            assert e.value.status == -1
        h.set_workspace(block)
        with pytest.raises(B.Wave2DError) as e:
            h.set_option("scheme", 1)                    # the fourth field is not there: choose the scheme first
        assert e.value.status == -2
        h.set_workspace(None)                            # back to memory of its own ...
        h.set_option("scheme", 1)                        # ... where the fourth field can be allocated
        assert h.workspace_bytes() == need // 3 * 4
        h.set_option("scheme", 0)
        h.set_workspace(block)
        phi = np.random.default_rng(1).uniform(-1, 1, (119, 199))
        h.set_initial(phi)
        with pytest.raises(B.Wave2DError) as e:
            h.set_workspace(None)                        # not once the ring holds data
        assert e.value.status == -2
        h.run(6)
        u = h.get()
    finally:
        h.close()
    assert relerr(u, oracle.solve(200, 120, 1.0, 0.004, 6, phi)) <= 1e-10
