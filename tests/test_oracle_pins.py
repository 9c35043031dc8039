"""Pins for the CPU oracle (oracle/wave2d_oracle.c) against things other than itself.

Each test names the passage of the paper / SURVEY.md pin it checks.  A plausible mistake in the oracle
(dropped term, wrong sign or index, transposed operand, wrong time level of c or g, swapped sweeps)
fails at least one of them.
"""
import math

import numpy as np
import pytest

from oracle import oracle
from tests.modal import modal_amplitudes

RNG = np.random.default_rng(12345)


# ------------------------------------------------------------------------------------------ pin 1
@pytest.mark.parametrize("n", [1, 2, 3, 7, 8, 33, 64])
def test_thomas_matches_dense_lu(n):
    """Line solve vs dense LU of the n x n matrix (SURVEY 8c pin 1), general (non-Toeplitz) coefficients."""
    a = -RNG.uniform(0.1, 1.0, n)
    c = -RNG.uniform(0.1, 1.0, n)
    b = 2.0 + RNG.uniform(0.0, 1.0, n) - a - c          # strictly diagonally dominant
    f = RNG.standard_normal(n)
    T = np.diag(b) + np.diag(a[1:], -1) + np.diag(c[:-1], 1)
    x = oracle.thomas(a, b, c, f)
    np.testing.assert_allclose(x, np.linalg.solve(T, f), rtol=0, atol=1e-14 * np.abs(f).max() * 10)
    assert np.abs(T @ x - f).max() <= 1e-13 * np.abs(f).max()


@pytest.mark.parametrize("n,alpha", [(127, 0.5), (1023, 1.0), (1000, 50.0), (16383, 0.125)])
def test_thomas_residual_toeplitz(n, alpha):
    """||T x - r|| / ||r|| < 1e-13 for the scheme's own matrices tridiag(-a, gamma + 2a, -a) (north_star)."""
    f = RNG.standard_normal(n)
    a = np.full(n, -alpha)
    b = np.full(n, 2.0 + 2 * alpha)
    x = oracle.thomas(a, b, a, f)
    xp = np.pad(x, 1)
    res = -alpha * xp[:-2] + (2.0 + 2 * alpha) * x - alpha * xp[2:] - f
    assert np.abs(res).max() <= 1e-13 * np.abs(f).max()


# ------------------------------------------------------------------------------------------ pin 2
def _K(n):
    return 2.0 * np.eye(n) - np.eye(n, k=1) - np.eye(n, k=-1)      # -(undivided second difference), zero ghosts


def _dense_reference(N1, N2, l, tau, M, phi, psi, s, c_half, g_half, gamma, kappa, steps):
    """Brute force: assemble I (x) T_x resp. T_y (x) I densely and solve by LU, half-step by half-step."""
    n1, n2 = N1 - 1, N2 - 1
    I1, I2 = np.eye(n1), np.eye(n2)
    Kx = np.kron(I2, _K(n1))       # acts along i (fastest index)
    Ky = np.kron(_K(n2), I1)       # acts along j
    w_prev = (phi - 0.5 * tau * psi).reshape(-1)
    w_cur = phi.reshape(-1).copy()
    for n in range(2 * steps):
        K, hd = (Kx, l / N1) if n % 2 == 0 else (Ky, l / N2)
        ap = tau ** 2 * c_half[n + 1] / (2 * hd ** 2)
        am = tau ** 2 * c_half[max(n - 1, 0)] / (2 * hd ** 2)
        A = gamma * np.eye(n1 * n2) + ap * K
        rhs = gamma * (2 * w_cur - w_prev) - am * (K @ w_prev) + kappa * tau ** 2 * g_half[n] * s.reshape(-1)
        w_prev, w_cur = w_cur, np.linalg.solve(A, rhs)
    return w_cur.reshape(n2, n1), w_prev.reshape(n2, n1)


@pytest.mark.parametrize("N1,N2", [(8, 8), (9, 6), (3, 7), (2, 2)])
@pytest.mark.parametrize("gamma,kappa", [(2.0, 0.5), (1.0, 1.0)])
def test_half_steps_match_dense_kronecker_lu(N1, N2, gamma, kappa):
    """(2.11)/(2.12) step by step vs a dense Kronecker solve (SURVEY 8c pin 2): random phi, psi, s, c(t), g(t)."""
    n1, n2, M, l = N1 - 1, N2 - 1, 10, 1.3
    tau = 0.9 * l / max(N1, N2)
    phi = RNG.standard_normal((n2, n1))
    psi = RNG.standard_normal((n2, n1))
    s = RNG.standard_normal((n2, n1))
    c_half = RNG.uniform(0.5, 2.0, 2 * M + 1)
    g_half = RNG.standard_normal(2 * M)
    ref, ref_prev = _dense_reference(N1, N2, l, tau, M, phi, psi, s, c_half, g_half, gamma, kappa, M)
    o = oracle.Wave2DOracle(N1, N2, l, tau, M)
    o.set_option("gamma", gamma)
    o.set_option("kappa", kappa)
    o.set_speed(c_half)
    o.set_source(s, g_half)
    o.set_initial(phi, psi)
    o.run(M)
    scale = max(np.abs(ref).max(), 1.0)
    assert np.abs(o.get() - ref).max() <= 5e-14 * scale
    assert np.abs(o.get_prev() - ref_prev).max() <= 5e-14 * scale


# ------------------------------------------------------------------------------------------ pin 3
def _mode(N1, N2, m, n):
    x = np.arange(1, N1) / N1
    y = np.arange(1, N2) / N2
    return np.outer(np.sin(n * np.pi * y), np.sin(m * np.pi * x))


def test_modal_recurrence_general():
    """Full 2D run vs the exact discrete modal closed form: N1 != N2, tau = 1.3 min h, c(t) varying, psi != 0."""
    N1, N2, M, l = 48, 20, 40, 1.0
    tau = 1.3 * min(l / N1, l / N2)
    t = np.arange(2 * M + 1) * tau / 2
    c_half = 1.0 + 0.4 * np.sin(3.0 * t) + 0.1 * t
    modes = [(1, 1, 1.0, 0.3), (3, 5, -0.7, 2.0), (7, 2, 0.25, -1.0)]
    phi = sum(A * _mode(N1, N2, m, n) for m, n, A, B in modes)
    psi = sum(B * _mode(N1, N2, m, n) for m, n, A, B in modes)
    u = oracle.solve(N1, N2, l, tau, M, phi, psi, c_half=c_half)
    ref = sum(modal_amplitudes(N1, N2, l, tau, m, n, A, B, c_half, 2 * M)[-1] * _mode(N1, N2, m, n)
              for m, n, A, B in modes)
    assert np.abs(u - ref).max() <= 1e-13 * np.abs(ref).max()


def test_modal_recurrence_with_source():
    """Source that is an eigenmode, time-varying g (pins the g time level of reading A8 and kappa)."""
    N1, N2, M, l = 24, 36, 30, 2.0
    tau = 0.8 * min(l / N1, l / N2)
    t = np.arange(2 * M + 1) * tau / 2
    c_half = 1.5 + 0.5 * np.cos(2.0 * t)
    g_half = np.sin(5.0 * t[:-1]) + 0.2
    m, n, S = 2, 3, 0.75
    x = np.arange(1, N1) * l / N1
    y = np.arange(1, N2) * l / N2
    mode = np.outer(np.sin(n * np.pi * y / l), np.sin(m * np.pi * x / l))
    u = oracle.solve(N1, N2, l, tau, M, np.zeros_like(mode), None, c_half=c_half, s=S * mode, g_half=g_half)
    hist = modal_amplitudes(N1, N2, l, tau, m, n, 0.0, 0.0, c_half, 2 * M, S=S, g_half=g_half)
    a = hist[-1]
    assert abs(a) > 1e-4
    assert np.abs(u - a * mode).max() <= 1e-13 * max(abs(v) for v in hist)


def test_cfg1_modal_amplitude_golden():
    """Config 1 (N=128, tau=h/2, M=100): the (1,1) amplitude after 200 half-steps.

    tests/golden/cfg1_modal.txt was written by tests/golden/make_golden.py from the oracle's full 2D run;
    here it must agree with the independent scalar recurrence, and differ from the PDE's cos(pi sqrt2 T)
    only by the O(tau) error the paper claims.
    """
    import os
    N, M = 128, 100
    tau = 0.5 / N
    a = modal_amplitudes(N, N, 1.0, tau, 1, 1, 1.0, 0.0, np.ones(2 * M + 1), 2 * M)[-1]
    path = os.path.join(os.path.dirname(__file__), "golden", "cfg1_modal.txt")
    gold = float([ln for ln in open(path) if not ln.startswith("#")][0].split()[0])
    # Rounding noise of a marginally stable three-level recurrence is amplified by 1/theta ~ 2/(omega tau)
    # ~ 115 per injected ulp at this config, so the 2D run (O(10) roundings per point per half-step) and the
    # scalar recurrence agree to ~1e-12, not 1e-15; 1e-11 still catches any O(tau^2) modelling slip (1.5e-5).
    assert abs(a - gold) <= 1e-11
    T = M * tau
    assert abs(a - math.cos(math.pi * math.sqrt(2.0) * T)) < 1.5 * tau      # 4.2e-3 expected
    phi = _mode(N, N, 1, 1)
    u = oracle.solve(N, N, 1.0, tau, M, phi)
    assert np.abs(u - a * phi).max() <= 1e-11


# ------------------------------------------------------------------------------------------ pin 4
def _pde_error(N, T=0.5, gamma=None, kappa=None, c=1.0):
    tau = 1.0 / N
    M = int(round(T / tau))
    phi = _mode(N, N, 1, 1)
    u = oracle.solve(N, N, 1.0, tau, M, phi, c_half=[c], gamma=gamma, kappa=kappa)
    exact = phi * math.cos(math.pi * math.sqrt(2.0 * c) * M * tau)
    return np.abs(u - exact).max()


def test_pde_standing_wave_order_one():
    """u = sin(pi x) sin(pi y) cos(pi sqrt(2c) t) (north_star); observed order ~1 = O(tau + h^2)."""
    errs = [_pde_error(N) for N in (32, 64, 128, 256)]
    # survey-time probe values: 2.5e-2, 1.3e-2, 6.8e-3, 3.4e-3
    for e, ref in zip(errs, (2.5e-2, 1.3e-2, 6.8e-3, 3.4e-3)):
        assert 0.8 * ref < e < 1.2 * ref
    orders = [math.log2(errs[i] / errs[i + 1]) for i in range(3)]
    assert all(0.85 < o < 1.1 for o in orders), orders
    assert _pde_error(64, c=2.0) < 0.05


def test_literal_scheme_solves_a_different_pde():
    """Reading A2: with gamma = kappa = 1 (the scheme exactly as printed) the (1,1) mode oscillates like
    cos(2 pi t), i.e. u_tt = 2 c Lap u, not cos(pi sqrt2 t)."""
    N, T = 128, 0.390625
    tau = 0.5 / N
    M = int(round(T / tau))
    phi = _mode(N, N, 1, 1)
    u = oracle.solve(N, N, 1.0, tau, M, phi, gamma=1.0, kappa=1.0)
    amp = u[N // 2 - 1, N // 2 - 1] / phi[N // 2 - 1, N // 2 - 1]
    assert abs(amp - math.cos(2 * math.pi * T)) < 0.01
    assert abs(amp - math.cos(math.pi * math.sqrt(2) * T)) > 0.5


# ------------------------------------------------------------------------------------------ pin 5
def test_forced_response_pins_kappa():
    """c = 1, phi = psi = 0, s = mode (1,1), g = 1: amplitude -> (1 - cos wT)/w^2, w^2 = 2 pi^2 (SURVEY pin 5)."""
    N, T = 256, 0.5
    tau = 1.0 / N
    M = int(round(T / tau))
    mode = _mode(N, N, 1, 1)
    u = oracle.solve(N, N, 1.0, tau, M, np.zeros_like(mode), s=mode)
    amp = u[N // 2 - 1, N // 2 - 1]
    w2 = 2 * math.pi ** 2
    exact = (1 - math.cos(math.sqrt(w2) * T)) / w2
    assert abs(amp - exact) < 0.005 * exact          # probe: 0.081520 vs 0.081346
    u2 = oracle.solve(N, N, 1.0, tau, M, np.zeros_like(mode), s=mode, kappa=1.0)
    assert abs(u2[N // 2 - 1, N // 2 - 1] / amp - 2.0) < 1e-12


def test_initial_velocity_first_order_start():
    """Reading A1: w_{-1} = phi - (tau/2) psi.  phi = 0, psi = mode: u(T) ~ sin(wT)/w (first order in tau)."""
    N, T = 128, 0.25
    tau = 1.0 / N
    M = int(round(T / tau))
    mode = _mode(N, N, 1, 1)
    o = oracle.Wave2DOracle(N, N, 1.0, tau, M)
    o.set_initial(np.zeros_like(mode), mode)
    np.testing.assert_allclose(o.get_prev(), -0.5 * tau * mode, rtol=0, atol=1e-18)
    np.testing.assert_array_equal(o.get(), np.zeros_like(mode))
    o.run(M)
    w = math.pi * math.sqrt(2.0)
    amp = o.get()[N // 2 - 1, N // 2 - 1]
    assert abs(amp - math.sin(w * T) / w) < 0.02 * abs(math.sin(w * T) / w) + 2 * tau


# ------------------------------------------------------------------------------------------ pin 6
def _random_problem(N1=40, N2=28, M=12):
    l = 1.0
    tau = 1.1 * min(l / N1, l / N2)
    t = np.arange(2 * M + 1) * tau / 2
    return dict(N1=N1, N2=N2, l=l, tau=tau, M=M, c_half=1.0 + 0.5 * np.sin(7 * t))


def test_linearity():
    p = _random_problem()
    n1, n2 = p["N1"] - 1, p["N2"] - 1
    a, b = RNG.standard_normal((n2, n1)), RNG.standard_normal((n2, n1))
    ua = oracle.solve(phi=a, **p)
    ub = oracle.solve(phi=b, **p)
    uc = oracle.solve(phi=2 * a - 3 * b, **p)
    assert np.abs(uc - (2 * ua - 3 * ub)).max() <= 1e-12 * np.abs(uc).max()


def test_reflection_symmetries_and_no_transpose_symmetry():
    p = _random_problem(N1=32, N2=32, M=16)
    a = RNG.standard_normal((31, 31))
    u = oracle.solve(phi=a, **p)
    ux = oracle.solve(phi=a[:, ::-1].copy(), **p)
    uy = oracle.solve(phi=a[::-1, :].copy(), **p)
    assert np.abs(ux[:, ::-1] - u).max() <= 1e-13 * np.abs(u).max()
    assert np.abs(uy[::-1, :] - u).max() <= 1e-13 * np.abs(u).max()
    # reading A9: x sweep first, so transposing the data does NOT transpose the result
    sym = a + a.T
    us = oracle.solve(phi=sym, **p)
    assert np.abs(us - us.T).max() > 1e-3 * np.abs(us).max()


def test_zero_in_zero_out_and_boundaries():
    p = _random_problem()
    z = np.zeros((p["N2"] - 1, p["N1"] - 1))
    assert np.all(oracle.solve(phi=z, **p) == 0.0)


def test_sweep_order_x_then_y():
    """First half-step is implicit in x: a field varying only in y is then NOT smoothed in y.
    With phi = phi(y) * sin(pi x) (an x-eigenmode), after ONE half-step the result is exactly
    2 gamma phi - (gamma + am mu) phi over (gamma + ap mu): a pure scalar multiple of phi, whatever phi(y) is."""
    N1, N2, l = 16, 12, 1.0
    tau = 0.05
    y = RNG.standard_normal(N2 - 1)
    x = np.sin(np.pi * np.arange(1, N1) / N1)
    phi = np.outer(y, x)
    h1 = l / N1
    ap = am = tau ** 2 / (2 * h1 ** 2)
    out = oracle.half_step(0, ap, am, 2.0, 0.0, phi, phi)
    mu = 4 * math.sin(math.pi / (2 * N1)) ** 2
    factor = (2 * 2.0 - (2.0 + am * mu)) / (2.0 + ap * mu)
    assert np.abs(out - factor * phi).max() <= 1e-14
    out_y = oracle.half_step(1, ap, am, 2.0, 0.0, phi, phi)
    assert np.abs(out_y - factor * phi).max() > 1e-3


def test_unconditional_stability_large_tau():
    """unconditionally stable.  tau = 64 h for 1000 steps stays bounded."""
    N, M = 32, 1000
    tau = 64.0 / N
    phi = RNG.uniform(-1, 1, (N - 1, N - 1))
    u = oracle.solve(N, N, 1.0, tau, M, phi)
    assert np.isfinite(u).all() and np.abs(u).max() < 50 * np.abs(phi).max()


def test_mode_orthogonality():
    N = 64
    tau = 1.0 / N
    phi = _mode(N, N, 3, 2)
    u = oracle.solve(N, N, 1.0, tau, 40, phi)
    amp = (u * phi).sum() / (phi * phi).sum()
    assert np.abs(u - amp * phi).max() <= 1e-13


# ------------------------------------------------------------------------------------------ API
def test_handle_state_machine_and_argument_checks():
    o = oracle.Wave2DOracle(8, 8, 1.0, 0.1, 3)
    with pytest.raises(oracle.OracleError):
        o.run(1)                                      # no initial data yet
    with pytest.raises(oracle.OracleError):
        o.set_speed(np.array([1.0, -1.0, 1, 1, 1, 1, 1]))   # c must be positive
    with pytest.raises(oracle.OracleError):
        o.set_speed(np.ones(4))                       # count must be 1 or 2M+1
    o.set_initial(np.ones((7, 7)))
    o.run(2)
    assert o.steps_done() == 2
    with pytest.raises(oracle.OracleError):
        o.run(2)                                      # beyond M
    with pytest.raises(oracle.OracleError):
        o.set_speed([2.0])                            # after first run
    o.set_initial(np.ones((7, 7)))                    # resets k
    assert o.steps_done() == 0
