"""Pins for the oracle's second scheme: the factorised form of the unsplit scheme (2.8) (
SURVEY.md 8f NEXT-2; oracle_factored_step) -- against dense linear algebra written out here, the modal closed
form (tests/modal.py), the unsplit scheme itself, the PDE, and symmetries.  A dropped term, a wrong sign, a wrong
time level of c or g, swapped h1/h2 or a transposed operand fails at least one."""
import math

import numpy as np
import pytest

from oracle import oracle
from tests.modal import modal_amplitudes_factored

RNG = np.random.default_rng(2468)


def _K(n):
    return 2.0 * np.eye(n) - np.eye(n, k=1) - np.eye(n, k=-1)      # -(undivided second difference), zero ghosts


def _dense_run(N1, N2, l, tau, phi, psi, s, c_half, g_half, K, factored=True):
    """Level k -> k+1 by dense LU of the Kronecker operators; factored=False solves the UNSPLIT (2.8)."""
    n1, n2 = N1 - 1, N2 - 1
    Kx, Ky = np.kron(np.eye(n2), _K(n1)), np.kron(_K(n2), np.eye(n1))
    I = np.eye(n1 * n2)
    h1, h2 = l / N1, l / N2
    u0, u1 = phi.reshape(-1), (phi + tau * psi).reshape(-1)
    for k in range(1, K):
        def op(c):
            ax, ay = tau ** 2 * c / (2 * h1 ** 2), tau ** 2 * c / (2 * h2 ** 2)
            return (I + ax * Kx) @ (I + ay * Ky) if factored else I + ax * Kx + ay * Ky
        rhs = 2 * u1 - op(c_half[2 * (k - 1)]) @ u0 + tau ** 2 * g_half[2 * k] * s.reshape(-1)
        u0, u1 = u1, np.linalg.solve(op(c_half[2 * (k + 1)]), rhs)
    return u1.reshape(n2, n1)


def _oracle_run(N1, N2, l, tau, M, phi, psi, s, c_half, g_half, K):
    return oracle.solve(N1, N2, l, tau, M, phi, psi, c_half=c_half, s=s, g_half=g_half, steps=K, scheme=1)


@pytest.mark.parametrize("N1,N2", [(8, 8), (9, 6), (4, 11)])
def test_brute_force_dense_kronecker(N1, N2):
    l, M = 1.3, 9
    tau = 0.7 * l / max(N1, N2)
    shape = (N2 - 1, N1 - 1)
    phi, psi, s = (RNG.standard_normal(shape) for _ in range(3))
    c_half = RNG.uniform(0.5, 2.0, 2 * M + 1)
    g_half = RNG.standard_normal(2 * M)
    for K in (1, 2, 3, M):
        got = _oracle_run(N1, N2, l, tau, M, phi, psi, s, c_half, g_half, K)
        want = _dense_run(N1, N2, l, tau, phi, psi, s, c_half, g_half, K)
        np.testing.assert_allclose(got, want, rtol=0, atol=5e-13 * max(1.0, np.abs(want).max()))


def test_one_step_function_matches_dense():
    n1, n2 = 6, 9
    up, uc, s = (RNG.standard_normal((n2, n1)) for _ in range(3))
    axp, axm, ayp, aym, q = 0.7, 0.4, 0.2, 0.9, 0.3
    Kx, Ky = np.kron(np.eye(n2), _K(n1)), np.kron(_K(n2), np.eye(n1))
    I = np.eye(n1 * n2)
    rhs = 2 * uc.reshape(-1) - (I + axm * Kx) @ (I + aym * Ky) @ up.reshape(-1) + q * s.reshape(-1)
    want = np.linalg.solve((I + axp * Kx) @ (I + ayp * Ky), rhs).reshape(n2, n1)
    np.testing.assert_allclose(oracle.factored_step(axp, axm, ayp, aym, q, up, uc, s), want, atol=1e-13)


def test_modal_closed_form():
    N1, N2, l, M = 48, 20, 1.0, 40
    tau = 1.3 * min(l / N1, l / N2)
    x, y = np.arange(1, N1) * l / N1, np.arange(1, N2) * l / N2
    c_half = 1.0 + 0.5 * np.sin(np.arange(2 * M + 1) * 0.21)
    g_half = np.cos(np.arange(2 * M) * 0.4)
    modes = [(3, 5, 0.7, -0.4, 0.9), (1, 1, -1.1, 0.3, 0.0), (7, 2, 0.2, 0.0, -0.5)]
    for m, n, A, Bc, S in modes:
        shape = np.outer(np.sin(n * np.pi * y / l), np.sin(m * np.pi * x / l))
        amps = modal_amplitudes_factored(N1, N2, l, tau, m, n, A, Bc, c_half, M, S=S, g_half=g_half)
        for K in (1, 2, 17, M):
            u = _oracle_run(N1, N2, l, tau, M, A * shape, Bc * shape, S * shape, c_half, g_half, K)
            assert np.abs(u - amps[K] * shape).max() <= 2e-13 * max(1.0, abs(amps[K]))


def test_differs_from_the_unsplit_scheme_by_the_factorisation_term_only():
    """factorised - unsplit = O(tau^4) per step (the a^2 Dx Dy terms): halving tau at fixed T divides the
    difference by ~4 (two orders beyond the schemes' own first-order accuracy is not visible; the local term is
    tau^4, accumulated over T/tau steps twice integrated: tau^2)."""
    N, l, T = 10, 1.0, 0.4
    x = np.arange(1, N) / N
    phi = np.outer(np.sin(np.pi * x), np.sin(2 * np.pi * x)) + 0.3 * np.outer(np.sin(3 * np.pi * x), np.sin(np.pi * x))
    zero = np.zeros_like(phi)
    diffs = []
    for M in (8, 16, 32):
        tau = T / M
        c_half, g_half = np.ones(2 * M + 1), np.zeros(2 * M)
        a = _dense_run(N, N, l, tau, phi, zero, zero, c_half, g_half, M, factored=True)
        b = _dense_run(N, N, l, tau, phi, zero, zero, c_half, g_half, M, factored=False)
        assert np.abs(_oracle_run(N, N, l, tau, M, phi, zero, zero, c_half, g_half, M) - a).max() <= 1e-12
        diffs.append(np.abs(a - b).max())
    assert diffs[0] > 1e-6
    assert 3.0 <= diffs[0] / diffs[1] <= 5.5 and 3.0 <= diffs[1] / diffs[2] <= 5.5


def test_pde_convergence_orders():
    """u = sin(pi x) sin(pi y) cos(pi sqrt(2 c) t): with (2.9) as printed (psi = 0 -> u^1 = u^0) the start is first
    order (P:77's O(tau + |h|^2)); started from the exact u^1 (psi := (u(tau) - u(0)) / tau) the three-level scheme
    with weights 1/2, 0, 1/2 shows its second order."""
    c, l, T = 1.0, 1.0, 0.5
    om = math.pi * math.sqrt(2 * c) / l
    e1, e2 = [], []
    for N in (16, 32, 64):
        M = N // 2
        tau = T / M
        x = np.arange(1, N) / N
        phi = np.outer(np.sin(np.pi * x), np.sin(np.pi * x))
        exact = phi * math.cos(om * T)
        u = oracle.solve(N, N, l, tau, M, phi, None, c_half=np.full(2 * M + 1, c), scheme=1)
        e1.append(np.abs(u - exact).max())
        psi = phi * (math.cos(om * tau) - 1.0) / tau
        u = oracle.solve(N, N, l, tau, M, phi, psi, c_half=np.full(2 * M + 1, c), scheme=1)
        e2.append(np.abs(u - exact).max())
    o1 = [math.log2(e1[i] / e1[i + 1]) for i in range(2)]
    o2 = [math.log2(e2[i] / e2[i + 1]) for i in range(2)]
    assert all(0.8 <= o <= 1.3 for o in o1), (e1, o1)
    assert all(1.8 <= o <= 2.3 for o in o2), (e2, o2)


def test_forced_response_pins_the_source_weight():
    """phi = psi = 0, s = mode (1,1), g = 1, c = 1: amplitude -> (1 - cos(w T)) / w^2, w^2 = 2 pi^2 (full tau^2 f^k)."""
    N, T = 128, 0.5
    M = 128
    tau = T / M
    x = np.arange(1, N) / N
    mode = np.outer(np.sin(np.pi * x), np.sin(np.pi * x))
    u = oracle.solve(N, N, 1.0, tau, M, np.zeros_like(mode), None, c_half=np.ones(2 * M + 1), s=mode, scheme=1)
    amp = float((u * mode).sum() / (mode * mode).sum())
    w2 = 2 * math.pi ** 2
    assert abs(amp - (1 - math.cos(math.sqrt(w2) * T)) / w2) <= 2e-3 * (1 - math.cos(math.sqrt(w2) * T)) / w2 * 10
    assert np.abs(u - amp * mode).max() <= 1e-12


def test_symmetries_and_linearity():
    N, M = 24, 12
    tau = 0.9 / N
    shape = (N - 1, N - 1)
    phi1, phi2, psi, s = (RNG.standard_normal(shape) for _ in range(4))
    c_half = RNG.uniform(0.6, 1.7, 2 * M + 1)
    g_half = RNG.standard_normal(2 * M)
    run = lambda p, q, src: oracle.solve(N, N, 1.0, tau, M, p, q, c_half=c_half, s=src, g_half=g_half, scheme=1)
    u = run(phi1, psi, s)
    # unlike the split scheme (2.11)-(2.12), the factorised scheme commutes with the transposition x <-> y (h1 = h2)
    np.testing.assert_allclose(run(phi1.T.copy(), psi.T.copy(), s.T.copy()), u.T, atol=1e-12)
    np.testing.assert_allclose(run(phi1[:, ::-1].copy(), psi[:, ::-1].copy(), s[:, ::-1].copy()), u[:, ::-1], atol=1e-12)
    lin = run(2 * phi1 - 3 * phi2, 2 * psi, 2 * s) - (2 * u - 3 * run(phi2, np.zeros(shape), np.zeros(shape)))
    assert np.abs(lin).max() <= 1e-11
    assert np.array_equal(run(np.zeros(shape), None, None), np.zeros(shape))


def test_anisotropic_grid_uses_h1_in_x_and_h2_in_y():
    N1, N2, M = 12, 30, 6
    tau = 0.05
    x, y = np.arange(1, N1) / N1, np.arange(1, N2) / N2
    shape = np.outer(np.sin(2 * np.pi * y), np.sin(np.pi * x))
    amps = modal_amplitudes_factored(N1, N2, 1.0, tau, 1, 2, 1.0, 0.5, np.ones(2 * M + 1), M)
    u = oracle.solve(N1, N2, 1.0, tau, M, shape, 0.5 * shape, scheme=1)
    assert np.abs(u - amps[M] * shape).max() <= 1e-13
    wrong = modal_amplitudes_factored(N2, N1, 1.0, tau, 1, 2, 1.0, 0.5, np.ones(2 * M + 1), M)
    assert abs(wrong[M] - amps[M]) > 1e-3


def test_unconditionally_stable_at_large_time_steps():
    """the implicit three-level scheme is unconditionally stable; so is its factorised form (per mode the
    recurrence A_{k+1} = (2 A_k - d A_{k-1}) / d with d >= 1 has |roots| = 1): tau = 64 h for 300 steps stays bounded."""
    N, M = 32, 300
    tau = 64.0 / N
    x = np.arange(1, N) / N
    phi = np.outer(np.sin(np.pi * x), np.sin(2 * np.pi * x)) + 0.5 * np.outer(np.sin(5 * np.pi * x), np.sin(3 * np.pi * x))
    u = oracle.solve(N, N, 1.0, tau, M, phi, None, scheme=1)
    assert np.isfinite(u).all() and np.abs(u).max() <= 1.0 + 1e-9 + np.abs(phi).max()
