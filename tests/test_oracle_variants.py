"""Pins for two oracle options of SURVEY.md 8f NEXT-4 (`-m "not gpu"`):

  sigma  weight of the implicit operator in the split scheme; sigma = 1 with gamma = 1, c = 1 is the tridiagonal system
         Listing 1 prints: a = c = tau^2, b = 2 tau^2 + h^2, f = h^2 u^{k-1} - 2 h^2 u^k.
  start  2: second-order start of the three-level scheme (2.8) (scheme 1); 1: (2.9) as printed.

A wrong weight, a weight on the wrong time level, a dropped source or Laplacian term in the start, or swapped h1 / h2
fails at least one test."""
import math

import numpy as np
import pytest

from oracle import oracle

RNG = np.random.default_rng(1357)


def _K(n):
    return 2.0 * np.eye(n) - np.eye(n, k=1) - np.eye(n, k=-1)      # -(undivided second difference), zero ghosts


def test_sigma_one_is_the_system_of_listing_1():
    """Listing 1, one line, written out with the printed coefficients: the sub-, main and super-diagonal
    a = tau^2, b = 2 tau^2 + h^2, c = tau^2 and f = h^2 Unn - 2 h^2 uu0 belong to  a x_{p-1} - b x_p + c x_{p+1} = f
    (the signs that make it the fully implicit three-level step with Unn = u^{k-1}, uu0 = u^k)."""
    N, tau = 12, 0.05
    n, h = N - 1, 1.0 / N
    unn, uu0 = RNG.standard_normal(n), RNG.standard_normal(n)
    a = np.full(n, tau * tau)
    b = np.full(n, 2 * tau * tau + h * h)
    c = np.full(n, tau * tau)
    f = h * h * unn - 2 * h * h * uu0
    T = np.diag(-b) + np.diag(a[1:], -1) + np.diag(c[:-1], 1)
    want = np.linalg.solve(T, f)
    # the oracle's x half-step with sigma = 1, gamma = 1, c = 1 on a grid whose rows are all this line
    ap, am = 1.0 * tau * tau / (h * h), 0.0
    got = oracle.half_step(0, ap, am, 1.0, 0.0, np.tile(unn, (3, 1)), np.tile(uu0, (3, 1)))
    np.testing.assert_allclose(got, np.tile(want, (3, 1)), rtol=0, atol=1e-13 * np.abs(want).max())
    # and through the handle: option sigma = 1, gamma = 1 gives exactly these weights in both directions
    N1, N2, M = 12, 7, 2
    phi, psi = RNG.standard_normal((N2 - 1, N1 - 1)), RNG.standard_normal((N2 - 1, N1 - 1))
    u = oracle.solve(N1, N2, 1.0, tau, M, phi, psi, steps=1, gamma=1.0, sigma=1.0)
    w0, wm = phi, phi - 0.5 * tau * psi
    w1 = oracle.half_step(0, tau * tau * N1 * N1, 0.0, 1.0, 0.0, wm, w0)
    w2 = oracle.half_step(1, tau * tau * N2 * N2, 0.0, 1.0, 0.0, w0, w1)
    np.testing.assert_allclose(u, w2, rtol=0, atol=1e-13 * np.abs(w2).max())


@pytest.mark.parametrize("sigma", [0.5, 0.75, 1.0])
@pytest.mark.parametrize("N1,N2", [(8, 8), (9, 6)])
def test_sigma_brute_force_dense_kronecker(sigma, N1, N2):
    """gamma (w_{n+1} - 2 w_n + w_{n-1}) + sigma tau^2 c_{n+1}/h_d^2 K_d w_{n+1} + (1 - sigma) tau^2 c_{n-1}/h_d^2 K_d w_{n-1}
    = kappa tau^2 g_n s, solved densely, ten half-steps with random data and time-varying c and g."""
    l, M, gamma, kappa = 1.2, 5, 2.0, 0.5
    n1, n2 = N1 - 1, N2 - 1
    tau = 0.9 * l / max(N1, N2)
    phi, psi, s = (RNG.standard_normal((n2, n1)) for _ in range(3))
    c = RNG.uniform(0.5, 2.0, 2 * M + 1)
    g = RNG.standard_normal(2 * M)
    Kd = [np.kron(np.eye(n2), _K(n1)), np.kron(_K(n2), np.eye(n1))]
    hd = [l / N1, l / N2]
    I = np.eye(n1 * n2)
    wm, w0 = (phi - 0.5 * tau * psi).reshape(-1), phi.reshape(-1)
    for n in range(2 * M):
        d = n & 1
        ap = sigma * tau ** 2 * c[n + 1] / hd[d] ** 2
        am = (1 - sigma) * tau ** 2 * c[max(n - 1, 0)] / hd[d] ** 2
        rhs = gamma * (2 * w0 - wm) - am * (Kd[d] @ wm) + kappa * tau ** 2 * g[n] * s.reshape(-1)
        wm, w0 = w0, np.linalg.solve(gamma * I + ap * Kd[d], rhs)
    got = oracle.solve(N1, N2, l, tau, M, phi, psi, c_half=c, s=s, g_half=g, sigma=sigma)
    np.testing.assert_allclose(got, w0.reshape(n2, n1), rtol=0, atol=5e-13 * max(1.0, np.abs(w0).max()))


def test_sigma_half_is_bit_identical_to_the_default():
    N1, N2, M = 20, 14, 6
    phi, psi = RNG.standard_normal((N2 - 1, N1 - 1)), RNG.standard_normal((N2 - 1, N1 - 1))
    c = RNG.uniform(0.5, 2.0, 2 * M + 1)
    a = oracle.solve(N1, N2, 1.0, 0.03, M, phi, psi, c_half=c)
    b = oracle.solve(N1, N2, 1.0, 0.03, M, phi, psi, c_half=c, sigma=0.5)
    np.testing.assert_array_equal(a, b)


def test_sigma_one_stays_bounded_at_large_tau_and_damps():
    """The fully implicit weight is unconditionally stable and dissipative: at tau = 64 h a mode's amplitude decays."""
    N, M = 64, 40
    x = np.arange(1, N) / N
    phi = np.outer(np.sin(3 * np.pi * x), np.sin(2 * np.pi * x))
    u = oracle.solve(N, N, 1.0, 64.0 / N, M, phi, sigma=1.0)
    assert np.isfinite(u).all() and np.abs(u).max() < 0.5 * np.abs(phi).max()


def _exact(x, y, t, w):
    return np.outer(np.sin(np.pi * y), np.sin(np.pi * x)) * (math.cos(w * t) + math.sin(w * t) / w)


def _err(N, start):
    """u = sin(pi x) sin(pi y) (cos wt + sin wt / w), w = pi sqrt(2): psi = sin sin != 0, f = 0, c = 1; tau = h."""
    w = math.pi * math.sqrt(2.0)
    x = np.arange(1, N) / N
    tau, T = 1.0 / N, 0.5
    M = int(round(T / tau))
    phi = _exact(x, x, 0.0, w)
    psi = np.outer(np.sin(np.pi * x), np.sin(np.pi * x))
    u = oracle.solve(N, N, 1.0, tau, M, phi, psi, scheme=1, start=start)
    return float(np.abs(u - _exact(x, x, M * tau, w)).max())


def test_second_order_start_gives_order_two_with_psi_nonzero():
    """(2.9) as printed is a first-order start (O(tau + |h|^2)); with u^1 = phi + tau psi + tau^2/2 (c Lap_h phi + f^0)
    the three-level scheme (2.8) is second order in tau and h.  Observed orders under tau = h refinement."""
    e1 = [_err(N, 1) for N in (16, 32, 64)]
    e2 = [_err(N, 2) for N in (16, 32, 64)]
    o1 = [math.log2(e1[i] / e1[i + 1]) for i in range(2)]
    o2 = [math.log2(e2[i] / e2[i + 1]) for i in range(2)]
    assert all(0.8 < o < 1.3 for o in o1), (e1, o1)
    assert all(1.8 < o < 2.2 for o in o2), (e2, o2)
    assert e2[-1] < 0.1 * e1[-1]


def test_second_order_start_formula_including_source_and_h1_h2():
    """u^1 after set_initial + run(0 steps is not enough: the term is added at the first run) -- compare level 2 with a
    dense step from the hand-built u^1; h1 != h2, c^0 != 1, source with g^0 != 1."""
    N1, N2, M, l, tau = 9, 6, 3, 1.1, 0.04
    n1, n2 = N1 - 1, N2 - 1
    phi, psi, s = (RNG.standard_normal((n2, n1)) for _ in range(3))
    c = RNG.uniform(0.5, 2.0, 2 * M + 1)
    g = RNG.standard_normal(2 * M)
    h1, h2 = l / N1, l / N2
    Kx, Ky = np.kron(np.eye(n2), _K(n1)), np.kron(_K(n2), np.eye(n1))
    lap = -(Kx / h1 ** 2 + Ky / h2 ** 2) @ phi.reshape(-1)
    u1 = phi.reshape(-1) + tau * psi.reshape(-1) + 0.5 * tau ** 2 * (c[0] * lap + g[0] * s.reshape(-1))
    I = np.eye(n1 * n2)

    def op(cv):
        return (I + tau ** 2 * cv / (2 * h1 ** 2) * Kx) @ (I + tau ** 2 * cv / (2 * h2 ** 2) * Ky)
    u2 = np.linalg.solve(op(c[4]), 2 * u1 - op(c[0]) @ phi.reshape(-1) + tau ** 2 * g[2] * s.reshape(-1))
    got = oracle.solve(N1, N2, l, tau, M, phi, psi, c_half=c, s=s, g_half=g, steps=2, scheme=1, start=2)
    np.testing.assert_allclose(got, u2.reshape(n2, n1), rtol=0, atol=5e-13 * max(1.0, np.abs(u2).max()))


def test_options_are_refused_where_they_do_not_apply():
    o = oracle.Wave2DOracle(8, 8, 1.0, 0.1, 4)
    try:
        o.set_option("start", 2)
        o.set_initial(np.ones((7, 7)))
        with pytest.raises(oracle.OracleError):      # (2.9) belongs to scheme 1
            o.run(1)
    finally:
        o.close()
    o = oracle.Wave2DOracle(8, 8, 1.0, 0.1, 4)
    try:
        o.set_option("scheme", 1)
        o.set_option("sigma", 1.0)
        o.set_initial(np.ones((7, 7)))
        with pytest.raises(oracle.OracleError):      # (2.8) has the weight 1/2 by definition
            o.run(1)
        with pytest.raises(oracle.OracleError):
            o.set_option("sigma", 0.0)
    finally:
        o.close()
