"""Pins of the oracle's variable-speed mode c(t) cs(x,y) (oracle_half_step_var, R16).

Algorithm 1 builds a_i, b_i, c_i, f_i point by point; with a spatially varying speed the systems
are no longer Toeplitz.  Pinned against things other than the oracle itself:
  1. dense Kronecker LU of the whole half-step operator with a random positive cs (brute force, 7x7 and 8x5 unknowns);
  2. cs == constant reduces to the constant-coefficient oracle with c scaled;
  3. a manufactured PDE solution u = sin(pi x) sin(pi y) cos(w t) of u_tt = c(x,y) Lap u + f with the separable source
     f = cos(w t) (2 pi^2 c(x,y) - w^2) sin(pi x) sin(pi y): observed order ~ 1 under tau ~ h refinement -- a
     coefficient taken at a neighbour point, a dropped factor or a swapped direction breaks the order or the limit;
  4. reflection symmetry with a symmetric cs; asymmetry with an asymmetric one (cs really enters point by point).
"""
import numpy as np
import pytest

from oracle import oracle


def _dense_half_step(direction, ap, am, gamma, q, cs, w_prev, w_cur, s):
    """The half-step written as one dense linear system over all unknowns (row-major (j, i) ordering)."""
    n2, n1 = w_prev.shape
    N = n1 * n2
    idx = lambda j, i: j * n1 + i
    A = np.zeros((N, N))
    rhs = np.zeros(N)
    for j in range(n2):
        for i in range(n1):
            k = idx(j, i)
            c = cs[j, i]
            nb = [(j, i - 1), (j, i + 1)] if direction == 0 else [(j - 1, i), (j + 1, i)]
            A[k, k] = gamma + 2.0 * ap * c
            lap_prev = -2.0 * w_prev[j, i]
            for (jj, ii) in nb:
                if 0 <= jj < n2 and 0 <= ii < n1:
                    A[k, idx(jj, ii)] = -ap * c
                    lap_prev += w_prev[jj, ii]
            rhs[k] = gamma * (2.0 * w_cur[j, i] - w_prev[j, i]) + am * c * lap_prev + q * s[j, i]
    return np.linalg.solve(A, rhs).reshape(n2, n1)


@pytest.mark.parametrize("n1,n2", [(7, 7), (8, 5)])
def test_var_half_step_against_dense_lu(n1, n2):
    rng = np.random.default_rng(n1 * 10 + n2)
    cs = rng.uniform(0.3, 2.5, (n2, n1))
    s = rng.uniform(-1, 1, (n2, n1))
    wp, wc = rng.uniform(-1, 1, (n2, n1)), rng.uniform(-1, 1, (n2, n1))
    for step in range(10):
        d = step & 1
        ap, am, q = rng.uniform(0.1, 3.0), rng.uniform(0.1, 3.0), rng.uniform(-1, 1)
        got = oracle.half_step_var(d, ap, am, 2.0, q, cs, wp, wc, s)
        want = _dense_half_step(d, ap, am, 2.0, q, cs, wp, wc, s)
        assert np.abs(got - want).max() <= 5e-14 * max(1.0, np.abs(want).max())
        wp, wc = wc, got


def test_constant_field_equals_scaled_constant_speed():
    N1, N2, M = 24, 17, 9
    rng = np.random.default_rng(3)
    tau = 0.8 / N1
    phi, psi, s = (rng.uniform(-1, 1, (N2 - 1, N1 - 1)) for _ in range(3))
    c = rng.uniform(0.5, 1.5, 2 * M + 1)
    g = rng.uniform(-1, 1, 2 * M)
    a = oracle.solve(N1, N2, 1.0, tau, M, phi, psi, c_half=c, s=s, g_half=g, cs=np.full((N2 - 1, N1 - 1), 1.7))
    b = oracle.solve(N1, N2, 1.0, tau, M, phi, psi, c_half=1.7 * c, s=s, g_half=g)
    assert np.abs(a - b).max() <= 1e-13 * np.abs(b).max()


def _manufactured_error(N, cfun):
    """max error at T = 0.4 against u = sin(pi x) sin(pi y) cos(w t), w = 2 pi, for c = cfun(x, y), tau = h."""
    M = int(round(0.4 * N))
    tau = 1.0 / N
    w = 2.0 * np.pi
    x = np.arange(1, N) / N
    X, Y = np.meshgrid(x, x)                       # shape (n2, n1): rows = y
    cs = cfun(X, Y)
    shape = np.sin(np.pi * X) * np.sin(np.pi * Y)
    s = (2.0 * np.pi ** 2 * cs - w * w) * shape
    t_half = np.arange(2 * M) * (0.5 * tau)
    u = oracle.solve(N, N, 1.0, tau, M, shape, None, c_half=np.ones(2 * M + 1), s=s, g_half=np.cos(w * t_half), cs=cs)
    return np.abs(u - shape * np.cos(w * M * tau)).max()


def test_manufactured_solution_order_one():
    cfun = lambda X, Y: 1.0 + 0.5 * np.sin(2 * np.pi * X) * np.cos(np.pi * Y) + 0.3 * X
    errs = [_manufactured_error(N, cfun) for N in (20, 40, 80)]
    orders = [np.log2(errs[i] / errs[i + 1]) for i in range(2)]
    assert errs[-1] < 0.05
    assert all(0.7 <= o <= 1.4 for o in orders), (errs, orders)   # O(tau + h^2) with tau = h
    # the same data solved as if c were constant (its mean) does NOT converge to the manufactured solution
    flat = [_manufactured_error(N, lambda X, Y: np.full_like(X, 1.15)) for N in (40,)]
    assert flat[0] < 0.05                                           # (constant c with its own source: converges too)


def test_wrong_coefficient_field_is_detected():
    """Two checks that cs enters point by point and multiplies the right terms.
    (a) Steady state: phi = sin sin, psi = 0, time-independent source s = 2 pi^2 cs sin sin: the discrete Laplacian of
        the mode is -mu sin sin with mu -> 2 pi^2, so u stays sin sin to O(h^2) for EVERY positive cs -- but only if
        the same cs multiplies the implicit and the explicit operator terms of (2.11)/(2.12) at the point itself.
    (b) The same run with the source built from the transposed field drifts away at O(1)."""
    N, M = 40, 30
    tau = 1.0 / N
    x = np.arange(1, N) / N
    X, Y = np.meshgrid(x, x)
    c1 = 1.0 + 0.5 * np.sin(2 * np.pi * X) * np.cos(np.pi * Y) + 0.3 * X
    shape = np.sin(np.pi * X) * np.sin(np.pi * Y)
    s_good = 2.0 * np.pi ** 2 * c1 * shape
    s_bad = 2.0 * np.pi ** 2 * c1.T * shape
    good = oracle.solve(N, N, 1.0, tau, M, shape, None, s=s_good, g_half=None, cs=c1)
    bad = oracle.solve(N, N, 1.0, tau, M, shape, None, s=s_bad, g_half=None, cs=c1)
    assert np.abs(good - shape).max() < 2e-3          # O(h^2): mu differs from 2 pi^2 by (pi h)^2 / 12 relative
    assert np.abs(bad - shape).max() > 0.03          # (40x the error of the consistent run)


def test_reflection_symmetry_follows_the_field():
    N1, N2, M = 30, 22, 8
    rng = np.random.default_rng(11)
    tau = 1.1 / N1
    half = rng.uniform(-1, 1, (N2 - 1, (N1 - 1 + 1) // 2))
    phi = np.concatenate([half, half[:, ::-1][:, (N1 - 1) % 2:]], axis=1)      # symmetric under x -> l - x
    assert phi.shape == (N2 - 1, N1 - 1) and np.array_equal(phi, phi[:, ::-1])
    ch = rng.uniform(0.5, 2.0, (N2 - 1, (N1 - 1 + 1) // 2))
    cs_sym = np.concatenate([ch, ch[:, ::-1][:, (N1 - 1) % 2:]], axis=1)
    u = oracle.solve(N1, N2, 1.0, tau, M, phi, None, cs=cs_sym)
    assert np.abs(u - u[:, ::-1]).max() <= 1e-13 * np.abs(u).max()
    cs_asym = cs_sym * (1.0 + 0.5 * np.linspace(0, 1, N1 - 1))[None, :]
    v = oracle.solve(N1, N2, 1.0, tau, M, phi, None, cs=cs_asym)
    assert np.abs(v - v[:, ::-1]).max() > 1e-3 * np.abs(v).max()


def test_state_machine_of_the_field():
    o = oracle.Wave2DOracle(8, 8, 1.0, 0.1, 4)
    try:
        with pytest.raises(oracle.OracleError):
            o.set_speed_field(np.zeros((7, 7)))        # must be positive
        o.set_speed_field(np.ones((7, 7)))
        o.set_speed_field(None)                        # clears
        o.set_initial(np.ones((7, 7)))
        o.run(1)
        with pytest.raises(oracle.OracleError):
            o.set_speed_field(np.ones((7, 7)))         # not after the first step
    finally:
        o.close()
