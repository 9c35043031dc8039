"""Exact discrete modal closed form of the split scheme (SURVEY.md 8c pin 3) -- test helper.

For phi = A sin(m pi x/l) sin(n pi y/l) (psi = B times the same mode, source s = S times the same mode)
every half-level stays a multiple a_k of the mode, because the mode is an eigenvector of both undivided
second differences:  delta_x^2 mode = -h1^2 mu_x mode,  mu_x = (4/h1^2) sin^2(m pi h1 / (2 l)), same in y.
Substituting into (2.11)/(2.12) (times tau^2, reading A2) gives the scalar recurrence

    (gamma + tau^2 c_{k+1} mu_d / 2) a_{k+1} = 2 gamma a_k - (gamma + tau^2 c_{k-1} mu_d / 2) a_{k-1} + kappa tau^2 g_k S

with d = x for even k, y for odd k, a_0 = A, a_{-1} = A - (tau/2) B, c_{-1} := c_0.
This is derived from the mathematics (eigen-decomposition), not from the oracle's code; it contains no
tridiagonal solve and no grid.
"""
import math


def modal_amplitudes(N1, N2, l, tau, m, n, A, B, c_half, nhalf, S=0.0, g_half=None, gamma=2.0, kappa=0.5):
    """Return [a_0, a_1, ..., a_nhalf] (amplitudes at half-levels)."""
    h1, h2 = l / N1, l / N2
    mu = ((4.0 / (h1 * h1)) * math.sin(m * math.pi * h1 / (2 * l)) ** 2,
          (4.0 / (h2 * h2)) * math.sin(n * math.pi * h2 / (2 * l)) ** 2)
    a_prev, a_cur = A - 0.5 * tau * B, A
    out = [a_cur]
    t2 = tau * tau
    for k in range(nhalf):
        d = k & 1
        cp = c_half[k + 1]
        cm = c_half[k - 1] if k > 0 else c_half[0]
        g = 1.0 if g_half is None else g_half[k]
        lhs = gamma + t2 * cp * mu[d] / 2.0
        rhs = 2.0 * gamma * a_cur - (gamma + t2 * cm * mu[d] / 2.0) * a_prev + kappa * t2 * g * S
        a_prev, a_cur = a_cur, rhs / lhs
        out.append(a_cur)
    return out


def modal_amplitudes_factored(N1, N2, l, tau, m, n, A, B, c_half, K, S=0.0, g_half=None):
    """Factorised form of the unsplit scheme (2.8), same mode ansatz:
    -(undivided second difference) has the eigenvalue lam_d = 4 sin^2(m_d pi h_d / (2 l)) on the mode, so with
    a_d(c) = tau^2 c / (2 h_d^2) every integer level k obeys

        (1 + a_x(c_{k+1}) lam_x)(1 + a_y(c_{k+1}) lam_y) A_{k+1}
            = 2 A_k - (1 + a_x(c_{k-1}) lam_x)(1 + a_y(c_{k-1}) lam_y) A_{k-1} + tau^2 g_k S,

    A_0 = A, A_1 = A + tau B ((2.9)); c_k = c_half[2k], g_k = g_half[2k].  Returns [A_0 .. A_K]."""
    h1, h2 = l / N1, l / N2
    lam = (4.0 * math.sin(m * math.pi * h1 / (2 * l)) ** 2, 4.0 * math.sin(n * math.pi * h2 / (2 * l)) ** 2)
    t2 = tau * tau

    def op(c):
        return (1.0 + t2 * c / (2 * h1 * h1) * lam[0]) * (1.0 + t2 * c / (2 * h2 * h2) * lam[1])

    out = [A, A + tau * B]
    for k in range(1, K):
        g = 1.0 if g_half is None else g_half[2 * k]
        out.append((2.0 * out[k] - op(c_half[2 * (k - 1)]) * out[k - 1] + t2 * g * S) / op(c_half[2 * (k + 1)]))
    return out[:K + 1]
