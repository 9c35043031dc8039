"""Seeded synthetic inputs for the five BASELINE.json workloads (and scaled-down copies of them).

This module holds NONE of the method's arithmetic: it only produces the input arrays
(phi, psi, s, c_half, g_half) and the grid parameters, as numpy fp64, that are handed byte-for-byte
to both the CPU oracle and the CUDA library.  Recipe: SURVEY.md section 8d / DESIGN.md "Inputs".

The paper has no dataset; its own runs are c = 1 on 1024^2 .. 8192^2 meshes, which
configs 2, 3 and 5 bracket.  Nodes are x_i = i*l/N1, y_j = j*l/N2; arrays hold interior nodes only,
shape (n2, n1) = (N2-1, N1-1), x fastest.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

SEED_CFG4 = 20061014
SEED_CFG5 = 20061015


@dataclass
class Workload:
    name: str
    N1: int
    N2: int
    l: float
    tau: float
    M: int
    dtype: str                      # "f64" or "f32" (storage/arithmetic type of the GPU run)
    phi: np.ndarray
    psi: Optional[np.ndarray]
    c_half: np.ndarray              # 2M+1 samples c(n tau/2)
    s: Optional[np.ndarray] = None
    g_half: Optional[np.ndarray] = None   # 2M samples g(n tau/2)
    modes: list = field(default_factory=list)   # [(m, n, A)] when phi is a sum of sine modes

    @property
    def n1(self):
        return self.N1 - 1

    @property
    def n2(self):
        return self.N2 - 1

    @property
    def points(self):
        return self.n1 * self.n2


def grid(N1: int, N2: int, l: float = 1.0):
    x = np.arange(1, N1, dtype=np.float64) * (l / N1)
    y = np.arange(1, N2, dtype=np.float64) * (l / N2)
    return x, y


def half_times(tau: float, count: int) -> np.ndarray:
    return np.arange(count, dtype=np.float64) * (0.5 * tau)


def jacobi_smooth(a: np.ndarray, passes: int) -> np.ndarray:
    """new = (W + E + S + N)/4 with zero ghosts, `passes` times (config 4's phi recipe)."""
    for _ in range(passes):
        p = np.pad(a, 1)
        a = 0.25 * (p[1:-1, :-2] + p[1:-1, 2:] + p[:-2, 1:-1] + p[2:, 1:-1])
    return a


def ricker(t: np.ndarray, fp: float = 25.0) -> np.ndarray:
    t0 = 1.5 / fp
    a = (np.pi * fp * (t - t0)) ** 2
    return (1.0 - 2.0 * a) * np.exp(-a)


def cfg1(N: int = 128, M: int = 100) -> Workload:
    """Standing wave: tau = h/2, c = 1, f = 0, phi = sin(pi x) sin(pi y)."""
    x, y = grid(N, N)
    tau = 0.5 / N
    phi = np.outer(np.sin(np.pi * y), np.sin(np.pi * x))
    return Workload("cfg1", N, N, 1.0, tau, M, "f64", phi, None, np.ones(2 * M + 1), modes=[(1, 1, 1.0)])


def cfg2(N: int = 1024, M: int = 500) -> Workload:
    """Gaussian bump, c(t) = 1 + 0.5 sin(2 pi t), tau = h."""
    x, y = grid(N, N)
    tau = 1.0 / N
    phi = np.outer(np.exp(-((y - 0.5) ** 2) / 0.01), np.exp(-((x - 0.5) ** 2) / 0.01))
    c = 1.0 + 0.5 * np.sin(2.0 * np.pi * half_times(tau, 2 * M + 1))
    return Workload("cfg2", N, N, 1.0, tau, M, "f64", phi, None, c)


def cfg3(N: int = 4096, M: int = 1000) -> Workload:
    """Zero initial data, narrow Gaussian source (sigma = 2h) at (0.3, 0.6), Ricker wavelet in time."""
    x, y = grid(N, N)
    tau = 1.0 / N
    sigma = 2.0 / N
    sx = np.exp(-((x - 0.3) ** 2) / (2 * sigma * sigma))
    sy = np.exp(-((y - 0.6) ** 2) / (2 * sigma * sigma))
    s = np.outer(sy, sx) / (2.0 * np.pi * sigma * sigma)
    g = ricker(half_times(tau, 2 * M))
    phi = np.zeros((N - 1, N - 1))
    return Workload("cfg3", N, N, 1.0, tau, M, "f64", phi, None, np.ones(2 * M + 1), s=s, g_half=g)


def cfg4(N1: int = 8192, N2: int = 2048, M: int = 1000, dtype: str = "f64", seed: int = SEED_CFG4) -> Workload:
    """Anisotropic grid, random smoothed phi (rounded to fp32 for both variants), c(t) = 1 + 0.3 cos(4 pi t)."""
    tau = min(1.0 / N1, 1.0 / N2)
    rng = np.random.default_rng(seed)
    phi = rng.uniform(-1.0, 1.0, size=(N2 - 1, N1 - 1))
    phi = jacobi_smooth(phi, 5).astype(np.float32).astype(np.float64)
    c = 1.0 + 0.3 * np.cos(4.0 * np.pi * half_times(tau, 2 * M + 1))
    return Workload("cfg4_" + dtype, N1, N2, 1.0, tau, M, dtype, phi, None, c)


def cfg5(N: int = 16384, M: int = 200, seed: int = SEED_CFG5) -> Workload:
    """Sum of 4 seeded sine modes, c = 2, tau = h."""
    x, y = grid(N, N)
    tau = 1.0 / N
    rng = np.random.default_rng(seed)
    ms = rng.integers(1, 33, size=4)
    ns = rng.integers(1, 33, size=4)
    As = rng.uniform(0.0, 1.0, size=4)
    phi = np.zeros((N - 1, N - 1))
    modes = []
    for m, n, A in zip(ms, ns, As):
        phi += A * np.outer(np.sin(n * np.pi * y), np.sin(m * np.pi * x))
        modes.append((int(m), int(n), float(A)))
    return Workload("cfg5", N, N, 1.0, tau, M, "f64", phi, None, np.full(2 * M + 1, 2.0), modes=modes)


def by_name(name: str, **kw) -> Workload:
    table = {"cfg1": cfg1, "cfg2": cfg2, "cfg3": cfg3, "cfg4": cfg4, "cfg4_f64": cfg4, "cfg5": cfg5}
    if name == "cfg4_f32":
        return cfg4(dtype="f32", **kw)
    return table[name](**kw)


ALL = ["cfg1", "cfg2", "cfg3", "cfg4_f64", "cfg4_f32", "cfg5"]
