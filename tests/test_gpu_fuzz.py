"""Seeded random differential test of the CUDA path against the oracle (`-m gpu`): sizes from 1 unknown per line up to a
few panels and tiles, tau from 0.2 h to 30 h (so every solver family is reached: small-grid cluster kernels, streamed
sweeps, whole-line solvers), both dtypes, both schemes, sigma, the second-order start, no / compact / dense source with
and without g(t), constant and time-varying c, the run split into two calls at a random step.  Every case must stay
within the north_star tolerance (fp64 1e-10; fp32 1e-4, widened with tau / h where the systems lose diagonal dominance).
Scheme 1 with rough random data is kept to tau <= 8 h: its carried field V = (I - a_y D_y) U and the tau^2 c Lap_h phi / 2
term of the second-order start amplify rounding like alpha^2 (1e-9 at alpha = 200), in the oracle's formulation and in
this one differently -- a conditioning fact of that regime, not of the solvers (the split scheme stays below 5e-13 at
the same tau)."""
import numpy as np
import pytest

from oracle import oracle
from paper_2006_10142_b200 import binding as B

pytestmark = pytest.mark.gpu


def _case(rng):
    big = rng.random() < 0.12
    N1 = int(rng.integers(2, 1800 if big else 500))
    N2 = int(rng.integers(2, 1800 if big else 500))
    M = int(rng.integers(2, 8))
    scheme = 1 if rng.random() < 0.25 else 0
    tf = float(np.exp(rng.uniform(np.log(0.2), np.log(8.0 if scheme else 30.0))))
    dtype = "f32" if rng.random() < 0.3 else "f64"
    shape = (N2 - 1, N1 - 1)
    phi = rng.uniform(-1, 1, shape)
    psi = rng.uniform(-1, 1, shape) if rng.random() < 0.7 else None
    mode = int(rng.integers(0, 3))                       # 0 no source, 1 dense, 2 compact window
    s = g = None
    if mode == 1:
        s = rng.uniform(-1, 1, shape)
    elif mode == 2:
        s = np.zeros(shape)
        j0, i0 = int(rng.integers(0, shape[0])), int(rng.integers(0, shape[1]))
        s[j0:j0 + int(rng.integers(1, 40)), i0:i0 + int(rng.integers(1, 40))] = 1.0 + rng.random()
    if s is not None and rng.random() < 0.7:
        g = rng.uniform(-1, 1, 2 * M)
    c = rng.uniform(0.5, 1.5, 2 * M + 1) if rng.random() < 0.6 else np.full(2 * M + 1, rng.uniform(0.5, 2.0))
    return dict(N1=N1, N2=N2, M=M, tau=tf / max(N1, N2), tf=tf, dtype=dtype, scheme=scheme, phi=phi, psi=psi, s=s, g=g, c=c,
                solver=int(rng.choice([0, 0, 1, 2])), sigma=float(rng.choice([0.5, 0.5, 0.75, 1.0])) if scheme == 0 else 0.5,
                start=int(rng.choice([1, 2])) if scheme == 1 else 1, split=float(rng.random()))


@pytest.mark.parametrize("seed", [11, 12, 13, 14])
def test_random_cases_match_the_oracle(seed):
    rng = np.random.default_rng(seed)
    ran = 0
    for _ in range(40):
        p = _case(rng)
        f32 = p["dtype"] == "f32"
        cast = (lambda a: None if a is None else a.astype(np.float32).astype(np.float64)) if f32 else (lambda a: a)
        r = oracle.solve(p["N1"], p["N2"], 1.0, p["tau"], p["M"], cast(p["phi"]), cast(p["psi"]), c_half=p["c"], s=cast(p["s"]),
                         g_half=p["g"], scheme=p["scheme"], sigma=p["sigma"] if p["scheme"] == 0 else None,
                         start=p["start"] if p["scheme"] == 1 else None)
        npdt = np.float32 if f32 else np.float64
        what = {k: p[k] for k in ("N1", "N2", "M", "tf", "dtype", "scheme", "solver", "sigma", "start")}
        h = B.Wave2D(p["N1"], p["N2"], 1.0, p["tau"], p["M"], p["dtype"])
        try:
            if p["scheme"]:
                h.set_option("scheme", 1)
                h.set_option("start", p["start"])
            else:
                h.set_option("sigma", p["sigma"])
            h.set_option("solver", p["solver"])
            h.set_speed(p["c"])
            if p["s"] is not None:
                h.set_source(p["s"].astype(npdt), p["g"])
            h.set_initial(p["phi"].astype(npdt), None if p["psi"] is None else p["psi"].astype(npdt))
            left = p["M"] - h.steps_done()
            k1 = int(p["split"] * (left + 1))
            try:
                h.run(k1)
                h.run(left - k1)
            except B.Wave2DError as e:
                assert e.status == -5 and p["solver"] == B.SOLVER_STREAM, what      # the streamed kernels may refuse a large tau
                continue
            u = h.get().astype(np.float64)
        finally:
            h.close()
        err = float(np.abs(u - r).max() / max(np.abs(r).max(), 1e-300))
        tol = 1e-4 * max(1.0, p["tf"]) if f32 else 1e-10   # observed: <= 1.7e-5 over the 38 fp32 cases of these seeds
        assert np.isfinite(u).all() and err <= tol, (what, err)
        ran += 1
    assert ran >= 30
