"""Row-block sharding with halo refresh (paper_2006_10142_b200/sharded.py).

CPU tests (`-m "not gpu"`): the geometry, and the sharded step itself with a numpy engine that takes the oracle's
half-step as its local solver -- in one process (LocalExchange) and as two ranks over gloo (DistExchange).  They check
the ALGORITHM (which rows are exchanged, when, how wide the halo must be) against the unsharded oracle.  The GPU test
runs the same driver on the CUDA library with three blocks on one GPU."""
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

from oracle import oracle
from paper_2006_10142_b200 import sharded as S

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

ENGINE_SRC = r'''
import numpy as np
from oracle import oracle


class NumpyEngine:
    """A row block stepped by the oracle's half-step (gamma = 2, kappa = 1/2); h2 from the block's own extent ly."""

    def __init__(self, N1, N2, l, ly, tau, M, dtype):
        self.N1, self.N2, self.n1, self.n2, self.tau, self.M, self.dtype = N1, N2, N1 - 1, N2 - 1, tau, M, dtype
        self.h1, self.h2 = l / N1, ly / N2
        self.k, self.s, self.g = 0, None, None

    def set_option(self, name, value):
        pass

    def set_speed(self, c):
        self.c = np.asarray(c, dtype=np.float64)

    def set_source(self, s, g_half=None):
        self.s = np.asarray(s, dtype=np.float64) if np.any(s) else None
        self.g = None if g_half is None else np.asarray(g_half, dtype=np.float64)

    def set_initial(self, phi, psi=None):
        self.w1 = np.array(phi, dtype=np.float64)
        self.w0 = self.w1 - (0.0 if psi is None else 0.5 * self.tau * np.asarray(psi, dtype=np.float64))

    def run(self, steps):
        for _ in range(2 * steps):
            n = 2 * self.k if not hasattr(self, "_half") else self._half
            d = n & 1
            hd = self.h1 if d == 0 else self.h2
            ap = self.tau ** 2 * self.c[n + 1] / (2 * hd * hd)
            am = self.tau ** 2 * self.c[max(n - 1, 0)] / (2 * hd * hd)
            g = 1.0 if self.g is None else self.g[n]
            w2 = oracle.half_step(d, ap, am, 2.0, 0.5 * self.tau ** 2 * g, self.w0, self.w1, self.s)
            self.w0, self.w1 = self.w1, w2
            self._half = n + 1
        self.k += steps

    def get_rows(self, level, j0, count, out=None):
        src = (self.w1 if level == 0 else self.w0)[j0:j0 + count]
        if out is None:
            return src.copy()
        out[...] = src
        return out

    def set_rows(self, level, j0, rows):
        (self.w1 if level == 0 else self.w0)[j0:j0 + len(rows)] = np.asarray(rows)
'''
exec(ENGINE_SRC)


def problem(N1=40, N2=150, M=12, seed=3):
    rng = np.random.default_rng(seed)
    shape = (N2 - 1, N1 - 1)
    phi, psi, s = (rng.uniform(-1, 1, shape) for _ in range(3))
    c = rng.uniform(0.8, 1.3, 2 * M + 1)
    g = rng.uniform(-1, 1, 2 * M)
    tau = 1.0 / max(N1, N2)
    return dict(N1=N1, N2=N2, l=1.0, tau=tau, M=M, phi=phi, psi=psi, s=s, c=c, g=g)


def test_geometry():
    assert S.split_rows(10, 3) == [(0, 4), (4, 7), (7, 10)]
    assert S.halo_rows(0.1716, 1e-17) == 25 and S.halo_rows(0.5, 1e-8) == 29
    b = S.Block(100, 0, 40, 25)
    assert (b.top, b.bot, b.lo, b.hi, b.rows, b.N2) == (0, 25, 0, 65, 65, 66)
    b = S.Block(100, 40, 70, 25)
    assert (b.top, b.bot, b.lo, b.hi) == (25, 25, 15, 95)
    b = S.Block(100, 70, 100, 25)
    assert (b.top, b.bot, b.hi) == (25, 0, 100)
    with pytest.raises(ValueError):
        S.Block(100, 50, 50, 25)


@pytest.mark.parametrize("world", [1, 2, 3])
def test_sharded_step_matches_the_unsharded_oracle(world):
    """Blocks with G halo rows, one exchange of u^{k+1}'s halo rows per step: the owned rows agree with the global
    solve to rounding; with a halo that is too narrow they do not (the width matters)."""
    p = problem()
    want = oracle.solve(p["N1"], p["N2"], p["l"], p["tau"], p["M"], p["phi"], p["psi"], c_half=p["c"], s=p["s"], g_half=p["g"])
    shards, G = S.make_shards(p["N1"], p["N2"], p["l"], p["tau"], p["M"], "f64", world, p["phi"], p["psi"], p["c"],
                              p["s"], p["g"], make_engine=NumpyEngine)
    assert 10 <= G <= 40
    S.run_local(shards, p["M"])
    got = S.gather_local(shards)
    assert got.shape == want.shape
    assert np.abs(got - want).max() <= 1e-13 * np.abs(want).max()
    if world > 1:
        shards, _ = S.make_shards(p["N1"], p["N2"], p["l"], p["tau"], p["M"], "f64", world, p["phi"], p["psi"], p["c"],
                                  p["s"], p["g"], make_engine=NumpyEngine, tol=1e-2)      # G = 5: visibly wrong
        S.run_local(shards, p["M"])
        assert np.abs(S.gather_local(shards) - want).max() > 1e-6 * np.abs(want).max()


def test_a_rank_must_own_at_least_the_halo():
    p = problem(N2=60)
    with pytest.raises(ValueError):
        S.make_shards(p["N1"], p["N2"], p["l"], p["tau"], p["M"], "f64", 4, p["phi"], make_engine=NumpyEngine)


WORKER = ENGINE_SRC + r'''
import os, sys
sys.path.insert(0, os.environ["W2D_ROOT"])
import torch.distributed as dist
from paper_2006_10142_b200 import sharded as S
from tests.test_sharded import problem
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
p = problem()
shards, G = S.make_shards(p["N1"], p["N2"], p["l"], p["tau"], p["M"], "f64", world, p["phi"], p["psi"], p["c"], p["s"], p["g"],
                          ranks=[rank], make_engine=NumpyEngine)
sh = shards[0]
ex = S.DistExchange(sh, rank, world)
for _ in range(p["M"]):
    sh.step(1)
    ex.refresh()
np.save(os.path.join(os.environ["W2D_OUT"], f"owned{rank}.npy"), sh.owned())
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
'''


def test_two_ranks_over_gloo(tmp_path):
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), W2D_ROOT=ROOT, W2D_OUT=str(tmp_path), PYTHONPATH=ROOT)
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True, cwd=ROOT))
    outs = [q.communicate(timeout=300)[0] for q in procs]
    for rank, (q, out) in enumerate(zip(procs, outs)):
        assert q.returncode == 0, out
    p = problem()
    want = oracle.solve(p["N1"], p["N2"], p["l"], p["tau"], p["M"], p["phi"], p["psi"], c_half=p["c"], s=p["s"], g_half=p["g"])
    got = np.concatenate([np.load(tmp_path / f"owned{r}.npy") for r in range(2)], axis=0)
    assert np.abs(got - want).max() <= 1e-13 * np.abs(want).max()


@pytest.mark.gpu
@pytest.mark.parametrize("dtype,tol", [("f64", 1e-10), ("f32", 1e-4)])
def test_three_blocks_on_one_gpu_match_the_oracle_and_the_single_handle(dtype, tol):
    """The CUDA library as the engine of every block (option "ly", wave2d_get_rows / wave2d_set_rows): three blocks of a
    700 x 1500 grid with a source and a time-varying speed, halo refresh through LocalExchange."""
    from paper_2006_10142_b200 import binding as B
    p = problem(N1=700, N2=1500, M=10, seed=11)
    if dtype == "f32":
        for k in ("phi", "psi", "s"):
            p[k] = p[k].astype(np.float32).astype(np.float64)
    want = oracle.solve(p["N1"], p["N2"], p["l"], p["tau"], p["M"], p["phi"], p["psi"], c_half=p["c"], s=p["s"], g_half=p["g"])
    shards, G = S.make_shards(p["N1"], p["N2"], p["l"], p["tau"], p["M"], dtype, 3, p["phi"], p["psi"], p["c"], p["s"], p["g"])
    try:
        S.run_local(shards, p["M"])
        got = S.gather_local(shards).astype(np.float64)
    finally:
        for s in shards:
            s.engine.close()
    assert np.abs(got - want).max() <= tol * np.abs(want).max()
    npdt = np.float64 if dtype == "f64" else np.float32
    h = B.Wave2D(p["N1"], p["N2"], p["l"], p["tau"], p["M"], dtype)
    try:
        h.set_speed(p["c"]); h.set_source(p["s"].astype(npdt), p["g"]); h.set_initial(p["phi"].astype(npdt), p["psi"].astype(npdt))
        h.run(p["M"])
        one = h.get().astype(np.float64)
        rows = h.get_rows(0, 100, 7)
        np.testing.assert_array_equal(rows, h.get()[100:107])
    finally:
        h.close()
    assert np.abs(got - one).max() <= (1e-12 if dtype == "f64" else 2e-5) * np.abs(want).max()


NCCL_WORKER = r'''
import os, sys
sys.path.insert(0, os.environ["W2D_ROOT"])
import numpy as np
import torch
import torch.distributed as dist
from paper_2006_10142_b200 import sharded as S
from tests.test_sharded import problem
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
torch.cuda.set_device(rank)
dev = torch.device("cuda", rank)
dist.init_process_group("nccl", device_id=dev)
p = problem(N1=700, N2=1500, M=10, seed=11)
shards, G = S.make_shards(p["N1"], p["N2"], p["l"], p["tau"], p["M"], "f64", world, p["phi"], p["psi"], p["c"], p["s"], p["g"],
                          ranks=[rank])
sh = shards[0]
ex = S.DistExchange(sh, rank, world, dev)
for _ in range(p["M"]):
    sh.step(1)
    ex.refresh()
np.save(os.path.join(os.environ["W2D_OUT"], f"owned{rank}.npy"), sh.owned())
sh.engine.close()
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
'''


@pytest.mark.gpu
def test_two_ranks_over_nccl_match_the_oracle(tmp_path):
    """DistExchange on the CUDA library, one rank per GPU: the halo rows arrive on NCCL's stream and are written by the
    engine's own stream, so the refresh has to order the two (it blocks the host on torch's current stream after the
    waits).  A stale halo shows up as an error far above the tolerance.  Needs two GPUs; skipped on a one-GPU box."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), W2D_ROOT=ROOT, W2D_OUT=str(tmp_path), PYTHONPATH=ROOT)
        procs.append(subprocess.Popen([sys.executable, "-c", NCCL_WORKER], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True, cwd=ROOT))
    outs = [q.communicate(timeout=600)[0] for q in procs]
    for q, out in zip(procs, outs):
        assert q.returncode == 0, out
    p = problem(N1=700, N2=1500, M=10, seed=11)
    want = oracle.solve(p["N1"], p["N2"], p["l"], p["tau"], p["M"], p["phi"], p["psi"], c_half=p["c"], s=p["s"], g_half=p["g"])
    got = np.concatenate([np.load(tmp_path / f"owned{r}.npy") for r in range(2)], axis=0)
    assert np.abs(got - want).max() <= 1e-10 * np.abs(want).max()
