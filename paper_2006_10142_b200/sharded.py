"""Row-block sharding of the split scheme over several GPUs ("GPU cluster").

The x half-step solves one system per grid row, the y half-step one per grid column: the two sweeps want orthogonal
partitions, so a sharded step needs an exchange.  The one used here follows from the decay of the LU recurrences
(DESIGN.md 7): a y line may be cut if the cut piece starts G rows early and ends G rows late with rho_y^G below the
rounding unit.  Rank r owns the grid rows [a_r, b_r) and keeps them in a handle of its own together with up to G halo
rows on either side (option "ly": the handle's grid is a row block of the domain).  One step of the block is then

    handle.run(1)               x half-step: exact on every local row (rows are independent, halo rows included);
                                y half-step: the local buffer ends where the halo ends, so the result is wrong by
                                O(rho^d) at distance d from those ends -- below rounding on the owned rows;
    refresh the halo rows of u^{k+1} from the neighbours' owned rows   (the only exchange: 2 G rows per neighbour)

u^{k+1/2} needs no exchange: the next x half-step recomputes its halo rows from valid inputs.  A block that touches the
physical boundary has no halo there (the true Dirichlet condition).  The exchange is point-to-point between neighbours
(`torch.distributed` isend / irecv: NCCL over NVLink on GPUs, gloo in the CPU test); `LocalExchange` moves the rows
inside one process, which is how the path is tested on one GPU.  No arithmetic of the method lives here: the engine is
the C ABI (binding.Wave2D), the halo width comes from the library's own decay ratio (wave2d_host_decay).
"""
from __future__ import annotations

import math

import numpy as np


def halo_rows(rho: float, tol: float) -> int:
    """Rows of halo G with rho^G <= tol (+ 2: the stencil row and one of margin)."""
    if not (0.0 < rho < 1.0):
        return 2
    return int(math.ceil(math.log(tol) / math.log(rho))) + 2


def split_rows(n2: int, world: int):
    """Owned rows [a_r, b_r) of every rank: contiguous, sizes differing by at most one."""
    base, extra = divmod(n2, world)
    out, a = [], 0
    for r in range(world):
        b = a + base + (1 if r < extra else 0)
        out.append((a, b))
        a = b
    return out


class Block:
    """Geometry of one rank's handle: owned rows [a, b) of n2, `top` / `bot` halo rows; local rows [a - top, b + bot)."""

    def __init__(self, n2: int, a: int, b: int, G: int):
        if b - a < 1:
            raise ValueError("a rank must own at least one grid row")
        self.n2, self.a, self.b = n2, a, b
        self.top, self.bot = min(G, a), min(G, n2 - b)
        self.lo, self.hi = a - self.top, b + self.bot
        self.rows = self.hi - self.lo                      # unknowns per y line of the local grid
        self.N2 = self.rows + 1                            # its interval count

    def local(self, field):
        return None if field is None else np.ascontiguousarray(field[self.lo:self.hi])


class LocalExchange:
    """All blocks live in this process (one GPU, or the CPU test): rows move by get_rows / set_rows."""

    def __init__(self, shards):
        self.shards = shards

    def refresh(self):
        sh = self.shards
        for r, s in enumerate(sh):
            if s.block.top:                                # my top halo = the last rows the upper neighbour owns
                up = sh[r - 1]
                s.engine.set_rows(0, 0, up.engine.get_rows(0, up.block.top + (up.block.b - up.block.a) - s.block.top,
                                                           s.block.top))
            if s.block.bot:
                dn = sh[r + 1]
                s.engine.set_rows(0, s.block.top + (s.block.b - s.block.a), dn.engine.get_rows(0, dn.block.top, s.block.bot))


class DistExchange:
    """One block per rank; neighbours trade rows with torch.distributed point-to-point calls."""

    def __init__(self, shard, rank: int, world: int, device=None):
        import torch
        import torch.distributed as dist
        self.torch, self.dist = torch, dist
        self.shard, self.rank, self.world, self.device = shard, rank, world, device

    def _buf(self, count):
        t = self.torch
        dt = t.float64 if self.shard.engine.dtype == "f64" else t.float32
        return t.empty((count, self.shard.engine.n1), dtype=dt, device=self.device or "cpu")

    def _rows(self, j0, count):
        out = self._buf(count)
        if out.is_cuda:
            self.shard.engine.get_rows(0, j0, count, out)
        else:
            out.copy_(self.torch.from_numpy(self.shard.engine.get_rows(0, j0, count)))
        return out

    def refresh(self):
        s, b, dist = self.shard, self.shard.block, self.dist
        own = b.b - b.a
        ops, recv = [], []
        # every rank sends min(G, what the neighbour's halo holds) rows: the neighbour's halo width is its min(G, ...),
        # which equals min(G, rows this rank owns above / below the cut) only if a rank owns at least G rows -- checked
        # at construction (ShardedWave2D)
        if self.rank > 0:
            send = self._rows(b.top, s.G_up)               # my first owned rows -> the upper neighbour's bottom halo
            ops.append(dist.P2POp(dist.isend, send, self.rank - 1))
            if b.top:
                got = self._buf(b.top)
                ops.append(dist.P2POp(dist.irecv, got, self.rank - 1))
                recv.append((0, got))
        if self.rank < self.world - 1:
            send = self._rows(b.top + own - s.G_dn, s.G_dn)   # my last owned rows -> the lower neighbour's top halo
            ops.append(dist.P2POp(dist.isend, send, self.rank + 1))
            if b.bot:
                got = self._buf(b.bot)
                ops.append(dist.P2POp(dist.irecv, got, self.rank + 1))
                recv.append((b.top + own, got))
        for w in dist.batch_isend_irecv(ops) if ops else []:
            w.wait()
        if self.device is not None and self.torch.device(self.device).type == "cuda":
            # On NCCL, wait() only makes torch's current stream wait for the transfer; the host goes on.  The engine copies
            # the halo rows on a non-blocking stream of its own, which is ordered after neither: block the host until the
            # rows have arrived (and the send buffers are no longer read) before set_rows touches them.
            self.torch.cuda.current_stream(self.device).synchronize()
        for j0, got in recv:
            s.engine.set_rows(0, j0, got if got.is_cuda else got.numpy())


class Shard:
    """One row block: its geometry and its engine (anything with run / get_rows / set_rows / n1 / dtype)."""

    def __init__(self, block: Block, engine, G_up: int, G_dn: int):
        self.block, self.engine, self.G_up, self.G_dn = block, engine, G_up, G_dn

    def step(self, steps: int = 1):
        self.engine.run(steps)

    def owned(self):
        """u^k on the rows this rank owns."""
        return self.engine.get_rows(0, self.block.top, self.block.b - self.block.a)


def y_decay(N2: int, l: float, tau: float, c_half, gamma: float = 2.0, sigma: float = 0.5) -> float:
    """rho of the y systems at the largest speed sample: computed by the library (wave2d_host_decay), not here."""
    from . import binding
    return binding.host_decay(N2, l, tau, float(np.max(c_half)), gamma, sigma)


def make_shards(N1: int, N2: int, l: float, tau: float, M: int, dtype: str, world: int, phi, psi=None, c_half=None,
                s=None, g_half=None, ranks=None, tol=None, make_engine=None, options=None):
    """Build the shards of `ranks` (default: all `world` of them, for LocalExchange) of the N1 x N2 problem.

    make_engine(N1, N2_local, l, ly_local, tau, M, dtype) -> engine; default: binding.Wave2D with option "ly"."""
    from . import binding
    n2 = N2 - 1
    c = np.ones(2 * M + 1) if c_half is None else np.atleast_1d(np.asarray(c_half, dtype=np.float64))
    if c.shape[0] == 1:
        c = np.full(2 * M + 1, c[0])
    opts = dict(options or {})
    tol = tol or (1e-17 if dtype == "f64" else 1e-8)
    G = halo_rows(y_decay(N2, l, tau, c, opts.get("gamma", 2.0), opts.get("sigma", 0.5)), tol)
    cuts = split_rows(n2, world)
    if world > 1 and min(b - a for a, b in cuts) < G:
        raise ValueError(f"every rank must own at least G = {G} rows (halo of the y sweep); {n2} rows over {world} ranks")
    npdt = np.float64 if dtype == "f64" else np.float32

    def default_engine(N1_, N2_, l_, ly_, tau_, M_, dtype_):
        h = binding.Wave2D(N1_, N2_, l_, tau_, M_, dtype_)
        h.set_option("ly", ly_)
        for k, v in opts.items():
            h.set_option(k, v)
        return h

    make_engine = make_engine or default_engine
    out = []
    for r in (range(world) if ranks is None else ranks):
        a, b = cuts[r]
        blk = Block(n2, a, b, G)
        eng = make_engine(N1, blk.N2, l, (l / N2) * blk.N2, tau, M, dtype)
        eng.set_speed(c)
        if s is not None:
            eng.set_source(blk.local(np.asarray(s)).astype(npdt), g_half)
        eng.set_initial(blk.local(np.asarray(phi)).astype(npdt),
                        None if psi is None else blk.local(np.asarray(psi)).astype(npdt))
        out.append(Shard(blk, eng, G_up=min(G, n2 - a) if r > 0 else 0, G_dn=min(G, b) if r < world - 1 else 0))
    return out, G


def run_local(shards, steps: int):
    """`steps` time steps of all shards in this process: step every block, then refresh every halo."""
    ex = LocalExchange(shards)
    for _ in range(steps):
        for s in shards:
            s.step(1)
        ex.refresh()


def gather_local(shards) -> np.ndarray:
    return np.concatenate([s.owned() for s in shards], axis=0)
