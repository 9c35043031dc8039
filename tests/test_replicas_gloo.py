"""The N > 1 path of bench.py on CPU: world_size 2, gloo backend ("replicas only").
Only the rank plumbing is exercised here (barrier, max-over-ranks time, whole-job rate); the replicas
themselves are the single-GPU path that the -m gpu tests cover."""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, time
sys.path.insert(0, os.environ["W2D_ROOT"])
from paper_2006_10142_b200.replicas import Ranks
r = Ranks("gloo")
assert r.world == 2
r.barrier()
mine = 1.0 + 2.0 * r.rank                      # rank 0 took 1 s, rank 1 took 3 s
assert r.max_over_ranks(mine) == 3.0           # the job is as slow as its slowest replica
rate = r.whole_job_rate(units_per_rank=6.0, seconds_this_rank=mine)
assert abs(rate - 2 * 6.0 / 3.0) < 1e-12       # all ranks' units / max time, never a sum of per-rank rates
r.barrier()
r.close()
print("ok", r.rank)
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_ranks_gloo_max_over_ranks_and_whole_job_rate():
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), W2D_ROOT=ROOT)
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=180)[0] for p in procs]
    for rank, (p, out) in enumerate(zip(procs, outs)):
        assert p.returncode == 0, out
        assert f"ok {rank}" in out


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    from paper_2006_10142_b200.replicas import Ranks
    env = {k: os.environ.pop(k) for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK") if k in os.environ}
    try:
        r = Ranks("gloo")
        assert r.world == 1 and r.max_over_ranks(2.5) == 2.5 and r.whole_job_rate(10.0, 2.0) == 5.0
        r.barrier()
        r.close()
    finally:
        os.environ.update(env)
