"""World-size-2 gloo test (CPU) of the rank plumbing behind ``bench.py --gpus N``: replicas only, no data-path
collective.  Checks the barrier, the max-over-ranks timing, the aggregate value, that
only rank 0 of ``--impl reference`` prints, and the contiguous split of independent problems."""
import json
import os
import socket
import subprocess
import sys

import pytest

from paper_2108_01786_b200 import ranks

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys, time
sys.path.insert(0, {root!r})
from paper_2108_01786_b200 import ranks
r = ranks.from_env("gloo")
assert r.world == 2 and r.backend == "gloo" and r.device == "cpu"
ranks.barrier(r)
# rank 1 is the slow replica: every rank must see ITS time and the sum of the units
secs = 0.25 if r.rank == 0 else 0.75
units = 100.0 * (r.rank + 1)
value, tmax, total = ranks.aggregate_value(r, units, secs)
ranks.barrier(r)
print(json.dumps({{"rank": r.rank, "root": r.is_root, "value": value, "tmax": tmax, "total": total,
                  "mx": ranks.max_over_ranks(r, float(r.rank))}}), flush=True)
ranks.finish(r)
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _spawn(code_or_argv, world=2, timeout=180):
    port = _free_port()
    procs = []
    for rk in range(world):
        env = dict(os.environ, RANK=str(rk), LOCAL_RANK=str(rk), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), OMP_NUM_THREADS="2")
        argv = [sys.executable, "-c", code_or_argv] if isinstance(code_or_argv, str) else [sys.executable] + code_or_argv
        procs.append(subprocess.Popen(argv, env=env, cwd=ROOT, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        try:
            o, e = p.communicate(timeout=timeout)
        except subprocess.TimeoutExpired:
            for q in procs:
                q.kill()
            raise
        assert p.returncode == 0, e[-2000:]
        outs.append(o)
    return outs


def test_world2_gloo_max_time_and_aggregate_value():
    outs = _spawn(WORKER.format(root=ROOT))
    rows = [json.loads([l for l in o.splitlines() if l.startswith("{")][-1]) for o in outs]
    rows.sort(key=lambda d: d["rank"])
    assert [d["root"] for d in rows] == [True, False]
    for d in rows:
        assert d["tmax"] == 0.75          # the slow replica decides
        assert d["total"] == 300.0        # units of both replicas
        assert d["value"] == pytest.approx(400.0)
        assert d["mx"] == 1.0


def test_world1_needs_no_process_group(monkeypatch):
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        monkeypatch.delenv(k, raising=False)
    r = ranks.from_env("gloo")
    assert (r.world, r.rank, r.backend) == (1, 0, None)
    ranks.barrier(r)
    assert ranks.max_over_ranks(r, 3.5) == 3.5
    assert ranks.aggregate_value(r, 10.0, 2.0) == (5.0, 2.0, 10.0)
    ranks.finish(r)


def test_assign_replicas_covers_everything_once():
    for n, w in [(4, 1), (4, 2), (4, 3), (12, 8), (3, 8), (0, 2)]:
        parts = ranks.assign_replicas(n, w)
        assert len(parts) == w
        assert [i for p in parts for i in p] == list(range(n))
        assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1


def test_reference_arm_only_rank0_prints():
    """bench.py --impl reference under a 2-rank launch: rank 0 prints ONE JSON line with impl=reference, the other
    rank exits 0 without work (and without needing a process group or a GPU)."""
    outs = _spawn(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--config", "1",
                   "--cpu-seconds", "2"], timeout=300)
    lines0 = [l for l in outs[0].splitlines() if l.startswith("{")]
    assert len(lines0) == 1 and outs[1].strip() == ""
    d = json.loads(lines0[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["value"] > 0 and d["unit"] == "Gentries/s"
