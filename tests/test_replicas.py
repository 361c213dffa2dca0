"""CPU test (gloo, world_size 2): the N > 1 path of bench.py is N independent replicas, so
the only cross-rank logic is the bookkeeping in paper_2606_07881_b200/replicas.py: rendezvous from the torchrun
environment, barrier, MAX of the per-rank times, SUM of the per-rank work.  Also: `bench.py --impl reference`
under a 2-rank launch prints on rank 0 only and the other rank exits 0 without work."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, {root!r})
from paper_2606_07881_b200 import replicas
rank, world, local = replicas.init_from_env(backend="gloo")
replicas.barrier()
# rank r "measured" (10 + 5 r) ms for (100 + r) units
tput, ms = replicas.whole_job_throughput(10.0 + 5.0 * rank, 100.0 + rank, device="cpu")
replicas.barrier()
print(json.dumps({{"rank": rank, "world": world, "local": local, "ms": ms, "tput": tput}}))
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _launch(code_or_args, world, extra_env=None, is_code=True, timeout=240):
    port = _free_port()
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="", OMP_NUM_THREADS="2")
        env.update(extra_env or {})
        cmd = [sys.executable, "-c", code_or_args] if is_code else [sys.executable] + code_or_args
        procs.append(subprocess.Popen(cmd, env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True, cwd=ROOT))
    outs = []
    for p in procs:
        try:
            o, e = p.communicate(timeout=timeout)
        except subprocess.TimeoutExpired:
            for q in procs:
                q.kill()
            raise
        outs.append((p.returncode, o, e))
    return outs


def test_two_replicas_max_time_sum_work():
    outs = _launch(WORKER.format(root=ROOT), 2)
    rows = []
    for rc, o, e in outs:
        assert rc == 0, e[-2000:]
        rows.append(json.loads(o.strip().splitlines()[-1]))
    rows.sort(key=lambda d: d["rank"])
    assert [d["rank"] for d in rows] == [0, 1] and all(d["world"] == 2 for d in rows)
    for d in rows:                                   # every rank sees the same aggregate
        assert d["ms"] == pytest.approx(15.0)        # MAX over ranks
        assert d["tput"] == pytest.approx(201.0 / 15e-3)   # SUM of the work over the slowest rank's time


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    from paper_2606_07881_b200 import replicas
    assert replicas.aggregate(7.0, 3.0) == (7.0, 3.0)
    tput, ms = replicas.whole_job_throughput(20.0, 50.0)
    assert ms == 20.0 and tput == pytest.approx(2500.0)


def test_reference_arm_prints_on_rank0_only():
    """bench.py --impl reference under a 2-rank launch: rank 0 times the oracle on a tiny config and prints the
    one JSON line; rank 1 exits 0 without work or output."""
    outs = _launch(["bench.py", "--impl", "reference", "--config", "tiny", "--gpus", "2", "--steps", "1", "--warmup", "0"],
                   2, is_code=False)
    (rc0, o0, e0), (rc1, o1, e1) = outs
    assert rc0 == 0 and rc1 == 0, (e0[-1500:], e1[-1500:])
    line = json.loads(o0.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert o1.strip() == ""
