"""CPU test (gloo, world_size 3): the stage-per-GPU driver -- Algorithm 1's local event loop with
point-to-point boundary messages -- driven with a stand-in stage that keeps Alg. 1's counters and does trivial
arithmetic, under deliberately UNEQUAL stage times.  Real asynchronous execution has no canonical interleaving, so
what is checked is what the paper guarantees for any timing: Delta_{m,i} <= ceil((N - i) / a) (Eq. 10),
the admission cap q <= N - i + 1 in flight (Eq. 9 / PAPER.md:463), FIFO order, one update per a local backwards, and
that every payload arrives intact and in order."""
import json
import math
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys, time
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
from paper_2606_07881_b200 import replicas
from paper_2606_07881_b200.stage_per_gpu import BoundaryGroups, StageWorker

class FakeStage:
    # Alg. 1 lines 1-3 + P:66: counters only; F: out = in + (s + 1); B: din = 2 * dout (last stage: dout = m + 1)
    def __init__(self, s, S, k, delay):
        self.s, self.S, self.k, self.delay = s, S, k, delay
        self.version, self.c, self.unresolved, self.vF, self.delta, self.fifo = 0, 0, 0, {{}}, {{}}, []
    def forward(self, m, inp, tgt, out):
        assert self.unresolved <= self.S - 1 - self.s, "admission rule violated"
        time.sleep(self.delay)
        self.vF[m] = self.version; self.fifo.append(m); self.unresolved += 1
        if self.s == self.S - 1:
            out.fill_(float(inp.flatten()[0]))           # "loss" = the value that travelled through all stages
        else:
            out.copy_((inp.float() if self.s == 0 else inp) + (self.s + 1))
    def backward(self, m, dout, din):
        assert self.fifo.pop(0) == m, "FIFO violated"
        time.sleep(2 * self.delay)
        self.delta[m] = self.version - self.vF[m]; self.c += 1; self.unresolved -= 1
        if din is not None:
            din.copy_(2.0 * dout if dout is not None else torch.full_like(din, m + 1.0))
        self.last_dout = None if dout is None else float(dout.flatten()[0])
    def maybe_step(self, lr):
        if self.c != self.k: return 0
        self.version += 1; self.c = 0; return 1
    def crossed_updates(self, m): return self.delta[m]

rank, world, local = replicas.init_from_env(backend="gloo")
S, n, k = world, {n}, {k}
groups = BoundaryGroups(world)
delays = {delays!r}
st = FakeStage(rank, S, k, delays[rank])
w = StageWorker(st, rank, S, lambda: torch.zeros(2, 3), groups, depth={depth})
losses = [torch.zeros(1) for _ in range(n)]
seen = []
class Probe(FakeStage): pass
orig_bwd = st.backward
def bwd(m, dout, din):
    orig_bwd(m, dout, din); seen.append((m, st.last_dout))
st.backward = bwd
rep = w.run(n, 1e-3, inputs=lambda m: torch.full((2, 3), 100 * m, dtype=torch.int32), targets=lambda m: None,
            losses=losses, poll_sleep=1e-4)
dist.barrier()
print(json.dumps(dict(rank=rank, delta=rep["delta"], version=rep["version"], max_q=rep["max_q"],
                      events=rep["events"], losses=[float(x) for x in losses], seen=seen)))
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _run(world, n, k, delays, depth):
    port = _free_port()
    code = WORKER.format(root=ROOT, n=n, k=k, delays=delays, depth=depth)
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="", OMP_NUM_THREADS="1")
        procs.append(subprocess.Popen([sys.executable, "-c", code], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True, cwd=ROOT))
    rows = {}
    for p in procs:
        try:
            o, e = p.communicate(timeout=240)
        except subprocess.TimeoutExpired:
            for q in procs:
                q.kill()
            raise
        assert p.returncode == 0, e[-3000:]
        d = json.loads(o.strip().splitlines()[-1])
        rows[d["rank"]] = d
    return rows


def _check(rows, S, n, k):
    for s in range(S):
        d = rows[s]
        bound = math.ceil((S - 1 - s) / k)                                  # Eq. 10 with i = s + 1
        assert len(d["delta"]) == n and max(d["delta"]) <= bound and min(d["delta"]) >= 0, (s, d["delta"])
        assert d["max_q"] <= S - s                                          # stage i carries at most N - i + 1
        assert d["version"] == n // k                                       # one update per k local backwards
        fs = [m for kind, m in d["events"] if kind == "F"]
        bs = [m for kind, m in d["events"] if kind == "B"]
        assert fs == list(range(n)) and bs == list(range(n))                # FIFO in micro-batch id
        pos = {(kind, m): i for i, (kind, m) in enumerate(d["events"])}
        assert all(pos[("F", m)] < pos[("B", m)] for m in range(n))
        us = [i for i, (kind, _) in enumerate(d["events"]) if kind == "U"]
        for j, i in enumerate(us):                                           # U right after every k-th backward
            assert d["events"][i - 1] == ["B", (j + 1) * k - 1]
    assert max(rows[S - 1]["delta"]) == 0                                    # the last stage never crosses (i = N)
    # payloads: forward adds s + 1 at every stage but the last; the last stage's "loss" is what arrived
    add = sum(s + 1 for s in range(S - 1))
    assert rows[S - 1]["losses"] == [100.0 * m + add for m in range(n)]
    # backward: the last stage emits m + 1, every stage doubles: stage s sees (m + 1) * 2^(S - 2 - s)
    for s in range(S - 1):
        assert rows[s]["seen"] == [[m, (m + 1.0) * 2 ** (S - 2 - s)] for m in range(n)], s


def test_three_stages_slow_last_stage():
    S, n, k = 3, 12, 2
    _check(_run(S, n, k, [0.0, 0.001, 0.004], depth=S), S, n, k)


def test_three_stages_slow_first_stage_k1_small_ring():
    S, n, k = 3, 9, 1
    rows = _run(S, n, k, [0.004, 0.0, 0.001], depth=2)
    _check(rows, S, n, k)


def test_two_stages_k4_reaches_the_bound_or_stays_below():
    S, n, k = 2, 16, 4
    rows = _run(S, n, k, [0.0, 0.002], depth=2)
    _check(rows, S, n, k)
    assert max(rows[0]["delta"]) <= 1
