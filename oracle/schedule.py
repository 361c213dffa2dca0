"""ORACLE (test infrastructure): Algorithm 1 as a discrete-event simulator.

Each of the S stages runs the paper's local event rule independently; stages only interact
through messages (h_{m,i} forward, grad h_{m,i-1} backward; Alg. 1 lines 8 and 14).  Time is an
integer virtual clock: a forward at stage s takes tF[s] ticks, a backward tB[s], an update tU[s]
(default 0), a message sent at the end of an op becomes visible `lat` ticks later.  A stage does
one op at a time.

State per stage (Alg. 1 lines 1-3): G (not modelled here), backward counter c,
unresolved-forward counter q, local update index `version`.

Rule (0-based stage s, d_s = S-1-s = the paper's N-i):
  forward of micro-batch m admitted iff its input is visible and q <= d_s (Alg. 1 line 5, Eq. 9
  P:394; P:396 states q < N+1-i and q <= N-i are the same rule);  then vF[m] = version, q += 1.
  backward of m when its input is visible: delta[m] = version - vF[m] (Eq. 8; the update
  triggered by m's own backward is NOT counted -- version is read before line 16's test,
  DESIGN.md R3); then c += 1, q -= 1; if c == k: update, version += 1, c = 0 (lines 16-19).
  Backwards arrive in micro-batch order (all queues FIFO, R4).  When both a forward and a
  backward are ready the backward goes first by default (R1; `backward_first=False` flips it).
  The last stage's backward input is its own loss, visible when its forward ends.

mode="flush" is the synchronous comparator: micro-batches are grouped m_f at a
time, each stage updates once after its m_f-th backward of the group (k := m_f), and no forward
of group g+1 is admitted at a stage before that stage has applied update g, so delta == 0.

The *canonical parity schedule* is tF = tB = 1, tU = 0, lat = 0 (DESIGN.md R-schedule): the
order of ops per stage is then forced, and the CUDA driver reproduces it op for op.
"""
from __future__ import annotations

import math


def delta_bound(n_stages: int, i: int, a: int) -> int:
    """Eq. 10: Delta_{m,i} <= ceil((N - i) / a), i one-based."""
    return math.ceil((n_stages - i) / a)


def eta_flush(m: int, n_stages: int) -> float:
    """Eq. 3: eta_flush(m, N) = m / (m + N - 1)."""
    return m / (m + n_stages - 1)


def eta_inter(m: int, n_stages: int, v: int) -> float:
    """Eq. 4: interleaved 1F1B with V virtual stages per device, eta = m V / (m V + N - 1)."""
    return m * v / (m * v + n_stages - 1)


def simulate(S, n_mb, k, tF=None, tB=None, tU=None, lat=0, mode="paci", m_f=None,
             backward_first=True):
    """Run Alg. 1 on S stages for n_mb micro-batches.  Returns a dict:
       ops      : list of (start, end, stage, kind, mb) with kind in "F","B","U", in start order
                  (ties broken by stage index); "U" carries the new version in place of mb
       delta    : delta[s][m]  (Eq. 8)
       vF, vB   : local update index at forward / backward of (s, m)
       version  : final local update index per stage
       max_q    : largest unresolved-forward count seen per stage (after admission)
       makespan : end time of the last op
    """
    tF = list(tF) if tF is not None else [1] * S
    tB = list(tB) if tB is not None else [1] * S
    tU = list(tU) if tU is not None else [0] * S
    assert min(tF) >= 1 and min(tB) >= 1 and min(tU) >= 0 and lat >= 0
    if mode == "flush":
        assert m_f is not None and m_f >= 1
        k = m_f
    INF = float("inf")
    fwd_vis = [[0 if s == 0 else INF for _ in range(n_mb)] for s in range(S)]
    bwd_vis = [[INF] * n_mb for _ in range(S)]
    free_at = [0] * S
    q = [0] * S
    c = [0] * S
    version = [0] * S
    nf = [0] * S          # next micro-batch to forward
    nb = [0] * S          # oldest unresolved forward = next backward (FIFO)
    vF = [[None] * n_mb for _ in range(S)]
    vB = [[None] * n_mb for _ in range(S)]
    max_q = [0] * S
    ops = []
    t = 0
    while any(nb[s] < n_mb for s in range(S)):
        progressed = False
        for s in range(S):
            if free_at[s] > t:
                continue
            d_s = S - 1 - s
            b_ready = nb[s] < nf[s] and bwd_vis[s][nb[s]] <= t
            f_ready = nf[s] < n_mb and fwd_vis[s][nf[s]] <= t and q[s] <= d_s
            if mode == "flush" and f_ready:
                f_ready = (nf[s] // m_f) == version[s]
            do_b = b_ready and (backward_first or not f_ready)
            if do_b:
                m = nb[s]
                vB[s][m] = version[s]
                end = t + tB[s]
                ops.append((t, end, s, "B", m))
                if s > 0:
                    bwd_vis[s - 1][m] = end + lat
                nb[s] += 1
                c[s] += 1
                q[s] -= 1
                if c[s] == k:
                    version[s] += 1
                    c[s] = 0
                    ops.append((end, end + tU[s], s, "U", version[s]))
                    end += tU[s]
                free_at[s] = end
                progressed = True
            elif f_ready:
                m = nf[s]
                vF[s][m] = version[s]
                end = t + tF[s]
                ops.append((t, end, s, "F", m))
                if s < S - 1:
                    fwd_vis[s + 1][m] = end + lat
                else:
                    bwd_vis[s][m] = end          # own loss, no message
                nf[s] += 1
                q[s] += 1
                max_q[s] = max(max_q[s], q[s])
                free_at[s] = end
                progressed = True
        # jump to the next instant at which anything can change
        cand = [x for x in free_at if x > t]
        for s in range(S):
            if nf[s] < n_mb and fwd_vis[s][nf[s]] != INF and fwd_vis[s][nf[s]] > t:
                cand.append(fwd_vis[s][nf[s]])
            if nb[s] < nf[s] and bwd_vis[s][nb[s]] != INF and bwd_vis[s][nb[s]] > t:
                cand.append(bwd_vis[s][nb[s]])
        if not cand:
            if not progressed:
                raise RuntimeError("schedule deadlock")
            continue
        t = min(cand)
    ops.sort(key=lambda o: (o[0], o[2], "UFB".index(o[3])))   # U precedes the next op of its stage
    delta = [[vB[s][m] - vF[s][m] for m in range(n_mb)] for s in range(S)]
    return dict(ops=ops, delta=delta, vF=vF, vB=vB, version=version, max_q=max_q,
                makespan=max(o[1] for o in ops))


def canonical_ops(S, n_mb, k, mode="paci", m_f=None):
    """The canonical parity schedule: unit durations, zero latency (see module docstring)."""
    return simulate(S, n_mb, k, mode=mode, m_f=m_f)
