"""ORACLE (test infrastructure): memory-constrained pipeline partitioning (App. D.5).

Split L sequential layers across N stages by cut points 0 = c_0 < c_1 < ... < c_N = L (contiguous groups
G_j = {c_{j-1}+1 .. c_j}, j = 1..N), minimising the slowest stage's time subject to a per-device memory budget:

    T(a, b)   = sum_{l=a+1..b} t_l                                             (Eq. 14)
    M_j(a, b) = sum_{l=a+1..b} s_l + w_j * sum_{l=a+1..b} a_l,   w_j = N - j + 1   (Eq. 12, 14)
    min max_j T(G_j)   s.t.  M_j(G_j) <= B  for all j                          (Eq. 13)

w_j is printed garbled ("w_j = N j + 1"); the parenthesis "the first stage carries N microbatches, the last
carries one" fixes it to N - j + 1 (R20).

Algorithm, as the paper states it: a two-pass dynamic program.
  pass 1  D[i][j] = min over j-1 <= x < i with M_j(x, i) <= B of max(D[x][j-1], T(x, i)),   D[i][1] = T(0, i) if
          M_1(0, i) <= B else +inf                                             (Eq. 15); cuts by backtracking pi[i][j].
  pass 2  (only if D[L][N] = +inf) the same recursion "over pairs (o, t) ordered lexicographically, where
          o = max(0, M_j(G_j) - B) is the per-stage overshoot": minimise the worst overshoot first, the maximum stage
          time as tie-breaker.  max of two pairs is taken component-wise; min is lexicographic.

Pinned by brute-force enumeration of all cut points for small L (tests/test_oracle_partition.py).
"""
from __future__ import annotations

import itertools
import math


def _prefix(v):
    p = [0.0]
    for x in v:
        p.append(p[-1] + x)
    return p


def stage_memory(j, n_stages, s_sum, a_sum):
    """Eq. 12 with w_j = N - j + 1 (j one-based)."""
    return s_sum + (n_stages - j + 1) * a_sum


def partition(t, s, a, n_stages, budget):
    """Returns dict(cuts [N+1], max_time, max_overshoot, fallback: bool).  Raises ValueError if L < N."""
    L, N = len(t), n_stages
    if not (len(s) == len(a) == L) or N < 1 or L < N:
        raise ValueError("need at least one layer per stage")
    pt, ps, pa = _prefix(t), _prefix(s), _prefix(a)
    T = lambda x, i: pt[i] - pt[x]
    M = lambda j, x, i: stage_memory(j, N, ps[i] - ps[x], pa[i] - pa[x])
    INF = math.inf
    # ---- pass 1 (Eq. 15)
    D = [[INF] * (N + 1) for _ in range(L + 1)]
    pi = [[-1] * (N + 1) for _ in range(L + 1)]
    for i in range(1, L + 1):
        if M(1, 0, i) <= budget:
            D[i][1] = T(0, i)
            pi[i][1] = 0
    for j in range(2, N + 1):
        for i in range(j, L + 1):
            for x in range(j - 1, i):
                if M(j, x, i) > budget or D[x][j - 1] == INF:
                    continue
                v = max(D[x][j - 1], T(x, i))
                if v < D[i][j]:
                    D[i][j], pi[i][j] = v, x
    if D[L][N] < INF:
        cuts = _backtrack(pi, L, N)
        return dict(cuts=cuts, max_time=D[L][N], max_overshoot=0.0, fallback=False)
    # ---- pass 2: pairs (overshoot, time), lexicographic min of component-wise max
    BIG = (INF, INF)
    E = [[BIG] * (N + 1) for _ in range(L + 1)]
    pi = [[-1] * (N + 1) for _ in range(L + 1)]
    over = lambda j, x, i: max(0.0, M(j, x, i) - budget)
    for i in range(1, L + 1):
        E[i][1] = (over(1, 0, i), T(0, i))
        pi[i][1] = 0
    for j in range(2, N + 1):
        for i in range(j, L + 1):
            for x in range(j - 1, i):
                if E[x][j - 1] == BIG:
                    continue
                v = (max(E[x][j - 1][0], over(j, x, i)), max(E[x][j - 1][1], T(x, i)))
                if v < E[i][j]:
                    E[i][j], pi[i][j] = v, x
    cuts = _backtrack(pi, L, N)
    return dict(cuts=cuts, max_time=E[L][N][1], max_overshoot=E[L][N][0], fallback=True)


def _backtrack(pi, L, N):
    cuts = [L]
    i = L
    for j in range(N, 0, -1):
        i = pi[i][j]
        cuts.append(i)
    return cuts[::-1]


def evaluate(cuts, t, s, a, budget):
    """(max stage time, max overshoot) of a given partition: the definitions of Eq. 12-13 written out."""
    N = len(cuts) - 1
    worst_t, worst_o = 0.0, 0.0
    for j in range(1, N + 1):
        lo, hi = cuts[j - 1], cuts[j]
        worst_t = max(worst_t, sum(t[lo:hi]))
        worst_o = max(worst_o, max(0.0, stage_memory(j, N, sum(s[lo:hi]), sum(a[lo:hi])) - budget))
    return worst_t, worst_o


def brute_force(t, s, a, n_stages, budget):
    """All C(L-1, N-1) cut sets.  Returns (best feasible max time or None, min worst overshoot)."""
    L, N = len(t), n_stages
    best_t, best_o = None, math.inf
    for inner in itertools.combinations(range(1, L), N - 1):
        cuts = [0, *inner, L]
        wt, wo = evaluate(cuts, t, s, a, budget)
        best_o = min(best_o, wo)
        if wo == 0.0 and (best_t is None or wt < best_t):
            best_t = wt
    return best_t, best_o
