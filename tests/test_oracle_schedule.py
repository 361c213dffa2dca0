"""Pins for oracle/schedule.py: the paper's bound (Eq. 2/10/11) under arbitrary stage times,
the values the paper prints, and the closed forms of the canonical schedule.  SURVEY.md 8(c-5)."""
import os
import random

import pytest

from oracle import schedule

GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")) as f:
    for line in f:
        line = line.split("#")[0].strip()
        if "=" in line:
            key, val = line.rsplit("=", 1)
            GOLD[key.strip()] = float(val)


def test_bound_function_reproduces_printed_values():
    assert schedule.delta_bound(8, 1, 4) == GOLD["bound N=8 a=4"]
    assert schedule.delta_bound(8, 1, 8) == GOLD["bound N=8 a=8"]
    assert schedule.delta_bound(32, 1, 96) == GOLD["bound N=32 a=96"]
    assert abs(schedule.eta_flush(4, 9) - GOLD["eta_flush m=4 N=9"]) < 1e-15
    assert abs(148.64 / 87.99 - GOLD["speedup 148.64/87.99"]) < 5e-3     # Table 4 is self-consistent
    assert abs(227.62 / 111.51 - GOLD["speedup 227.62/111.51"]) < 5e-3
    assert abs(124.27 / 87.89 - GOLD["speedup 124.27/87.89"]) < 5e-3


@pytest.mark.parametrize("seed", range(25))
def test_bound_holds_under_random_stage_times(seed):
    """P:404 "without relying on balanced stage times": Eq. 10 for every (m, i), any durations,
    any latency, either F/B priority; last stage never crosses an update (i = N)."""
    rnd = random.Random(seed)
    S = rnd.randint(1, 9)
    k = rnd.choice([1, 2, 3, 4, 8, 16])
    n = rnd.randint(1, 40)
    r = schedule.simulate(S, n, k, tF=[rnd.randint(1, 9) for _ in range(S)],
                          tB=[rnd.randint(1, 17) for _ in range(S)],
                          tU=[rnd.randint(0, 5) for _ in range(S)], lat=rnd.randint(0, 6),
                          backward_first=rnd.random() < 0.5)
    for s in range(S):
        assert r["max_q"][s] <= S - s                                 # P:463 / Eq. 9
        assert r["version"][s] == n // k                              # tail window does not update
        for m in range(n):
            assert 0 <= r["delta"][s][m] <= schedule.delta_bound(S, s + 1, k)
    assert all(d == 0 for d in r["delta"][S - 1])


def test_canonical_schedule_example_S2_k4():
    """SURVEY 8(c-2) example, obtained there by brute-force event counting."""
    r = schedule.simulate(2, 16, 4)
    st0 = " ".join(f"{kd}{m}" for (_, _, s, kd, m) in r["ops"] if s == 0)
    assert st0.startswith("F0 F1 B0 F2 B1 F3 B2 F4 B3 U1 F5 B4") and st0.endswith("F15 B14 B15 U4")
    st1 = " ".join(f"{kd}{m}" for (_, _, s, kd, m) in r["ops"] if s == 1)
    assert st1.startswith("F0 B0 F1 B1 F2 B2 F3 B3 U1 F4 B4")
    assert r["delta"][0] == [1 if m in (4, 8, 12) else 0 for m in range(16)]
    assert r["delta"][1] == [0] * 16 and r["version"] == [4, 4]
    assert r["makespan"] == 2 * 16 + 2 * (2 - 1)


@pytest.mark.parametrize("S", [1, 2, 3, 4, 8, 9])
@pytest.mark.parametrize("k", [1, 2, 3, 4, 8, 16])
def test_canonical_closed_form_attains_bound(S, k):
    """Under unit times stage s runs F x (d_s+1), then (B,F) pairs, then the remaining Bs, so between
    F_m and B_m exactly the backwards m-d_s .. m-1 complete:
        delta[s][m] = floor(m/k) - floor(max(m-d_s,0)/k),
    which reaches ceil(d_s/k) -- the bound of Eq. 10 is tight."""
    n = 48
    r = schedule.simulate(S, n, k)
    for s in range(S):
        d = S - 1 - s
        assert r["max_q"][s] == min(d + 1, n)
        for m in range(n):
            assert r["delta"][s][m] == m // k - max(m - d, 0) // k
        if n > d + k:
            assert max(r["delta"][s]) == schedule.delta_bound(S, s + 1, k)


def test_paper_configuration_k_sweep():
    """N=8: max crossed updates for a = 1, 2, 4, 8 is ceil(7/a); P:144 prints a=4 -> 2, a=8 -> 1."""
    got = {k: max(max(d) for d in schedule.simulate(8, 32, k)["delta"]) for k in (1, 2, 4, 8)}
    assert got == {1: 7, 2: 4, 4: 2, 8: 1}
    assert got[4] == GOLD["bound N=8 a=4"] and got[8] == GOLD["bound N=8 a=8"]
    r = schedule.simulate(8, 16, 4)
    assert r["delta"][0] == [0, 0, 0, 0, 1, 1, 1, 1, 2, 2, 2, 1, 2, 2, 2, 1]
    assert r["max_q"][0] == GOLD["inflight first N=8"] and r["max_q"][7] == GOLD["inflight last N=8"]


@pytest.mark.parametrize("m_f", [1, 2, 4, 8])
def test_flush_has_no_drift_and_follows_eq3(m_f):
    """Flush: delta == 0.  With equal op times a flush group takes (m_f+N-1)(tF+tB) and PACI's
    steady state m_f (tF+tB) per m_f micro-batches, so the throughput ratio is Eq. 3."""
    S, groups, tF, tB = 8, 40, 2, 3
    n = m_f * groups
    rf = schedule.simulate(S, n, None, tF=[tF] * S, tB=[tB] * S, mode="flush", m_f=m_f)
    rp = schedule.simulate(S, n, m_f, tF=[tF] * S, tB=[tB] * S)
    assert all(d == 0 for row in rf["delta"] for d in row)
    assert rf["version"] == [groups] * S
    assert rf["makespan"] == groups * (m_f + S - 1) * (tF + tB)
    assert rp["makespan"] == n * (tF + tB) + (S - 1) * (tF + tB)
    steady_paci = m_f * (tF + tB)
    assert abs(steady_paci / (rf["makespan"] / groups) - schedule.eta_flush(m_f, S)) < 1e-15


def test_single_window_never_crosses():
    """Exactly k micro-batches: the only update comes after the last backward, so delta == 0 and
    PACI's op order equals flush with m_f = k."""
    for S in (1, 2, 4):
        a = schedule.simulate(S, 4, 4)
        b = schedule.simulate(S, 4, None, mode="flush", m_f=4)
        assert a["ops"] == b["ops"] and all(d == 0 for row in a["delta"] for d in row)
