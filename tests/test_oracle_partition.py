"""Pins for oracle/partition.py (App. D.5, Eq. 12-15) and parity of the library's paci_partition (host code behind
the C ABI, no GPU needed) against it.  The oracle's DP is pinned by brute-force enumeration of every cut set."""
import ctypes as C
import math

import numpy as np
import pytest

from oracle import partition as opart


def _random_problem(rng, L):
    t = rng.uniform(0.5, 3.0, L).tolist()
    s = rng.uniform(1.0, 4.0, L).tolist()
    a = rng.uniform(0.2, 1.5, L).tolist()
    return t, s, a


def test_in_flight_count_is_N_minus_j_plus_1():
    """"the first stage carries N microbatches, the last carries one" (the printed formula is garbled, R20)."""
    N = 8
    assert opart.stage_memory(1, N, 0.0, 1.0) == 8.0 and opart.stage_memory(N, N, 0.0, 1.0) == 1.0
    assert opart.stage_memory(3, N, 5.0, 2.0) == 5.0 + 6 * 2.0            # Eq. 12: static once, activations w_j times


@pytest.mark.parametrize("seed", range(30))
def test_first_pass_is_the_exact_constrained_min_max(seed):
    rng = np.random.default_rng(seed)
    L, N = int(rng.integers(4, 12)), int(rng.integers(2, 5))
    t, s, a = _random_problem(rng, L)
    # a budget between "comfortable" and "tight": some instances infeasible, some binding, some slack
    budget = float(rng.uniform(0.5, 1.6) * (sum(s) + N * sum(a)) / N)
    got = opart.partition(t, s, a, N, budget)
    best_t, best_o = opart.brute_force(t, s, a, N, budget)
    cuts = got["cuts"]
    assert cuts[0] == 0 and cuts[-1] == L and all(x < y for x, y in zip(cuts, cuts[1:]))
    wt, wo = opart.evaluate(cuts, t, s, a, budget)
    assert abs(wt - got["max_time"]) < 1e-12 and abs(wo - got["max_overshoot"]) < 1e-9
    if best_t is not None:
        assert not got["fallback"] and abs(got["max_time"] - best_t) < 1e-12     # Eq. 13's optimum
    else:
        assert got["fallback"] and abs(got["max_overshoot"] - best_o) < 1e-9      # "minimizes the worst overshoot first"


def test_unconstrained_case_reduces_to_linear_partitioning_and_budget_binds():
    t = [1, 1, 1, 1, 4, 1, 1, 1]
    s = [1] * 8
    a = [1] * 8
    free = opart.partition(t, s, a, 3, 1e9)
    assert free["max_time"] == 4 and not free["fallback"]                   # textbook min-max: {1,1,1,1}{4}{1,1,1}
    # the first stage holds N = 3 in-flight micro-batches: 4 layers there cost 4 + 3*4 = 16
    tight = opart.partition(t, s, a, 3, 15.0)
    assert not tight["fallback"] and tight["cuts"][1] <= 3 and tight["max_time"] > 4
    none = opart.partition(t, s, a, 3, 5.0)
    assert none["fallback"] and none["max_overshoot"] > 0


@pytest.fixture(scope="module")
def pb():
    from paper_2606_07881_b200 import build
    build.build(verbose=False)
    from paper_2606_07881_b200 import binding
    return binding


@pytest.mark.parametrize("seed", range(40))
def test_library_partitioner_matches_oracle(pb, seed):
    rng = np.random.default_rng(1000 + seed)
    L, N = int(rng.integers(3, 40)), int(rng.integers(1, 9))
    N = min(N, L)
    t, s, a = _random_problem(rng, L)
    budget = float(rng.uniform(0.4, 1.8) * (sum(s) + N * sum(a)) / N)
    ref = opart.partition(t, s, a, N, budget)
    got = pb.partition(t, s, a, N, budget)
    assert got["fallback"] == ref["fallback"]
    assert abs(got["max_time"] - ref["max_time"]) < 1e-12 and abs(got["max_overshoot"] - ref["max_overshoot"]) < 1e-9
    assert got["cuts"] == ref["cuts"]                                        # same DP, same tie-breaking (first minimum)


def test_library_partitioner_rejects_bad_input(pb):
    with pytest.raises(pb.PaciError):
        pb.partition([1.0, 2.0], [1.0, 1.0], [1.0, 1.0], 3, 10.0)           # fewer layers than stages
