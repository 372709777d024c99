"""CPU pins of oracle/cascade_sched_oracle.py: what the paper's formulation fixes (PAPER.md:145-195,
Eqs. 1-7; Alg. 1), closed forms, invariants and brute force on tiny instances."""
import itertools

import pytest

from oracle import cascade_sched_oracle as so
from paper_2607_01701_b200 import inputs


def _check_valid(lat, deg, preds, N, s, e, T):
    n = len(lat)
    for c in range(n):
        assert e[c] == s[c] + lat[c]                                     # Eq. 2
        for p in preds[c]:
            assert s[c] >= e[p]                                          # Eq. 4
    assert T == max(e)                                                   # Eqs. 1, 3
    for t in sorted(set(s)):                                             # Eq. 7 can only be violated at a launch time
        assert sum(deg[c] for c in range(n) if s[c] <= t < e[c]) <= N


def test_closed_forms():
    # all cascades need every GPU -> serial; independent unit-degree cascades on enough GPUs -> the longest one
    lat = [3.0, 1.0, 2.5, 0.5]
    assert so.list_schedule(lat, [4] * 4, [[]] * 4, 4)[2] == sum(lat)
    assert so.list_schedule(lat, [1] * 4, [[]] * 4, 4)[2] == max(lat)
    # a chain is serial whatever the degrees; a diamond: longest path
    assert so.list_schedule(lat, [1, 2, 1, 2], [[], [0], [1], [2]], 8)[2] == sum(lat)
    s, e, T = so.list_schedule([1.0, 2.0, 5.0, 1.0], [1, 1, 1, 1], [[], [0], [0], [1, 2]], 4)
    assert T == 1.0 + 5.0 + 1.0 and s[3] == 6.0
    # critical-path priority: with 1 GPU free at t = 0 the cascade heading the longer chain goes first
    s, e, T = so.list_schedule([1.0, 1.0, 10.0], [1, 1, 1], [[], [], [1]], 1)
    assert s[1] == 0.0 and s[2] == 1.0 and s[0] == 11.0 and T == 12.0   # 1 heads the 11-long chain; then 2 (10) outranks 0 (1)
    # the motivating shape of PAPER.md:41: one long cascade and several short ones on 16 GPUs in 4 groups of 4:
    # the long one alone sets the makespan; packing the short ones beside it costs nothing
    lat = [58.6, 6.0, 6.0, 6.0, 6.0, 6.0, 6.0]
    assert so.list_schedule(lat, [4] * 7, [[]] * 7, 16)[2] == 58.6
    with pytest.raises(ValueError):
        so.list_schedule([1.0], [5], [[]], 4)


def test_list_schedule_invariants_and_bounds_on_seeded_instances():
    for seed in range(6):
        inst = inputs.cascade_instance(seed, n_samples=6 + seed)
        K, L, preds, N = inst["K"], inst["L"], inst["preds"], inst["N"]
        n = len(L)
        for pick in (0, -1):
            ch = [[j for j in range(len(K)) if inst["feasible"][c][j]][pick] for c in range(n)]
            lat, deg = [L[c][ch[c]] for c in range(n)], [K[ch[c]] for c in range(n)]
            s, e, T = so.list_schedule(lat, deg, preds, N)
            _check_valid(lat, deg, preds, N, s, e, T)
            succs = [[d for d in range(n) if c in preds[d]] for c in range(n)]
            assert T >= max(so.critical_path(lat, succs)) - 1e-12      # no schedule beats the longest chain
            assert T >= sum(l * d for l, d in zip(lat, deg)) / N - 1e-12   # ... nor the GPU-time / N bound


def test_list_schedule_against_exhaustive_order_search_tiny():
    # 5 independent cascades, degrees 2,2,1,3,2 on 4 GPUs: optimum over ALL launch orders (serial generation scheme)
    lat, deg, N = [4.0, 3.0, 2.0, 2.0, 1.0], [2, 2, 1, 3, 2], 4
    best = float("inf")
    for order in itertools.permutations(range(5)):
        t_free = []          # (end, deg) of running
        now, running, T = 0.0, [], 0.0
        for c in order:
            while sum(d for _, d in running) + deg[c] > N:
                now = min(e for e, _ in running)
                running = [(e, d) for e, d in running if e > now]
            running.append((now + lat[c], deg[c])); T = max(T, now + lat[c])
        best = min(best, T)
    T = so.list_schedule(lat, deg, [[]] * 5, N)[2]
    assert best <= T <= 2 * best                                         # Graham-type bound for list scheduling
    assert T == 7.0 and best == 6.0       # computed by hand: LPT order 0,1 | 2 .. ; the heuristic is not optimal here


def test_rng_is_a_fixed_function():
    u = so.uniform(7, 1, 2, 3, 4)
    assert 0.0 <= u < 1.0 and u == so.uniform(7, 1, 2, 3, 4) and u != so.uniform(7, 1, 2, 3, 5)
    xs = [so.uniform(1, g, c, 0, 0) for g in range(20) for c in range(50)]
    assert abs(sum(xs) / len(xs) - 0.5) < 0.03


def test_genetic_matches_brute_force_on_tiny_and_never_gets_worse():
    inst = inputs.cascade_instance(3, n_samples=3, degrees=(1, 2, 4), n_gpus=4)
    args = (inst["K"], inst["L"], inst["feasible"], inst["preds"], inst["N"])
    opt_T, _ = so.brute_force(*args)
    T, ch, s, e, hist = so.genetic(*args, p=24, G=12, mu=0.2, eps=2, seed=5)
    assert all(b <= a for a, b in zip(hist, hist[1:]))                   # elitism: T* never increases
    assert T == hist[-1] == opt_T                                        # 3^6 = 729 chromosomes: found
    lat, deg = [inst["L"][c][ch[c]] for c in range(len(ch))], [inst["K"][ch[c]] for c in range(len(ch))]
    s2, e2, T2 = so.list_schedule(lat, deg, inst["preds"], inst["N"])
    assert (s2, e2, T2) == (s, e, T)                                     # the returned schedule IS the chromosome's
    _check_valid(lat, deg, inst["preds"], inst["N"], s, e, T)
    assert all(inst["feasible"][c][ch[c]] for c in range(len(ch)))       # Eq. 6
    # bigger instance: better than both seed heuristics (all-min and all-max degree), which are chromosomes 0 and 1
    inst = inputs.cascade_instance(1, n_samples=10)
    args = (inst["K"], inst["L"], inst["feasible"], inst["preds"], inst["N"])
    T, ch, s, e, hist = so.genetic(*args, p=32, G=25, mu=0.1, eps=2, seed=1)
    assert T <= hist[0]
