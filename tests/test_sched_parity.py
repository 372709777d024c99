"""CPU parity: libarachne_sched.so (C++, include/arachne_sched.h) against oracle/cascade_sched_oracle.py on the same seeded
instances — schedules, chromosomes and makespans VALUE FOR VALUE (same counter-based random numbers, R27; same fp64
operation order, -ffp-contract=off), plus the ABI's error codes."""
import ctypes
import os
import re

import pytest

from oracle import cascade_sched_oracle as so
from paper_2607_01701_b200 import inputs, scheduler

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_exports_every_declared_symbol():
    src = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", "arachne_sched.h")).read(), flags=re.S)
    names = sorted(set(re.findall(r"\b(arachne_[a-z0-9_]+)\s*\(", src)))
    assert names == sorted(scheduler.EXPORTS)
    for n in names:
        assert hasattr(scheduler._lib, n)


def test_uniform_bit_for_bit():
    for args in [(0, 0, 0, 0, 0), (7, 1, 2, 3, 4), (2**63 + 5, 99, 1000, 17, 5), (1, 2, 3, 4, 5)]:
        assert scheduler.uniform(*args) == so.uniform(*args)


@pytest.mark.parametrize("seed", range(6))
def test_list_schedule_equals_oracle(seed):
    inst = inputs.cascade_instance(seed, n_samples=5 + 3 * seed)
    K, L, preds, N = inst["K"], inst["L"], inst["preds"], inst["N"]
    n = len(L)
    for pick in (0, -1, seed % 2):
        ch = [[j for j in range(len(K)) if inst["feasible"][c][j]][pick if pick < 1 else min(pick, sum(inst["feasible"][c]) - 1)] for c in range(n)]
        lat, deg = [L[c][ch[c]] for c in range(n)], [K[ch[c]] for c in range(n)]
        assert scheduler.list_schedule(lat, deg, preds, N) == so.list_schedule(lat, deg, preds, N)


@pytest.mark.parametrize("seed,n_samples,p,G,mu,eps", [(0, 4, 8, 5, 0.2, 1), (1, 10, 32, 12, 0.1, 2), (2, 16, 24, 8, 0.05, 4),
                                                       (3, 3, 24, 12, 0.2, 2), (4, 25, 16, 6, 0.3, 0)])
def test_genetic_equals_oracle(seed, n_samples, p, G, mu, eps):
    inst = inputs.cascade_instance(seed, n_samples=n_samples)
    args = (inst["K"], inst["L"], inst["feasible"], inst["preds"], inst["N"])
    got = scheduler.genetic(*args, p=p, G=G, mu=mu, eps=eps, seed=100 + seed)
    ref = so.genetic(*args, p=p, G=G, mu=mu, eps=eps, seed=100 + seed)
    assert got[0] == ref[0] and got[1] == ref[1] and got[2] == ref[2] and got[3] == ref[3] and got[4] == ref[4]


def test_error_codes():
    with pytest.raises(scheduler.SchedError) as e:
        scheduler.list_schedule([1.0], [5], [[]], 4)
    assert e.value.status == 2
    with pytest.raises(scheduler.SchedError) as e:
        scheduler.list_schedule([1.0, 1.0], [1, 1], [[1], [0]], 4)        # cycle
    assert e.value.status == 4
    with pytest.raises(scheduler.SchedError) as e:
        scheduler.genetic([1, 2], [[1.0, 0.6]], [[False, False]], [[]], 4, p=4, G=2, mu=0.1, eps=1, seed=0)
    assert e.value.status == 3
    with pytest.raises(scheduler.SchedError) as e:
        scheduler.genetic([1, 2], [[1.0, 0.6]], [[True, True]], [[]], 4, p=1, G=2, mu=0.1, eps=1, seed=0)
    assert e.value.status == 2
    assert scheduler._lib.arachne_list_schedule(1, None, None, None, None, 1, None, None, None) == 1
