"""Oracle for the cascade planner pieces: list scheduler + genetic algorithm of Alg. 1
— TEST INFRASTRUCTURE, NOT PRODUCT CODE (only tests/ may import it; it imports nothing from the package).

What the paper fixes (Eqs. 1-7; Alg. 1 and the paragraph after it):
  * cascades c with direct predecessors P_c; a parallelism degree k in K per cascade (x_{c,k}), latency L_{c,k};
    e_c = s_c + L_{c,k} (Eq. 2); s_c >= e_p for p in P_c (Eq. 4); memory Mem_{c,k} <= W (Eq. 6: a degree is FEASIBLE
    or not, per cascade); at every time the degrees of the active cascades sum to at most N GPUs (Eq. 7);
    objective: makespan T = max e_c (Eqs. 1, 3).
  * a chromosome "encodes a complete assignment of parallelism degrees for all cascades"; its fitness is the
    makespan found by "a fast list scheduler that heuristically determines launch times by prioritizing the
    critical path"; the population "evolves through elitism, crossover, and mutation"; hyper-parameters p, G, mu, eps.
What it leaves open — readings (R23-R27):
  R23 priority of a cascade = length of the longest path from its start to a sink under the chosen latencies
      (its own latency included); ties -> lower cascade index.
  R24 list scheduling: at each event time, scan the READY cascades (all predecessors ended) in priority order and
      launch every one whose degree fits in the free GPUs (a blocked high-priority cascade does not block smaller
      ones); then advance to the earliest end time.
  R25 initial population: chromosome 0 = the smallest feasible degree everywhere, chromosome 1 = the largest; the
      rest uniform over the feasible degrees of each cascade.
  R26 next generation: the eps best chromosomes (by makespan, ties -> lower index) are copied; every other child
      takes each gene from one of two parents (uniform crossover), the parents each being the better of two uniformly
      drawn chromosomes (binary tournament); then each gene is redrawn uniformly from its feasible degrees with
      probability mu.
  R27 random numbers: u(seed, generation, child, gene, purpose) from a SplitMix64 counter hash -> 53-bit uniform in
      [0, 1); both implementations draw exactly these, so runs are comparable gene for gene.
Plain Python loops on purpose: instances are small (tens of cascades).
"""
from __future__ import annotations

M64 = (1 << 64) - 1


def _mix(z: int) -> int:
    z = (z + 0x9E3779B97F4A7C15) & M64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & M64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & M64
    return z ^ (z >> 31)


def uniform(seed: int, gen: int, child: int, gene: int, purpose: int) -> float:
    """R27.  purpose: 0 init, 1 tournament A, 2 tournament B, 3 crossover, 4 mutate?, 5 mutate value."""
    z = _mix(seed & M64)
    for v in (gen, child, gene, purpose):
        z = _mix(z ^ ((v + 1) & M64))
    return (z >> 11) / float(1 << 53)


def critical_path(lat, succs):
    """R23: longest path to a sink, own latency included.  lat[c] chosen latency; succs[c] direct successors."""
    n = len(lat)
    cp = [None] * n

    def go(c):
        if cp[c] is None:
            cp[c] = lat[c] + max([go(s) for s in succs[c]], default=0.0)
        return cp[c]

    for c in range(n):
        go(c)
    return cp


def list_schedule(lat, deg, preds, N):
    """R24.  lat[c], deg[c]: chosen latency and degree; preds[c]: direct predecessors; N GPUs.
    Returns (start[], end[], makespan).  Raises if a degree exceeds N."""
    n = len(lat)
    if any(d > N or d <= 0 for d in deg):
        raise ValueError("degree outside (0, N]")
    succs = [[] for _ in range(n)]
    for c in range(n):
        for p in preds[c]:
            succs[p].append(c)
    prio = critical_path(lat, succs)
    start, end = [None] * n, [None] * n
    free, t, done = N, 0.0, 0
    running = []
    while done < n:
        ready = [c for c in range(n) if start[c] is None and all(end[p] is not None and end[p] <= t for p in preds[c])]
        ready.sort(key=lambda c: (-prio[c], c))
        for c in ready:
            if deg[c] <= free:
                start[c], end[c] = t, t + lat[c]
                free -= deg[c]
                running.append(c)
        if not running:
            raise RuntimeError("deadlock: nothing running and nothing fits (cyclic dependencies?)")
        t = min(end[c] for c in running)
        for c in [c for c in running if end[c] <= t]:
            running.remove(c)
            free += deg[c]
            done += 1
    return start, end, max(end)


def genetic(K, L, feasible, preds, N, p, G, mu, eps, seed):
    """Alg. 1.  K[j]: the degrees; L[c][j]: latency of cascade c at degree K[j]; feasible[c][j]: Eq. 6 (and K[j] <= N).
    Returns (best makespan T*, best chromosome (degree INDEX per cascade), start[], end[], history of T* per generation)."""
    n = len(L)
    feas = [[j for j in range(len(K)) if feasible[c][j] and K[j] <= N] for c in range(n)]
    if any(not f for f in feas):
        raise ValueError("a cascade has no feasible degree")

    def draw(c, u):
        return feas[c][min(int(u * len(feas[c])), len(feas[c]) - 1)]

    def fitness(ch):
        lat = [L[c][ch[c]] for c in range(n)]
        deg = [K[ch[c]] for c in range(n)]
        return list_schedule(lat, deg, preds, N)

    pop = []
    for i in range(p):                                                       # R25
        if i == 0:
            pop.append([f[0] for f in feas])
        elif i == 1:
            pop.append([f[-1] for f in feas])
        else:
            pop.append([draw(c, uniform(seed, 0, i, c, 0)) for c in range(n)])
    best_T, best_ch, best_s, best_e, hist = float("inf"), None, None, None, []
    for g in range(1, G + 1):
        fit = [fitness(ch) for ch in pop]                                    # Alg. 1 line 7
        T = [f[2] for f in fit]
        i_best = min(range(p), key=lambda i: (T[i], i))                      # line 8
        if T[i_best] < best_T:                                               # lines 9-12
            best_T, best_ch, best_s, best_e = T[i_best], list(pop[i_best]), fit[i_best][0], fit[i_best][1]
        hist.append(best_T)
        order = sorted(range(p), key=lambda i: (T[i], i))                    # line 13, R26
        nxt = [list(pop[i]) for i in order[:eps]]
        for child in range(eps, p):
            def tournament(purpose):
                a = min(int(uniform(seed, g, child, 0, purpose) * p), p - 1)
                b = min(int(uniform(seed, g, child, 1, purpose) * p), p - 1)
                return a if (T[a], a) <= (T[b], b) else b
            pa, pb = tournament(1), tournament(2)
            ch = [pop[pa][c] if uniform(seed, g, child, c, 3) < 0.5 else pop[pb][c] for c in range(n)]
            for c in range(n):
                if uniform(seed, g, child, c, 4) < mu:
                    ch[c] = draw(c, uniform(seed, g, child, c, 5))
            nxt.append(ch)
        pop = nxt
    return best_T, best_ch, best_s, best_e, hist


def brute_force(K, L, feasible, preds, N):
    """Best list-scheduler makespan over ALL chromosomes (tiny instances only): the GA's search space, exhaustively."""
    import itertools

    n = len(L)
    feas = [[j for j in range(len(K)) if feasible[c][j] and K[j] <= N] for c in range(n)]
    best = (float("inf"), None)
    for ch in itertools.product(*feas):
        T = list_schedule([L[c][ch[c]] for c in range(n)], [K[ch[c]] for c in range(n)], preds, N)[2]
        if T < best[0]:
            best = (T, list(ch))
    return best
