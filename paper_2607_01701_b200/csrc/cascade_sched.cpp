// libarachne_sched.so — list scheduler + genetic algorithm for cascade scheduling (include/arachne_sched.h).
// Host-only C++; event-driven list scheduling with a heap of running cascades and indegree counting, fitness of a
// generation evaluated in parallel (OpenMP; every chromosome is independent, so the result does not depend on threads).
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <functional>
#include <limits>
#include <queue>
#include <utility>
#include <vector>

#include "../../include/arachne_sched.h"

namespace {

inline uint64_t mix(uint64_t z) {
  z += 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

// R27: u(seed, generation, child, gene, purpose), 53-bit uniform in [0, 1)
inline double uniform(uint64_t seed, uint64_t gen, uint64_t child, uint64_t gene, uint64_t purpose) {
  uint64_t z = mix(seed);
  z = mix(z ^ (gen + 1));
  z = mix(z ^ (child + 1));
  z = mix(z ^ (gene + 1));
  z = mix(z ^ (purpose + 1));
  return static_cast<double>(z >> 11) / 9007199254740992.0;
}

struct Graph {
  int n = 0;
  std::vector<int> succ_ptr, succ_idx, indeg, topo;   // successors in CSR form; a topological order
};

// returns false on a cycle or an out-of-range predecessor
bool build_graph(int n, const int32_t* pred_ptr, const int32_t* pred_idx, Graph& g) {
  g.n = n;
  g.indeg.assign(n, 0);
  g.succ_ptr.assign(n + 1, 0);
  for (int c = 0; c < n; ++c) {
    if (pred_ptr[c + 1] < pred_ptr[c]) return false;
    for (int e = pred_ptr[c]; e < pred_ptr[c + 1]; ++e) {
      const int p = pred_idx[e];
      if (p < 0 || p >= n || p == c) return false;
      ++g.succ_ptr[p + 1];
      ++g.indeg[c];
    }
  }
  for (int c = 0; c < n; ++c) g.succ_ptr[c + 1] += g.succ_ptr[c];
  g.succ_idx.assign(g.succ_ptr[n], 0);
  std::vector<int> fill(g.succ_ptr.begin(), g.succ_ptr.end() - 1);
  for (int c = 0; c < n; ++c)
    for (int e = pred_ptr[c]; e < pred_ptr[c + 1]; ++e) g.succ_idx[fill[pred_idx[e]]++] = c;
  std::vector<int> deg(g.indeg);
  g.topo.clear();
  for (int c = 0; c < n; ++c)
    if (deg[c] == 0) g.topo.push_back(c);
  for (size_t i = 0; i < g.topo.size(); ++i) {
    const int c = g.topo[i];
    for (int e = g.succ_ptr[c]; e < g.succ_ptr[c + 1]; ++e)
      if (--deg[g.succ_idx[e]] == 0) g.topo.push_back(g.succ_idx[e]);
  }
  return static_cast<int>(g.topo.size()) == n;
}

// R23 + R24.  Returns the makespan; start/end may be null (fitness only).
double list_schedule(const Graph& g, const double* lat, const int32_t* deg, int num_gpus, double* start, double* end) {
  const int n = g.n;
  std::vector<double> prio(n);
  for (int i = n - 1; i >= 0; --i) {              // longest path to a sink, own latency included
    const int c = g.topo[i];
    double best = 0.0;
    for (int e = g.succ_ptr[c]; e < g.succ_ptr[c + 1]; ++e) best = std::max(best, prio[g.succ_idx[e]]);
    prio[c] = lat[c] + best;
  }
  auto before = [&](int a, int b) { return prio[a] > prio[b] || (prio[a] == prio[b] && a < b); };
  std::vector<int> waiting(g.indeg), ready;
  std::vector<double> e_loc(n);
  for (int c = 0; c < n; ++c)
    if (waiting[c] == 0) ready.push_back(c);
  std::sort(ready.begin(), ready.end(), before);
  using Run = std::pair<double, int>;             // (end time, cascade)
  std::priority_queue<Run, std::vector<Run>, std::greater<Run>> running;
  int free_gpus = num_gpus, done = 0;
  double t = 0.0, makespan = 0.0;
  while (done < n) {
    // launch, in priority order, every ready cascade that fits (a blocked one does not block the smaller ones)
    size_t keep = 0;
    for (size_t i = 0; i < ready.size(); ++i) {
      const int c = ready[i];
      if (deg[c] <= free_gpus) {
        free_gpus -= deg[c];
        e_loc[c] = t + lat[c];
        if (start) start[c] = t;
        if (end) end[c] = e_loc[c];
        makespan = std::max(makespan, e_loc[c]);
        running.push(Run(e_loc[c], c));
      } else {
        ready[keep++] = c;
      }
    }
    ready.resize(keep);
    if (running.empty()) return std::numeric_limits<double>::quiet_NaN();   // cannot happen for validated input
    t = running.top().first;
    bool grew = false;
    while (!running.empty() && running.top().first <= t) {
      const int c = running.top().second;
      running.pop();
      free_gpus += deg[c];
      ++done;
      for (int e = g.succ_ptr[c]; e < g.succ_ptr[c + 1]; ++e)
        if (--waiting[g.succ_idx[e]] == 0) { ready.push_back(g.succ_idx[e]); grew = true; }
    }
    if (grew) std::sort(ready.begin(), ready.end(), before);
  }
  return makespan;
}

}  // namespace

extern "C" {

double arachne_sched_uniform(uint64_t seed, uint64_t gen, uint64_t child, uint64_t gene, uint64_t purpose) {
  return uniform(seed, gen, child, gene, purpose);
}

int arachne_list_schedule(int32_t n, const double* lat, const int32_t* deg, const int32_t* pred_ptr, const int32_t* pred_idx,
                          int32_t num_gpus, double* start, double* end, double* makespan) {
  if (!lat || !deg || !pred_ptr || !start || !end || !makespan) return 1;
  if (n <= 0 || num_gpus <= 0) return 2;
  if (pred_ptr[n] > 0 && !pred_idx) return 1;
  for (int c = 0; c < n; ++c)
    if (deg[c] <= 0 || deg[c] > num_gpus || !(lat[c] >= 0.0)) return 2;
  Graph g;
  if (!build_graph(n, pred_ptr, pred_idx, g)) return 4;
  *makespan = list_schedule(g, lat, deg, num_gpus, start, end);
  return 0;
}

int arachne_ga_schedule(int32_t n, int32_t nk, const int32_t* K, const double* L, const uint8_t* feasible,
                        const int32_t* pred_ptr, const int32_t* pred_idx, int32_t num_gpus, int32_t p, int32_t G, double mu,
                        int32_t eps, uint64_t seed, int32_t* best_choice, double* start, double* end, double* makespan,
                        double* history) {
  if (!K || !L || !feasible || !pred_ptr || !best_choice || !start || !end || !makespan) return 1;
  if (n <= 0 || nk <= 0 || num_gpus <= 0 || p < 2 || G < 1 || eps < 0 || eps > p || !(mu >= 0.0 && mu <= 1.0)) return 2;
  if (pred_ptr[n] > 0 && !pred_idx) return 1;
  for (int j = 0; j < nk; ++j)
    if (K[j] <= 0) return 2;
  Graph g;
  if (!build_graph(n, pred_ptr, pred_idx, g)) return 4;
  // feasible degree indices per cascade (Eq. 6 and K[j] <= N), in the order of K
  std::vector<std::vector<int>> feas(n);
  for (int c = 0; c < n; ++c) {
    for (int j = 0; j < nk; ++j)
      if (feasible[static_cast<size_t>(c) * nk + j] && K[j] <= num_gpus) feas[c].push_back(j);
    if (feas[c].empty()) return 3;
  }
  auto draw = [&](int c, double u) {
    const int m = static_cast<int>(feas[c].size());
    return feas[c][std::min(static_cast<int>(u * m), m - 1)];
  };
  std::vector<std::vector<int>> pop(p, std::vector<int>(n)), nxt(p, std::vector<int>(n));
  for (int i = 0; i < p; ++i)                                             // R25
    for (int c = 0; c < n; ++c)
      pop[i][c] = i == 0 ? feas[c].front() : (i == 1 ? feas[c].back() : draw(c, uniform(seed, 0, i, c, 0)));
  std::vector<double> T(p);
  double best_T = std::numeric_limits<double>::infinity();
  std::vector<int> best(n), order(p);
  auto fitness = [&](const std::vector<int>& ch, double* s, double* e) {
    std::vector<double> lat(n);
    std::vector<int32_t> deg(n);
    for (int c = 0; c < n; ++c) { lat[c] = L[static_cast<size_t>(c) * nk + ch[c]]; deg[c] = K[ch[c]]; }
    return list_schedule(g, lat.data(), deg.data(), num_gpus, s, e);
  };
  for (int gen = 1; gen <= G; ++gen) {
#pragma omp parallel for schedule(dynamic)
    for (int i = 0; i < p; ++i) T[i] = fitness(pop[i], nullptr, nullptr);  // Alg. 1 line 7
    for (int i = 0; i < p; ++i) order[i] = i;
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return T[a] < T[b]; });   // ties -> lower index
    if (T[order[0]] < best_T) { best_T = T[order[0]]; best = pop[order[0]]; }                 // lines 8-12
    if (history) history[gen - 1] = best_T;
    for (int i = 0; i < eps; ++i) nxt[i] = pop[order[i]];                                      // line 13, R26
    for (int child = eps; child < p; ++child) {
      auto tournament = [&](uint64_t purpose) {
        const int a = std::min(static_cast<int>(uniform(seed, gen, child, 0, purpose) * p), p - 1);
        const int b = std::min(static_cast<int>(uniform(seed, gen, child, 1, purpose) * p), p - 1);
        return (T[a] < T[b] || (T[a] == T[b] && a <= b)) ? a : b;
      };
      const int pa = tournament(1), pb = tournament(2);
      for (int c = 0; c < n; ++c) {
        int gene = uniform(seed, gen, child, c, 3) < 0.5 ? pop[pa][c] : pop[pb][c];
        if (uniform(seed, gen, child, c, 4) < mu) gene = draw(c, uniform(seed, gen, child, c, 5));
        nxt[child][c] = gene;
      }
    }
    pop.swap(nxt);
  }
  for (int c = 0; c < n; ++c) best_choice[c] = best[c];
  *makespan = fitness(best, start, end);
  return 0;
}

}  // extern "C"
