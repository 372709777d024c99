/* arachne_sched.h — C ABI of libarachne_sched.so: the cascade-level planner pieces of the paper that consume this
 * repository's measured attention cost.  HOST code only (no GPU): all pointers are host memory.
 *
 * Problem (Eqs. 1-7): n cascades c with direct predecessors P_c; each picks ONE parallelism degree
 * K[j] (x_{c,j}); latency L[c][j]; e_c = s_c + L (Eq. 2); s_c >= e_p for p in P_c (Eq. 4); a degree is allowed for a
 * cascade iff feasible[c][j] != 0 (memory, Eq. 6) and K[j] <= N; at every time the degrees of the running cascades sum
 * to <= N (Eq. 7); minimise the makespan T = max e_c (Eqs. 1, 3).
 * Method (Alg. 1): a genetic algorithm over the degree assignment whose fitness is the makespan of a
 * list scheduler that prioritises the critical path.  Everything the paper leaves open is fixed by readings R23-R27
 * (restated in oracle/cascade_sched_oracle.py, the independent Python oracle these functions are tested
 * against value for value).
 *
 * Layout: L and feasible are row-major [n][nk].  Predecessors in CSR form: pred_ptr[n+1], pred_idx[pred_ptr[n]].
 * Return: 0 ok; 1 null pointer; 2 bad argument (n <= 0, nk <= 0, degree <= 0 or > N, index out of range, p < 2,
 * eps > p, ...); 3 a cascade has no feasible degree; 4 the dependency graph has a cycle.  Nothing is allocated
 * that outlives a call; the caller owns every array. */
#ifndef ARACHNE_SCHED_H_
#define ARACHNE_SCHED_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* List scheduler (R23, R24) for ONE degree assignment.
 *   lat[n], deg[n]        : chosen latency and degree of every cascade
 *   start[n], end[n] (out): s_c, e_c;  *makespan (out): T */
int arachne_list_schedule(int32_t n, const double* lat, const int32_t* deg, const int32_t* pred_ptr,
                          const int32_t* pred_idx, int32_t num_gpus, double* start, double* end, double* makespan);

/* Genetic algorithm of Alg. 1 (R25-R27): population p, G generations, mutation rate mu, elitism size eps, counter-based
 * random numbers from `seed`.
 *   best_choice[n] (out): index j into K of the best chromosome;  start[n], end[n], *makespan: its schedule;
 *   history[G] (out, nullable): T* after each generation (non-increasing). */
int arachne_ga_schedule(int32_t n, int32_t nk, const int32_t* K, const double* L, const uint8_t* feasible,
                        const int32_t* pred_ptr, const int32_t* pred_idx, int32_t num_gpus, int32_t p, int32_t G,
                        double mu, int32_t eps, uint64_t seed, int32_t* best_choice, double* start, double* end,
                        double* makespan, double* history);

/* The uniform of R27 (exported so that tests can compare it with the oracle's bit for bit). */
double arachne_sched_uniform(uint64_t seed, uint64_t gen, uint64_t child, uint64_t gene, uint64_t purpose);

#ifdef __cplusplus
}
#endif
#endif /* ARACHNE_SCHED_H_ */
