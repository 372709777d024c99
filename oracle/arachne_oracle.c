/* arachne_oracle.c — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU definition of what libarachne_attn computes.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build,
 * load or call this file.  It shares no code, header, table or constant with
 * paper_2607_01701_b200/csrc and neither side includes the other.
 *
 * What it follows.  The paper names the operation — "full self-attention over a unified
 * sequence of 3D patches of length L ... O(L^2)" (§III Obs. 2; Eq. 9
 * PAPER.md:212-214) — but prints no formula for it, nor for QK-RMSNorm / 3D RoPE.  The
 * method is EXACT softmax attention (no approximation), so this file is that textbook
 * definition written out, with the readings R1-R18 of DESIGN.md §3 (from BASELINE.json
 * north_star / configs[0]) for everything the paper leaves open.  Each step cites its
 * reading.  No tiling, no online softmax, no fusion: every score of a row is computed,
 * the row maximum is subtracted only for fp64 safety, then exp / sum / normalise.
 *
 * Pins (tests/test_oracle_*.py, all "-m 'not gpu'"): brute-force triple loop written
 * independently in the test; rows of P sum to 1 and V==1 => O==1; packed == each sequence
 * alone; permutation of sequences; central finite differences of l = sum(O*dO); equality
 * with torch SDPA (fp64) when norm and RoPE are off, and with a torch fp64 autograd
 * composite when on; closed forms (L=1, Q==0); RMSNorm scale invariance; RoPE norm
 * preservation / shift invariance / axis distinguishability; sum_j dV_j = sum_i dO_i;
 * row-subset + masked-dO mode == full mode restricted.  Joint text tokens (R21): brute force
 * with its own is-text switch, equality with the no-RoPE run when every token sits at the
 * origin, torch autograd composite.  dgamma (R22): finite differences in gamma, torch
 * autograd, and the invariant sum_d gq_d dGq_d == sum_d gk_d dGk_d (the loss is unchanged
 * by gamma_q -> c gamma_q, gamma_k -> gamma_k / c).
 *
 * One function does one (sequence, head) problem on gathered fp64 arrays; the Python
 * wrapper (oracle/arachne_oracle.py) loops over sequences and heads.  OpenMP over rows /
 * keys only (independent iterations; no reduction across threads).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
  int D;               /* head_dim                                                     */
  int rope_dims[3];    /* (d_t, d_h, d_w), R4/R6                                        */
  double theta;        /* R5                                                            */
  double eps;          /* R2                                                            */
  double scale;        /* softmax scale, R8 (caller passes 1/sqrt(D) by default)        */
  int no_norm;         /* debug: x^ = x                                                 */
  int no_rope;         /* debug: x~ = x^                                                */
  int pos_offset[3];   /* added to every (t,h,w) position (RoPE shift-invariance pin)   */
} oracle_cfg;

int arachne_oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* R7: token n (0-based inside its sequence) sits at (t,h,w) of a row-major [T,Hg,Wg] grid. */
static void token_pos(const oracle_cfg* c, const int grid[3], int n, int pos[3]) {
  const int Hg = grid[1], Wg = grid[2];
  pos[0] = n / (Hg * Wg) + c->pos_offset[0];
  pos[1] = (n / Wg) % Hg + c->pos_offset[1];
  pos[2] = n % Wg + c->pos_offset[2];
}

/* R1-R5: x~ = RoPE(gamma * x / sqrt(mean(x^2) + eps)).  Returns r = 1/sqrt(mean+eps). */
static double norm_rope_row(const oracle_cfg* c, const double* x, const double* gamma,
                            const int pos[3], int is_text, double* xt) {
  const int D = c->D;
  double r = 1.0;
  if (!c->no_norm) {
    double ms = 0.0;
    for (int d = 0; d < D; ++d) ms += x[d] * x[d];
    ms /= (double)D;                      /* R1: over head_dim, per (token, head)        */
    r = 1.0 / sqrt(ms + c->eps);          /* R2: eps inside the sqrt                     */
    for (int d = 0; d < D; ++d) xt[d] = gamma[d] * x[d] * r;
  } else {
    for (int d = 0; d < D; ++d) xt[d] = x[d];
  }
  if (!c->no_rope && !is_text) {          /* R3: norm, then RoPE; R21: text tokens are not rotated */
    int base = 0;
    for (int a = 0; a < 3; ++a) {         /* R4: contiguous axis slices, order t,h,w     */
      const int da = c->rope_dims[a];
      for (int p = 0; p < da / 2; ++p) {  /* R4: interleaved pair (2p, 2p+1)             */
        const double phi = (double)pos[a] * pow(c->theta, -2.0 * (double)p / (double)da); /* R5 */
        const double cs = cos(phi), sn = sin(phi);
        const double x0 = xt[base + 2 * p], x1 = xt[base + 2 * p + 1];
        xt[base + 2 * p] = x0 * cs - x1 * sn;
        xt[base + 2 * p + 1] = x0 * sn + x1 * cs;
      }
      base += da;
    }
  }
  return r;
}

/* Chain rule through norm_rope_row (R12): g~ = dl/dx~  ->  dl/dx.
 *   rotate each pair by -phi:  g0 = g~0 cos + g~1 sin ; g1 = -g~0 sin + g~1 cos
 *   u = gamma * g ;  dx_e = r u_e - r^3 x_e (sum_d u_d x_d) / D
 * (from x^_d = gamma_d x_d r, dr/dx_e = -r^3 x_e / D).
 * dx may be NULL (only the dgamma term wanted). */
static void norm_rope_row_bwd(const oracle_cfg* c, const double* x, const double* gamma,
                              const int pos[3], int is_text, double r, const double* gt, double* dx,
                              double* dgamma_row) {
  const int D = c->D;
  double* g = (double*)malloc(sizeof(double) * (size_t)D);
  for (int d = 0; d < D; ++d) g[d] = gt[d];
  if (!c->no_rope && !is_text) {
    int base = 0;
    for (int a = 0; a < 3; ++a) {
      const int da = c->rope_dims[a];
      for (int p = 0; p < da / 2; ++p) {
        const double phi = (double)pos[a] * pow(c->theta, -2.0 * (double)p / (double)da);
        const double cs = cos(phi), sn = sin(phi);
        const double g0 = gt[base + 2 * p], g1 = gt[base + 2 * p + 1];
        g[base + 2 * p] = g0 * cs + g1 * sn;
        g[base + 2 * p + 1] = -g0 * sn + g1 * cs;
      }
      base += da;
    }
  }
  if (!c->no_norm) {
    double ux = 0.0;
    for (int d = 0; d < D; ++d) ux += gamma[d] * g[d] * x[d];
    if (dx) for (int d = 0; d < D; ++d)
      dx[d] = r * gamma[d] * g[d] - r * r * r * x[d] * ux / (double)D;
    /* R22: x^_d = gamma_d x_d r  =>  this row's term of dl/dgamma_d is g_d x_d r */
    if (dgamma_row) for (int d = 0; d < D; ++d) dgamma_row[d] = g[d] * x[d] * r;
  } else {
    if (dx) for (int d = 0; d < D; ++d) dx[d] = g[d];
    if (dgamma_row) for (int d = 0; d < D; ++d) dgamma_row[d] = 0.0;   /* gamma unused */
  }
  free(g);
}

/* One (sequence, head) problem.
 *   R21 (joint text tokens; "hybrid dual/single-stream", PAPER.md:201
 *   text < 256 tokens): the sequence is the T*Hg*Wg video tokens of `grid` in row-major order followed by
 *   n_text text tokens (L = T*Hg*Wg + n_text).  Text tokens get the same QK-RMSNorm but NO RoPE; attention
 *   is full (bidirectional) over all L tokens.
 *   R22 (dgamma, NEXT-1): dGq[d] / dGk[d] = sum over the query / key rows of this problem of
 *   (R^T g~)_d x_d r, i.e. dl/dgamma_q, dl/dgamma_k restricted to this (sequence, head); the caller sums
 *   over sequences and heads (gamma is shared by all heads, R1).  Either may be NULL.
 *   L keys/values (all tokens 0..L-1 of the sequence), R query rows with in-sequence
 *   token indices qidx[0..R) (R == L and qidx[i] == i for the full problem).
 *   q  [R][D] raw query rows,   k, v [L][D] raw keys / values,   dO [R][D] or NULL.
 * Outputs (any may be NULL):
 *   O [R][D], LSE [R] (natural log, R9), P [R][L] (debug hook),
 *   dQ [R][D]  (exact for the given rows),
 *   dK, dV [L][D] = contributions of the given R rows only (== exact when R == L; this is
 *   the "masked-dO" quantity when R < L: dO is zero outside the row set).
 * Returns 0, or -1 on allocation failure / bad arguments. */
int arachne_oracle_head_joint(const oracle_cfg* c, const int grid[3], int n_text, int L, int R,
                              const int* qidx, const double* q, const double* k, const double* v,
                              const double* gamma_q, const double* gamma_k, const double* dO,
                              double* O, double* LSE, double* P, double* dQ, double* dK, double* dV,
                              double* dGq, double* dGk) {
  const int D = c->D;
  const int Lvid = grid[0] * grid[1] * grid[2];
  if (L < 1 || R < 1 || n_text < 0 || grid[0] < 0 || grid[1] < 1 || grid[2] < 1 || Lvid + n_text != L)
    return -1;                                        /* R16: L_b >= 1; a text-only sequence has T = 0 */
  const int need_bwd = (dO != NULL);
  double* kt = (double*)malloc(sizeof(double) * (size_t)L * D);   /* k~_j */
  double* rk = (double*)malloc(sizeof(double) * (size_t)L);
  double* qt = (double*)malloc(sizeof(double) * (size_t)R * D);   /* q~_i */
  double* rq = (double*)malloc(sizeof(double) * (size_t)R);
  double* Pm = (double*)malloc(sizeof(double) * (size_t)R * L);   /* P_ij */
  double* dS = need_bwd ? (double*)malloc(sizeof(double) * (size_t)R * L) : NULL;
  double* Oi = (double*)malloc(sizeof(double) * (size_t)R * D);
  /* per-row dgamma terms (summed serially afterwards: no cross-thread reduction) */
  double* dgq_rows = (need_bwd && dGq) ? (double*)malloc(sizeof(double) * (size_t)R * D) : NULL;
  double* dgk_rows = (need_bwd && dGk) ? (double*)malloc(sizeof(double) * (size_t)L * D) : NULL;
  if (!kt || !rk || !qt || !rq || !Pm || !Oi || (need_bwd && !dS) || (need_bwd && dGq && !dgq_rows) ||
      (need_bwd && dGk && !dgk_rows)) {
    free(kt); free(rk); free(qt); free(rq); free(Pm); free(dS); free(Oi); free(dgq_rows); free(dgk_rows);
    return -1;
  }

  /* step 1: k~_j for every key of the sequence (R1-R7, R10: V untouched) */
#pragma omp parallel for schedule(static)
  for (int j = 0; j < L; ++j) {
    int pos[3];
    token_pos(c, grid, j, pos);
    rk[j] = norm_rope_row(c, k + (size_t)j * D, gamma_k, pos, j >= Lvid, kt + (size_t)j * D);
  }

  /* step 2: per query row — scores, softmax, LSE, O (R8, R9, R11: no mask inside a sequence) */
#pragma omp parallel for schedule(dynamic, 4)
  for (int i = 0; i < R; ++i) {
    int pos[3];
    token_pos(c, grid, qidx[i], pos);
    double* qti = qt + (size_t)i * D;
    rq[i] = norm_rope_row(c, q + (size_t)i * D, gamma_q, pos, qidx[i] >= Lvid, qti);
    double* Pi = Pm + (size_t)i * L;
    double m = -INFINITY;
    for (int j = 0; j < L; ++j) {
      double s = 0.0;
      const double* ktj = kt + (size_t)j * D;
      for (int d = 0; d < D; ++d) s += qti[d] * ktj[d];
      s *= c->scale;                                   /* s_ij */
      Pi[j] = s;
      if (s > m) m = s;
    }
    double Z = 0.0;
    for (int j = 0; j < L; ++j) { Pi[j] = exp(Pi[j] - m); Z += Pi[j]; }
    const double lse = m + log(Z);                     /* LSE_i = ln sum_j exp(s_ij) */
    for (int j = 0; j < L; ++j) Pi[j] /= Z;            /* P_ij = exp(s_ij - LSE_i)   */
    double* o = Oi + (size_t)i * D;
    for (int d = 0; d < D; ++d) o[d] = 0.0;
    for (int j = 0; j < L; ++j) {
      const double p = Pi[j];
      const double* vj = v + (size_t)j * D;
      for (int d = 0; d < D; ++d) o[d] += p * vj[d];   /* O_i = sum_j P_ij V_j */
    }
    if (LSE) LSE[i] = lse;

    if (need_bwd) {
      /* step 3: dP_ij = dO_i . V_j ; D_i = dO_i . O_i ; dS_ij = P_ij (dP_ij - D_i) ;
       *         dq~_i = scale * sum_j dS_ij k~_j  -> through RoPE and RMSNorm -> dQ_i */
      const double* doi = dO + (size_t)i * D;
      double Di = 0.0;
      for (int d = 0; d < D; ++d) Di += doi[d] * o[d];
      double* dSi = dS + (size_t)i * L;
      double* gq = (double*)malloc(sizeof(double) * (size_t)D);
      for (int d = 0; d < D; ++d) gq[d] = 0.0;
      for (int j = 0; j < L; ++j) {
        const double* vj = v + (size_t)j * D;
        double dp = 0.0;
        for (int d = 0; d < D; ++d) dp += doi[d] * vj[d];
        const double ds = Pi[j] * (dp - Di);
        dSi[j] = ds;
        const double* ktj = kt + (size_t)j * D;
        for (int d = 0; d < D; ++d) gq[d] += ds * ktj[d];
      }
      for (int d = 0; d < D; ++d) gq[d] *= c->scale;
      if (dQ || dgq_rows)
        norm_rope_row_bwd(c, q + (size_t)i * D, gamma_q, pos, qidx[i] >= Lvid, rq[i], gq,
                          dQ ? dQ + (size_t)i * D : NULL, dgq_rows ? dgq_rows + (size_t)i * D : NULL);
      free(gq);
    }
  }
  if (O) memcpy(O, Oi, sizeof(double) * (size_t)R * D);
  if (P) memcpy(P, Pm, sizeof(double) * (size_t)R * L);

  /* step 4: per key — dV_j = sum_i P_ij dO_i ; dk~_j = scale * sum_i dS_ij q~_i -> dK_j */
  if (need_bwd && (dK || dV || dgk_rows)) {
#pragma omp parallel for schedule(static)
    for (int j = 0; j < L; ++j) {
      double* gv = (double*)malloc(sizeof(double) * 2 * (size_t)D);
      double* gk = gv + D;
      for (int d = 0; d < D; ++d) { gv[d] = 0.0; gk[d] = 0.0; }
      for (int i = 0; i < R; ++i) {
        const double p = Pm[(size_t)i * L + j], ds = dS[(size_t)i * L + j];
        const double* doi = dO + (size_t)i * D;
        const double* qti = qt + (size_t)i * D;
        for (int d = 0; d < D; ++d) { gv[d] += p * doi[d]; gk[d] += ds * qti[d]; }
      }
      if (dV) memcpy(dV + (size_t)j * D, gv, sizeof(double) * (size_t)D);
      if (dK || dgk_rows) {
        int pos[3];
        token_pos(c, grid, j, pos);
        for (int d = 0; d < D; ++d) gk[d] *= c->scale;
        norm_rope_row_bwd(c, k + (size_t)j * D, gamma_k, pos, j >= Lvid, rk[j], gk,
                          dK ? dK + (size_t)j * D : NULL, dgk_rows ? dgk_rows + (size_t)j * D : NULL);
      }
      free(gv);
    }
  }
  /* R22: dl/dgamma = sum of the per-row terms, rows in index order */
  if (dgq_rows) {
    for (int d = 0; d < D; ++d) dGq[d] = 0.0;
    for (int i = 0; i < R; ++i) for (int d = 0; d < D; ++d) dGq[d] += dgq_rows[(size_t)i * D + d];
  }
  if (dgk_rows) {
    for (int d = 0; d < D; ++d) dGk[d] = 0.0;
    for (int j = 0; j < L; ++j) for (int d = 0; d < D; ++d) dGk[d] += dgk_rows[(size_t)j * D + d];
  }
  free(kt); free(rk); free(qt); free(rq); free(Pm); free(dS); free(Oi); free(dgq_rows); free(dgk_rows);
  return 0;
}

/* The base problem of BASELINE.json north_star: video tokens only, no dgamma. */
int arachne_oracle_head(const oracle_cfg* c, const int grid[3], int L, int R, const int* qidx,
                        const double* q, const double* k, const double* v,
                        const double* gamma_q, const double* gamma_k, const double* dO,
                        double* O, double* LSE, double* P, double* dQ, double* dK, double* dV) {
  return arachne_oracle_head_joint(c, grid, 0, L, R, qidx, q, k, v, gamma_q, gamma_k, dO, O, LSE, P,
                                   dQ, dK, dV, NULL, NULL);
}

/* Debug hook for the RoPE / RMSNorm pins: x~ of one row. */
int arachne_oracle_norm_rope(const oracle_cfg* c, const int pos[3], const double* x,
                             const double* gamma, double* xt) {
  int p[3] = {pos[0] + c->pos_offset[0], pos[1] + c->pos_offset[1], pos[2] + c->pos_offset[2]};
  norm_rope_row(c, x, gamma, p, 0, xt);
  return 0;
}
