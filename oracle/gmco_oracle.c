/* gmco_oracle.c -- fp64 CPU ORACLE for the gL-BFGS hot path of gMCO (arXiv 1904.01567).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It
 * shares no code, header, table or helper with the CUDA path (paper_1904_01567_b200/)
 * and neither side includes or imports the other.
 *
 * Style: plain loops in double precision, one statement per formula of the paper, in
 * the paper's order and notation; no blocking, fusion or reordering.  The only
 * parallelism is an OpenMP "for" over independent plans in orc_evaluate/orc_optimize.
 * Inputs arrive as the SAME fp32 arrays the CUDA path gets and are promoted to double.
 *
 * What pins each function (tests/test_oracle_*.py, all -m "not gpu"):
 *   orc_eval_plan : brute-force dose sums, the 2x2 hand case tests/golden/eq1_eq2_hand_case.txt,
 *                   mean prostate dose == Rx at the uniform start, zero-penalty plan,
 *                   F(c w) = c F, permutation invariance, central finite differences (Eq. 3),
 *                   chain-rule identity g = 2 x o D^T r.
 *   orc_lbfgs     : SPD quadratic vs A^-1 b, monotone F, first step = -g/|g|, planted
 *                   least-squares solution, random starts -> same F.
 *   orc_dvh       : hand-built dose vectors incl. exact ties.
 *   orc_sa_chain  : the hand-worked chains of tests/golden/sa_chain_hand_case.txt (move width 0.1 t_j with its
 *                   0.01 tau floor, clip at 0, downhill / uphill accept / uphill reject with u on either side of
 *                   exp(-dF/T_n), T_n = temp0 cooling^n bracketed from both sides at n = 0..3; state after every
 *                   prefix); incremental dose == D t recomputed; zero-temperature monotonicity.
 *   orc_dose_rate : value at 1 cm, inverse-square law with g = 1, the r floor, role swap = transpose, axis
 *                   relabelling, element independence, the generator's numpy recipe (independent code).
 *   select_plan / pareto_front (oracle/__init__.py, written-out definitions): hand-built tables, a 2-D
 *                   sorting sweep, exhaustive enumeration, invariants (tests/test_oracle_pool.py).
 *   Absolute values printed by the paper: none exist (figures only) -> parity with the
 *   paper's figures is UNPINNED.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* One penalised point group.  Mirrors the INPUT table, not the CUDA headers. */
typedef struct {
  int32_t n_points;      /* rows of D, contiguous, in table order                      */
  double d_lo, d_hi;     /* D_min, D_max of Eq. 2 (Gy); -inf / +inf disables a side    */
  double w_lo, w_hi;     /* class-solution weights w_min, w_max of Eq. 2 / Table 1     */
  int32_t dvh_kind;      /* 0 none | 1 V(level % of Rx) | 2 D(level % of points)       */
  double dvh_level;      /* percent                                                    */
} orc_struct;

typedef struct {
  int32_t m;             /* history length                                             */
  int32_t iters;         /* iteration budget                                           */
  double eps;            /* 0 = run exactly iters (PAPER.md:119 stopping rule, A6)     */
  double c1;             /* Armijo constant, 1e-4                                      */
  int32_t max_trials;    /* 20                                                         */
  double eps_f;          /* relative objective-noise allowance of the approximate test (A5b); 0 = Armijo only */
} orc_lbfgs_opt;

typedef struct {
  int32_t iters_done;
  int32_t status;        /* 0 ran out of iterations | 1 converged (eps or g = 0) | 2 stalled */
  int32_t n_evals;       /* objective/gradient evaluations, start point included       */
  int32_t n_backtracks;  /* rejected trial steps                                       */
  int32_t n_skipped;     /* (s, y) pairs rejected by the curvature guard               */
  int32_t n_approx;      /* steps accepted by the approximate test only (A5b)          */
  int32_t n_bt_iters;    /* iterations in which at least one trial step was rejected   */
  int32_t max_bt_iter;   /* most rejected trial steps inside one iteration             */
} orc_lbfgs_stat;

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* ------------------------------------------------------------------------------------
 * c.1  One evaluation for ONE plan (Eqs. 1-4).
 *   D      [N][A] dose-rate matrix, point-major (Eq. 1: d-dot_ijl, l fastest)
 *   x      [A]    dwell weights, t_l = x_l^2
 *   w      [S][2] hidden weights of this plan (lo, hi) (Eq. 4's w_j, reading A3/A4)
 * Outputs (any may be NULL): dose[N], Fterm[S][2], r[N] = dF/dd_i, G[A] = D^T r,
 *   g[A] = dF/dx.  Returns F.
 */
double orc_eval_plan(const float* D, int64_t N, int64_t A, const orc_struct* st, int32_t S,
                     const float* w, const double* x,
                     double* dose, double* Fterm, double* r, double* G, double* g) {
  double* d = (double*)malloc(sizeof(double) * (size_t)N);
  double* rr = (double*)malloc(sizeof(double) * (size_t)N);
  double* t = (double*)malloc(sizeof(double) * (size_t)A);
  for (int64_t l = 0; l < A; ++l) t[l] = x[l] * x[l];                 /* t_l = x_l^2          */

  for (int64_t i = 0; i < N; ++i) {                                   /* Eq. 1                */
    double acc = 0.0;
    for (int64_t l = 0; l < A; ++l) acc += (double)D[i * A + l] * t[l];
    d[i] = acc;
  }

  double F = 0.0;
  int64_t row = 0;
  for (int32_t j = 0; j < S; ++j) {                                   /* Eq. 4: sum over organs */
    const double Wlo = (double)w[2 * j + 0] * st[j].w_lo;             /* w_j * w_min          */
    const double Whi = (double)w[2 * j + 1] * st[j].w_hi;             /* w_j * w_max          */
    const double inv_n = 1.0 / (double)st[j].n_points;                /* 1 / N_pnt,j          */
    double f_lo = 0.0, f_hi = 0.0;
    for (int32_t i = 0; i < st[j].n_points; ++i, ++row) {
      const double lo = fmin(d[row] - st[j].d_lo, 0.0);               /* < 0 iff d < D_min    */
      const double hi = fmax(d[row] - st[j].d_hi, 0.0);               /* > 0 iff d > D_max    */
      f_lo += Wlo * lo * lo;                                          /* Eq. 2, first branch  */
      f_hi += Whi * hi * hi;                                          /* Eq. 2, third branch  */
      rr[row] = 2.0 * inv_n * (Wlo * lo + Whi * hi);                  /* dF/dd_i              */
    }
    if (Fterm) { Fterm[2 * j + 0] = f_lo * inv_n; Fterm[2 * j + 1] = f_hi * inv_n; }
    F += (f_lo + f_hi) * inv_n;
  }

  if (G || g) {
    for (int64_t l = 0; l < A; ++l) {                                 /* G_l = sum_i D_il r_i */
      double acc = 0.0;
      for (int64_t i = 0; i < N; ++i) acc += (double)D[i * A + l] * rr[i];
      if (G) G[l] = acc;
      if (g) g[l] = 2.0 * x[l] * acc;                                 /* Eq. 3: 4 d-dot x w (d - D) summed */
    }
  }
  if (dose) memcpy(dose, d, sizeof(double) * (size_t)N);
  if (r) memcpy(r, rr, sizeof(double) * (size_t)N);
  free(d); free(rr); free(t);
  return F;
}

/* Batch of K plans, dwell TIMES in (fp32, promoted), x = sqrt(t).
 *   T [K][A] (or [A] if t_broadcast), weights [K][S][2]
 *   dose [N][K] (plan fastest, the layout gmco_evaluate writes), F [K], Fterm [K][S][2],
 *   grad_x [K][A], G [K][A]; any output may be NULL. */
int orc_evaluate(const float* D, int64_t N, int64_t A, const orc_struct* st, int32_t S,
                 const float* T, int32_t t_broadcast, const float* weights, int32_t K,
                 double* dose, double* F, double* Fterm, double* grad_x, double* G) {
  int64_t tot = 0;
  for (int32_t j = 0; j < S; ++j) tot += st[j].n_points;
  if (tot != N) return -1;
#pragma omp parallel for schedule(dynamic, 1)
  for (int32_t k = 0; k < K; ++k) {
    double* x = (double*)malloc(sizeof(double) * (size_t)A);
    double* dk = dose ? (double*)malloc(sizeof(double) * (size_t)N) : NULL;
    const float* Tk = t_broadcast ? T : T + (int64_t)k * A;
    for (int64_t l = 0; l < A; ++l) x[l] = sqrt((double)Tk[l]);
    double Fk = orc_eval_plan(D, N, A, st, S, weights + (int64_t)k * S * 2, x, dk,
                              Fterm ? Fterm + (int64_t)k * S * 2 : NULL, NULL,
                              G ? G + (int64_t)k * A : NULL, grad_x ? grad_x + (int64_t)k * A : NULL);
    if (F) F[k] = Fk;
    if (dose) { for (int64_t i = 0; i < N; ++i) dose[i * K + k] = dk[i]; free(dk); }
    free(x);
  }
  return 0;
}

/* ------------------------------------------------------------------------------------
 * c.2  L-BFGS (Liu & Nocedal 1989, cited PAPER.md:115; the paper omits the description,
 * PAPER.md:117, so every choice is DESIGN.md reading A5), generic over an objective
 * callback so the driver itself can be pinned on problems with known minimisers.
 */
typedef double (*orc_fg_fn)(const double* x, double* g, void* ctx);

static double dot(const double* a, const double* b, int64_t n) {
  double s = 0.0;
  for (int64_t i = 0; i < n; ++i) s += a[i] * b[i];
  return s;
}

int orc_lbfgs(orc_fg_fn fg, void* ctx, int64_t n, double* x, const orc_lbfgs_opt* opt,
              double* F_final, double* F_hist /* [iters+1] or NULL */, orc_lbfgs_stat* stat) {
  const int m = opt->m;
  double* g  = (double*)malloc(sizeof(double) * n);
  double* gn = (double*)malloc(sizeof(double) * n);
  double* xn = (double*)malloc(sizeof(double) * n);
  double* q  = (double*)malloc(sizeof(double) * n);
  double* p  = (double*)malloc(sizeof(double) * n);
  double* Sm = (double*)malloc(sizeof(double) * n * (m > 0 ? m : 1));  /* s_i, oldest first */
  double* Ym = (double*)malloc(sizeof(double) * n * (m > 0 ? m : 1));
  double* rho = (double*)malloc(sizeof(double) * (m > 0 ? m : 1));
  double* a = (double*)malloc(sizeof(double) * (m > 0 ? m : 1));
  int h = 0;                                    /* pairs held, index 0 = oldest, h-1 = newest */
  orc_lbfgs_stat s = {0, 0, 0, 0, 0, 0, 0, 0};

  double F = fg(x, g, ctx); s.n_evals = 1;
  if (F_hist) F_hist[0] = F;

  for (int it = 0; it < opt->iters; ++it) {
    const double gnorm = sqrt(dot(g, g, n));
    if (gnorm == 0.0) { s.status = 1; break; }                        /* A9 */

    /* two-loop recursion: p = -H g */
    memcpy(q, g, sizeof(double) * n);
    for (int i = h - 1; i >= 0; --i) {                                /* newest .. oldest */
      a[i] = rho[i] * dot(Sm + (int64_t)i * n, q, n);
      for (int64_t l = 0; l < n; ++l) q[l] -= a[i] * Ym[(int64_t)i * n + l];
    }
    double gamma;
    if (h > 0) {
      const double* sN = Sm + (int64_t)(h - 1) * n; const double* yN = Ym + (int64_t)(h - 1) * n;
      gamma = dot(sN, yN, n) / dot(yN, yN, n);
    } else {
      gamma = 1.0 / gnorm;
    }
    for (int64_t l = 0; l < n; ++l) q[l] *= gamma;                    /* r = gamma q */
    for (int i = 0; i < h; ++i) {                                     /* oldest .. newest */
      const double b = rho[i] * dot(Ym + (int64_t)i * n, q, n);
      for (int64_t l = 0; l < n; ++l) q[l] += Sm[(int64_t)i * n + l] * (a[i] - b);
    }
    for (int64_t l = 0; l < n; ++l) p[l] = -q[l];
    double gp = dot(g, p, n);
    if (gp >= 0.0) {                                                  /* not a descent direction */
      h = 0;
      for (int64_t l = 0; l < n; ++l) p[l] = -g[l] / gnorm;
      gp = dot(g, p, n);
    }

    /* backtracking line search: alpha = 1, 1/2, 1/4, ...; phi(alpha) = F(x + alpha p).
     * A trial step is accepted by the Armijo test, or -- reading A5b, the "approximate Wolfe"
     * test of Hager & Zhang (2005), needed once the decrease per step falls below what the
     * objective can resolve -- when F has not risen by more than eps_f |F| and the slope at the
     * trial point satisfies phi'(alpha) <= (2 c1 - 1) phi'(0) (identical to Armijo for a quadratic phi). */
    double alpha = 1.0, Fn = 0.0;
    int accepted = 0, rejected_here = 0;             /* rejected_here: a counter for the statistics only */
    for (int trial = 0; trial < opt->max_trials; ++trial) {
      for (int64_t l = 0; l < n; ++l) xn[l] = x[l] + alpha * p[l];
      Fn = fg(xn, gn, ctx); s.n_evals++;
      if (Fn <= F + opt->c1 * alpha * gp) { accepted = 1; break; }
      if (opt->eps_f > 0.0 && Fn <= F + opt->eps_f * fabs(F) &&
          dot(gn, p, n) <= (2.0 * opt->c1 - 1.0) * gp) { accepted = 1; s.n_approx++; break; }
      s.n_backtracks++; rejected_here++;
      alpha *= 0.5;
    }
    if (rejected_here > 0) s.n_bt_iters++;
    if (rejected_here > s.max_bt_iter) s.max_bt_iter = rejected_here;
    if (!accepted) { s.status = 2; break; }                           /* stalled: x unchanged */

    /* history update: s = x+ - x, y = g+ - g, curvature guard */
    if (m > 0) {
      double* sv = q;  /* reuse q as scratch for s, p as scratch for y */
      double* yv = p;
      for (int64_t l = 0; l < n; ++l) { sv[l] = xn[l] - x[l]; yv[l] = gn[l] - g[l]; }
      const double sy = dot(sv, yv, n);
      if (sy > 1e-10 * sqrt(dot(sv, sv, n)) * sqrt(dot(yv, yv, n))) {
        if (h == m) {                                                 /* drop the oldest */
          memmove(Sm, Sm + n, sizeof(double) * n * (m - 1));
          memmove(Ym, Ym + n, sizeof(double) * n * (m - 1));
          memmove(rho, rho + 1, sizeof(double) * (m - 1));
          h = m - 1;
        }
        memcpy(Sm + (int64_t)h * n, sv, sizeof(double) * n);
        memcpy(Ym + (int64_t)h * n, yv, sizeof(double) * n);
        rho[h] = 1.0 / sy;
        h++;
      } else {
        s.n_skipped++;
      }
    }

    const double Fold = F;
    memcpy(x, xn, sizeof(double) * n);
    memcpy(g, gn, sizeof(double) * n);
    F = Fn;
    s.iters_done = it + 1;
    if (F_hist) F_hist[it + 1] = F;
    if (opt->eps > 0.0 && fabs(Fold - F) <= opt->eps * fmax(Fold, 1e-30)) { s.status = 1; break; }
  }
  if (F_hist) for (int it = s.iters_done + 1; it <= opt->iters; ++it) F_hist[it] = F;
  if (F_final) *F_final = F;
  if (stat) *stat = s;
  free(g); free(gn); free(xn); free(q); free(p); free(Sm); free(Ym); free(rho); free(a);
  return 0;
}

/* objective callback of the gMCO problem for one plan */
typedef struct {
  const float* D; int64_t N, A; const orc_struct* st; int32_t S; const float* w;
} orc_plan_ctx;

static double plan_fg(const double* x, double* g, void* vctx) {
  const orc_plan_ctx* c = (const orc_plan_ctx*)vctx;
  return orc_eval_plan(c->D, c->N, c->A, c->st, c->S, c->w, x, NULL, NULL, NULL, NULL, g);
}

/* c.3  DVH indices of one plan from its dose vector (reading A17).
 *   kind 1: V_level = share of the structure's points with d >= (level/100) Rx, in % of points
 *   kind 2: D_level = dose of the ceil(level/100 * n)-th hottest point (nearest rank), in % of Rx */
static int cmp_desc(const void* a, const void* b) {
  const double x = *(const double*)a, y = *(const double*)b;
  return (x < y) - (x > y);
}

void orc_dvh(const double* dose, const orc_struct* st, int32_t S, double rx, double* out /* [S] */) {
  int64_t row = 0;
  for (int32_t j = 0; j < S; ++j) {
    const int32_t n = st[j].n_points;
    out[j] = 0.0;
    if (st[j].dvh_kind == 1) {
      const double thr = st[j].dvh_level / 100.0 * rx;
      int64_t cnt = 0;
      for (int32_t i = 0; i < n; ++i) cnt += (dose[row + i] >= thr);
      out[j] = 100.0 * (double)cnt / (double)n;
    } else if (st[j].dvh_kind == 2) {
      double* v = (double*)malloc(sizeof(double) * (size_t)n);
      memcpy(v, dose + row, sizeof(double) * (size_t)n);
      qsort(v, (size_t)n, sizeof(double), cmp_desc);
      int64_t rank = (int64_t)ceil((double)n * st[j].dvh_level / 100.0);
      if (rank < 1) rank = 1;
      if (rank > n) rank = n;
      out[j] = 100.0 * v[rank - 1] / rx;
      free(v);
    }
    row += n;
  }
}

/* K plans: x0 = sqrt(T0), run orc_lbfgs on each, then dose + DVH at the final point.
 *   T0 [K][A] or [A] (t0_broadcast); weights [K][S][2]
 *   T_out [K][A] = x^2, F [K], dvh [K][S], Fterm [K][S][2], stats [K], F_hist [K][iters+1]; NULL ok */
int orc_optimize(const float* D, int64_t N, int64_t A, const orc_struct* st, int32_t S, double rx,
                 const float* T0, int32_t t0_broadcast, const float* weights, int32_t K,
                 const orc_lbfgs_opt* opt,
                 double* T_out, double* F, double* dvh, double* Fterm, orc_lbfgs_stat* stats,
                 double* F_hist) {
  int64_t tot = 0;
  for (int32_t j = 0; j < S; ++j) tot += st[j].n_points;
  if (tot != N) return -1;
#pragma omp parallel for schedule(dynamic, 1)
  for (int32_t k = 0; k < K; ++k) {
    double* x = (double*)malloc(sizeof(double) * (size_t)A);
    double* d = (double*)malloc(sizeof(double) * (size_t)N);
    const float* Tk = t0_broadcast ? T0 : T0 + (int64_t)k * A;
    for (int64_t l = 0; l < A; ++l) x[l] = sqrt((double)Tk[l]);
    orc_plan_ctx ctx = {D, N, A, st, S, weights + (int64_t)k * S * 2};
    double Fk; orc_lbfgs_stat sk;
    orc_lbfgs(plan_fg, &ctx, A, x, opt, &Fk, F_hist ? F_hist + (int64_t)k * (opt->iters + 1) : NULL, &sk);
    Fk = orc_eval_plan(D, N, A, st, S, ctx.w, x, d, Fterm ? Fterm + (int64_t)k * S * 2 : NULL, NULL, NULL, NULL);
    if (F) F[k] = Fk;
    if (T_out) for (int64_t l = 0; l < A; ++l) T_out[(int64_t)k * A + l] = x[l] * x[l];
    if (dvh) orc_dvh(d, st, S, rx, dvh + (int64_t)k * S);
    if (stats) stats[k] = sk;
    free(x); free(d);
  }
  return 0;
}

/* ------------------------------------------------------------------------------------
 * c.5  Simulated annealing chain (BASELINE.json configs[4]; PAPER.md:96-113 gives the loop
 * of steps (ii)-(v) only, everything else is DESIGN.md reading A20/c.5).  The random
 * numbers are INPUTS: jdx[n] in [0, A), z[n] ~ N(0,1), u[n] ~ U[0,1).
 *   sigma = max(0.1 t_j, 0.01 tau);  t' = max(t_j + sigma z, 0);  d' = d + (t' - t_j) D[:, j]
 *   accept if dF <= 0, else if u < exp(-dF / T_n), T_n = temp0 * exp(n ln cooling)        */
static double penalty_sum(const double* d, const orc_struct* st, int32_t S, const float* w) {
  double F = 0.0; int64_t row = 0;
  for (int32_t j = 0; j < S; ++j) {
    const double Wlo = (double)w[2 * j] * st[j].w_lo, Whi = (double)w[2 * j + 1] * st[j].w_hi;
    double acc = 0.0;
    for (int32_t i = 0; i < st[j].n_points; ++i, ++row) {
      const double lo = fmin(d[row] - st[j].d_lo, 0.0), hi = fmax(d[row] - st[j].d_hi, 0.0);
      acc += Wlo * lo * lo + Whi * hi * hi;
    }
    F += acc / (double)st[j].n_points;
  }
  return F;
}

int orc_sa_chain(const float* D, int64_t N, int64_t A, const orc_struct* st, int32_t S,
                 const float* w, const float* T0, double tau, int64_t steps,
                 const int32_t* jdx, const double* z, const double* u, double temp0, double cooling,
                 double* t_out /* [A] */, double* d_out /* [N] or NULL */, double* F_out,
                 int64_t* n_accepted) {
  double* t = (double*)malloc(sizeof(double) * (size_t)A);
  double* d = (double*)malloc(sizeof(double) * (size_t)N);
  double* dn = (double*)malloc(sizeof(double) * (size_t)N);
  for (int64_t l = 0; l < A; ++l) t[l] = (double)T0[l];
  for (int64_t i = 0; i < N; ++i) {
    double acc = 0.0;
    for (int64_t l = 0; l < A; ++l) acc += (double)D[i * A + l] * t[l];
    d[i] = acc;
  }
  double F = penalty_sum(d, st, S, w);
  int64_t acc_cnt = 0;
  const double lc = log(cooling);
  for (int64_t n = 0; n < steps; ++n) {
    const int64_t j = jdx[n];
    const double sigma = fmax(0.1 * t[j], 0.01 * tau);
    const double tn = fmax(t[j] + sigma * z[n], 0.0);
    const double dt = tn - t[j];
    for (int64_t i = 0; i < N; ++i) dn[i] = d[i] + dt * (double)D[i * A + j];
    const double Fn = penalty_sum(dn, st, S, w);
    const double dF = Fn - F;
    int accept = 0;
    if (dF <= 0.0) accept = 1;
    else {
      const double Tn = temp0 * exp((double)n * lc);
      accept = (Tn > 0.0) && (u[n] < exp(-dF / Tn));
    }
    if (accept) { t[j] = tn; F = Fn; double* tmp = d; d = dn; dn = tmp; acc_cnt++; }
  }
  memcpy(t_out, t, sizeof(double) * (size_t)A);
  if (d_out) memcpy(d_out, d, sizeof(double) * (size_t)N);
  if (F_out) *F_out = F;
  if (n_accepted) *n_accepted = acc_cnt;
  free(t); free(d); free(dn);
  return 0;
}

/* ------------------------------------------------------------------------------------
 * Step (i): dose-rate matrix (PAPER.md:97 names the step; the model is BASELINE.json configs[0]'s TG-43
 * point-source approximation, A14-A15):  D_il = sk_lambda g(r) / r^2,  r = |p_i - q_l| in cm floored at
 * r_floor,  g(r) = sum_c coef[c] r^c.  Plain loops, fp64, one rounding to fp32.
 * Pins (tests/test_oracle_doserate.py): D = sk_lambda g(1) at r = 1 cm exactly; inverse-square law with g = 1;
 * the floor; translation / rotation invariance; the numpy recipe of gmco_cases (independent code).            */
int orc_dose_rate(const float* pts /* [N][3] mm */, int64_t N, const float* dwell /* [A][3] mm */, int64_t A,
                  const double* coef, int32_t n_coef, double sk_lambda, double r_floor_cm, float* D /* [N][A] */) {
  if (n_coef < 1 || r_floor_cm <= 0.0) return -1;
  for (int64_t i = 0; i < N; ++i)
    for (int64_t l = 0; l < A; ++l) {
      double r2 = 0.0;
      for (int a = 0; a < 3; ++a) {
        const double d = ((double)pts[3 * i + a] - (double)dwell[3 * l + a]) / 10.0;
        r2 += d * d;
      }
      double r = sqrt(r2);
      if (r < r_floor_cm) r = r_floor_cm;
      double g = 0.0, rp = 1.0;
      for (int32_t c = 0; c < n_coef; ++c) { g += coef[c] * rp; rp *= r; }      /* the polynomial as written */
      D[i * A + l] = (float)(sk_lambda * g / (r * r));
    }
  return 0;
}
