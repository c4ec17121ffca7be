/*
 * ckoracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * A plain, slow, double-precision restatement of what the hot path computes, written from the paper
 * (Niemeyer & Sung, arXiv 1309.2710; cited below as P:<line of /root/reference/PAPER.md>) step by step,
 * in the paper's order and notation.  It shares no code, header, table or constant generator with the
 * CUDA library under paper_1309_2710_b200/csrc/ (constants that appear in both are typed twice).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it.
 *
 * Build:  gcc -O2 -ffp-contract=off -fopenmp -fPIC -shared -o libckoracle.so ckoracle.c -lm
 * (no fast-math, no FMA contraction: what is written is what is evaluated).
 *
 * Readings of the paper where it is silent / ambiguous / garbled are marked Rn; the list with the
 * justification of each is DESIGN.md section 4 (same numbering as SURVEY.md section 9).
 *
 * Pins (tests/test_oracle_*.py, all run without a GPU):
 *   Table 1                  : 17+8 rooted-tree order conditions in exact rationals, row sums, R(z) incl. z^6/800
 *   ora_rkck_step            : y'=lambda y closed form R(z), R*(z); measured order 5 / 4 on y'=-y^2
 *   ora_rkc_coeffs/_step     : stage closed form a_j + b_j T_j(w0 + w1 z) for s = 2..200; Chebyshev bound
 *                              |P_s(z)| <= 1 on [-beta(s), 0]; measured order 2; c_1 = c_2/T_2'(w0)
 *   ora_spectral_radius      : linear operators with known spectrum; on the 9/13/53-species chemistry: same value and
 *                              same evaluation count as a textbook power iteration on an explicit central-difference
 *                              Jacobian, and the distribution of (returned value)/rho(J)
 *   ora_rhs                  : A->B, A->B->C (Bateman), A+B->C+D, A+M->B+M closed forms; Arrhenius in mpmath;
 *                              Sum Y and element mass invariants
 *   ora_rkck/rkc drivers     : tolerance proportionality, brute-force fixed-step reference, RKCK-vs-RKC
 *                              cross-check, linear invariants; and from the step traces (ora_rkck_trace /
 *                              ora_rkc_trace, tests/test_oracle_controllers.py): Eq. 16-17 with both exponents, S and
 *                              both limits; Eq. 30-32 against the closed form on y' = lambda y; Eq. 33-35
 *                              incl. the orientation of Eq. 34's memory term and the [0.1, 10] clamp; Eq. 36-38 by
 *                              hand; Eq. 39 truncated with dt sigma inside the stability interval; the 25-step /
 *                              after-rejection refresh of sigma.
 *   ora_fit_reverse / ora_equilibrium_constant / ora_reverse_parameters (Appendix A, tests/test_oracle_convert.py):
 *                              exact round trip of three points of a known Arrhenius law, numpy's 3 x 3 linear solve,
 *                              closed-form reverse parameters on species with a1, a6, a7 only (dnu = 0 and 1), the
 *                              equilibrium ratio reached by the integrated forward / fitted-reverse pair.
 *   PARITY UNPINNED (builder's reading, nothing in the paper or the mathematics fixes them; the traces pin that the
 *   code does what the reading says, not that the reading is the only possible one):
 *   R4 (RKCK first trial step), R5 (end-of-interval clipping), R6/R7 (failure codes), R10 (b_1 = b_2 for
 *   nonlinear f), R13 (controller memory dropped after a rejection), R14/R15 (initial-step weights and cap),
 *   R16 (sigma refreshed after a rejection only when stale), R17/R18 (power-method details and its 1.2 safety factor),
 *   R32 (the equilibrium constant in the Chemkin form), R33 (the three fitting temperatures).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* R20: physical constants (the paper gives none) */
#define ORA_RU 8.314462618e7   /* erg / (mol K)  */
#define ORA_RC 1.98720425864   /* cal / (mol K)  */

#define ORA_OK 0
#define ORA_EINVAL (-1)
#define ORA_ENOMEM (-2)

/* per-system status codes */
#define ST_OK 0
#define ST_MAXSTEPS 1
#define ST_UNDERFLOW 2
#define ST_NONFINITE 3
#define ST_SIGMA 4

typedef void (*ora_rhs_fn)(double t, const double *y, double *dydt, void *ctx);

/* ------------------------------------------------------------------------------------------------
 * Table 1, R1: rows 4-6 are scrambled in the extraction; these are the Cash-Karp values
 * every legible fragment of the table agrees with.  Pinned exactly by the order-condition test.
 * ---------------------------------------------------------------------------------------------- */
static const double CK_A[7] = {0, 0.0, 1.0 / 5.0, 3.0 / 10.0, 3.0 / 5.0, 1.0, 7.0 / 8.0};
static const double CK_B[7][6] = {
    {0},
    {0},
    {0, 1.0 / 5.0},
    {0, 3.0 / 40.0, 9.0 / 40.0},
    {0, 3.0 / 10.0, -9.0 / 10.0, 6.0 / 5.0},
    {0, -11.0 / 54.0, 5.0 / 2.0, -70.0 / 27.0, 35.0 / 27.0},
    {0, 1631.0 / 55296.0, 175.0 / 512.0, 575.0 / 13824.0, 44275.0 / 110592.0, 253.0 / 4096.0}};
static const double CK_C[7] = {0, 37.0 / 378.0, 0.0, 250.0 / 621.0, 125.0 / 594.0, 0.0, 512.0 / 1771.0};
static const double CK_CS[7] = {0, 2825.0 / 27648.0, 0.0, 18575.0 / 48384.0, 13525.0 / 55296.0,
                                277.0 / 14336.0, 1.0 / 4.0};

/* test access to the table as rationals' double values: out[0..5]=a, [6..35]=b (6x5 row-major, b_ij j=1..5),
 * [36..41]=c, [42..47]=c* */
void ora_rkck_tableau(double *out) {
  for (int i = 1; i <= 6; i++) out[i - 1] = CK_A[i];
  for (int i = 1; i <= 6; i++)
    for (int j = 1; j <= 5; j++) out[6 + (i - 1) * 5 + (j - 1)] = CK_B[i][j];
  for (int i = 1; i <= 6; i++) out[36 + i - 1] = CK_C[i];
  for (int i = 1; i <= 6; i++) out[42 + i - 1] = CK_CS[i];
}

/* ------------------------------------------------------------------------------------------------
 * One RKCK step of size h from (t, y): Eq. 7-15.  k1 = h f(t,y) is supplied by the caller
 * (Eq. 7).  ynew = 5th-order solution (Eq. 13), delta = y_{n+1} - y*_{n+1} (Eq. 15).
 * work: 6*n doubles.
 * ---------------------------------------------------------------------------------------------- */
static void rkck_attempt(ora_rhs_fn f, void *ctx, int n, double t, const double *y, const double *k1,
                         double h, double *ynew, double *delta, double *work) {
  double *k[7];
  k[1] = (double *)k1;
  for (int i = 2; i <= 6; i++) k[i] = work + (size_t)(i - 2) * n;
  double *ytmp = work + (size_t)5 * n;
  for (int i = 2; i <= 6; i++) { /* Eq. 8-12 */
    for (int c = 0; c < n; c++) {
      double s = y[c];
      for (int j = 1; j < i; j++) s += CK_B[i][j] * k[j][c];
      ytmp[c] = s;
    }
    f(t + CK_A[i] * h, ytmp, k[i], ctx);
    for (int c = 0; c < n; c++) k[i][c] *= h;
  }
  for (int c = 0; c < n; c++) {
    double s = y[c], d = 0.0;
    for (int i = 1; i <= 6; i++) {
      s += CK_C[i] * k[i][c];               /* Eq. 13 */
      d += (CK_C[i] - CK_CS[i]) * k[i][c];  /* Eq. 15 */
    }
    ynew[c] = s;
    delta[c] = d;
  }
}

/* fixed-step entry for the order / closed-form tests (controller off) */
void ora_rkck_step(ora_rhs_fn f, void *ctx, int n, double t, const double *y, double h, double *ynew,
                   double *delta) {
  double *work = (double *)malloc(sizeof(double) * (size_t)n * 7);
  double *k1 = work + (size_t)6 * n;
  f(t, y, k1, ctx);
  for (int c = 0; c < n; c++) k1[c] *= h; /* Eq. 7 */
  rkck_attempt(f, ctx, n, t, y, k1, h, ynew, delta, work);
  free(work);
}

static int all_finite(const double *v, int n) {
  for (int i = 0; i < n; i++)
    if (!isfinite(v[i])) return 0;
  return 1;
}

/* ------------------------------------------------------------------------------------------------
 * RKCK driver.  Integrates y from t0 to t1 in place.
 * stats[0]=RHS evaluations, [1]=accepted steps, [2]=rejected steps, [3]=0.  Returns a status code.
 * ---------------------------------------------------------------------------------------------- */
/* Step trace (test-only; the pins of the step-size controllers read it): one row of ORA_TRACE_COLS doubles per
 * step ATTEMPT, in order:  [0] t at the start of the attempt, [1] the step size attempted (after the R5 clip / the
 * R12 cap), [2] the error measure of the attempt (RKCK: errmax of Eq. 17; RKC: ||err|| of Eq. 31), [3] 1 accepted /
 * 0 rejected, [4] RKC: stages s of the attempt (RKCK: 6), [5] RKC: 1 if the spectral radius was re-estimated for
 * this attempt (the initial estimate counts for attempt 0), [6] RKC: sigma in use, [7] RKC, attempt 0 only: the
 * ||est|| of Eq. 37 that produced the first step (else 0).  Recording changes nothing in the arithmetic. */
#define ORA_TRACE_COLS 8
typedef struct { double *rows; int64_t cap, n; } ora_trace;
static void trace_row(ora_trace *tr, double t, double h, double err, int acc, int s, int refreshed, double sigma,
                      double est0) {
  if (!tr) return;
  if (tr->n < tr->cap) {
    double *r = tr->rows + ORA_TRACE_COLS * (size_t)tr->n;
    r[0] = t; r[1] = h; r[2] = err; r[3] = acc; r[4] = s; r[5] = refreshed; r[6] = sigma; r[7] = est0;
  }
  tr->n++;
}

static int rkck_driver(ora_rhs_fn f, void *ctx, int n, double *y, double t0, double t1, double rtol,
                       double atol, int32_t *stats, ora_trace *tr) {
  const double S = 0.9;
  const double u = 2.220446049250313e-16;     /* 2^-52 */
  double *buf = (double *)malloc(sizeof(double) * (size_t)n * 9);
  double *k1 = buf, *ynew = buf + n, *delta = buf + 2 * (size_t)n, *work = buf + 3 * (size_t)n;
  int32_t nfe = 0, nacc = 0, nrej = 0;
  int status = ST_OK;
  double t = t0;
  double h = t1 - t0;                         /* R4: first trial step = the whole global step */
  int have_k1 = 0;
  long attempts = 0;
  int saw_nonfinite = 0;
  while (1) {
    int last = 0;
    if (1.1 * h >= t1 - t) {                  /* R5: clip (with 10 % stretch) to hit t1 exactly */
      double hn = t1 - t;
      if (have_k1) { double r = hn / h; for (int c = 0; c < n; c++) k1[c] *= r; }
      h = hn;
      last = 1;
    }
    if (!have_k1) {
      f(t, y, k1, ctx);                       /* Eq. 7 */
      nfe++;
      for (int c = 0; c < n; c++) k1[c] *= h;
      have_k1 = 1;
    }
    if (++attempts > 1000000) { status = ST_MAXSTEPS; break; }           /* R7 */
    rkck_attempt(f, ctx, n, t, y, k1, h, ynew, delta, work);
    nfe += 5;
    /* Eq. 16 (R2: eps -> rtol, eps*delta -> atol) and Eq. 17 (R3: errmax = max |Delta_i| / Delta0_i) */
    double errmax = 0.0;
    int finite = all_finite(ynew, n);
    for (int c = 0; c < n; c++) {
      double d0 = rtol * (fabs(y[c]) + fabs(k1[c])) + atol;
      double e = fabs(delta[c]) / d0;
      if (!(e <= errmax)) errmax = e;          /* NaN propagates into errmax */
    }
    trace_row(tr, t, h, errmax, finite && errmax <= 1.0, 6, 0, 0.0, 0.0);
    if (finite && errmax <= 1.0) {             /* P:139 accept */
      nacc++;
      for (int c = 0; c < n; c++) y[c] = ynew[c];
      have_k1 = 0;
      if (last) { t = t1; break; }
      t += h;
      double fac = (errmax > 0.0) ? S * pow(errmax, -0.2) : 5.0;
      if (fac > 5.0) fac = 5.0;                /* P:144 increases limited to five */
      h *= fac;
    } else {                                   /* reject */
      nrej++;
      double fac;
      if (finite && isfinite(errmax)) {
        fac = S * pow(errmax, -0.25);
        if (fac < 0.1) fac = 0.1;              /* P:144 decreases limited to ten */
      } else {
        fac = 0.1;                             /* R7: non-finite -> plain rejection */
        saw_nonfinite = 1;
      }
      double hn = h * fac;
      for (int c = 0; c < n; c++) k1[c] *= fac; /* R25: k1 = hn f(t,y), rescaled not re-evaluated */
      h = hn;
      double tmax = fabs(t) > fabs(t1) ? fabs(t) : fabs(t1);
      if (!(h > 10.0 * u * tmax)) {            /* R6 */
        status = saw_nonfinite ? ST_NONFINITE : ST_UNDERFLOW;
        break;
      }
    }
  }
  if (stats) { stats[0] = nfe; stats[1] = nacc; stats[2] = nrej; stats[3] = 0; }
  free(buf);
  return status;
}

int ora_rkck_generic(ora_rhs_fn f, void *ctx, int n, double *y, double t0, double t1, double rtol,
                     double atol, int32_t *stats) {
  return rkck_driver(f, ctx, n, y, t0, t1, rtol, atol, stats, NULL);
}

/* test entry: the same driver, recording up to cap attempts into rows[cap][ORA_TRACE_COLS]; *n_rows = attempts made */
int ora_rkck_trace(ora_rhs_fn f, void *ctx, int n, double *y, double t0, double t1, double rtol, double atol,
                   int32_t *stats, double *rows, int64_t cap, int64_t *n_rows) {
  ora_trace tr = {rows, cap, 0};
  const int st = rkck_driver(f, ctx, n, y, t0, t1, rtol, atol, stats, &tr);
  if (n_rows) *n_rows = tr.n;
  return st;
}

/* ------------------------------------------------------------------------------------------------
 * RKC coefficients for s >= 2 stages: Eq. 22-29.  Arrays are indexed 0..s.
 *   R8 : w0 = 1 + eps/s^2 with eps = kappa = 2/13.
 *   R9 : a_j = 1 - b_j T_j(w0)  (used in Eq. 23, never defined in the paper).
 *   R10: b_0 = b_1 = b_2 (Eq. 24 prints b_1 = 1/w0, which contradicts Eq. 27's c_1 = c_2/T_2'(w0)).
 *   R11: c_1 = mu~_1, c_j = w1 T_j''/T_j' (2 <= j <= s-1), c_s = 1.
 * Chebyshev values by the recurrences obtained from Eq. 26 and its derivatives.
 * ---------------------------------------------------------------------------------------------- */
int ora_rkc_coeffs(int s, double *w0_out, double *w1_out, double *mu, double *nu, double *mut,
                   double *gamt, double *c, double *a, double *b) {
  if (s < 2) return ORA_EINVAL;
  double *T = (double *)malloc(sizeof(double) * (size_t)(s + 1) * 3);
  double *dT = T + (s + 1), *d2T = T + 2 * (s + 1);
  const double w0 = 1.0 + (2.0 / 13.0) / ((double)s * (double)s);
  T[0] = 1.0; T[1] = w0; dT[0] = 0.0; dT[1] = 1.0; d2T[0] = 0.0; d2T[1] = 0.0;
  for (int j = 2; j <= s; j++) {
    T[j] = 2.0 * w0 * T[j - 1] - T[j - 2];                          /* Eq. 26 */
    dT[j] = 2.0 * T[j - 1] + 2.0 * w0 * dT[j - 1] - dT[j - 2];
    d2T[j] = 4.0 * dT[j - 1] + 2.0 * w0 * d2T[j - 1] - d2T[j - 2];
  }
  const double w1 = dT[s] / d2T[s];                                  /* Eq. 25 */
  for (int j = 2; j <= s; j++) b[j] = d2T[j] / (dT[j] * dT[j]);      /* Eq. 24 */
  b[0] = b[2]; b[1] = b[2];                                          /* R10 */
  for (int j = 0; j <= s; j++) a[j] = 1.0 - b[j] * T[j];             /* R9 */
  mu[0] = nu[0] = mut[0] = gamt[0] = 0.0; c[0] = 0.0;
  mu[1] = nu[1] = gamt[1] = 0.0;
  mut[1] = b[1] * w1;                                                /* Eq. 22 */
  c[1] = mut[1];
  for (int j = 2; j <= s; j++) {                                     /* Eq. 23 */
    mu[j] = 2.0 * b[j] * w0 / b[j - 1];
    nu[j] = -b[j] / b[j - 2];
    mut[j] = 2.0 * b[j] * w1 / b[j - 1];
    gamt[j] = -a[j - 1] * mut[j];
    c[j] = (j < s) ? w1 * d2T[j] / dT[j] : 1.0;                      /* Eq. 28-29 */
  }
  *w0_out = w0; *w1_out = w1;
  free(T);
  return ORA_OK;
}

/* ------------------------------------------------------------------------------------------------
 * One RKC step with s stages: Eq. 18-21.  f0 = f(t, y).  If stages != NULL, stage vectors
 * w_1..w_s are stored there ([s][n]) for the closed-form test.  Evaluates f at w_1..w_{s-1}: s-1 calls.
 * ---------------------------------------------------------------------------------------------- */
static void rkc_step(ora_rhs_fn f, void *ctx, int n, double t, const double *y, const double *f0,
                     double h, int s, double *ynew, double *stages, double *work /* 3n */) {
  double *wjm1 = work, *wjm2 = work + n, *fj = work + 2 * (size_t)n;
  double *cf = (double *)malloc(sizeof(double) * 7 * (size_t)(s + 1));
  double *mu = cf, *nu = cf + (s + 1), *mut = cf + 2 * (s + 1), *gamt = cf + 3 * (s + 1),
         *c = cf + 4 * (s + 1), *a = cf + 5 * (s + 1), *b = cf + 6 * (s + 1);
  double w0, w1;
  ora_rkc_coeffs(s, &w0, &w1, mu, nu, mut, gamt, c, a, b);
  for (int i = 0; i < n; i++) {            /* Eq. 18-19 */
    wjm2[i] = y[i];
    wjm1[i] = y[i] + mut[1] * h * f0[i];
  }
  if (stages) memcpy(stages, wjm1, sizeof(double) * n);
  for (int j = 2; j <= s; j++) {           /* Eq. 20 */
    f(t + c[j - 1] * h, wjm1, fj, ctx);
    for (int i = 0; i < n; i++) {
      double wj = (1.0 - mu[j] - nu[j]) * y[i] + mu[j] * wjm1[i] + nu[j] * wjm2[i] +
                  mut[j] * h * fj[i] + gamt[j] * h * f0[i];
      wjm2[i] = wjm1[i];
      wjm1[i] = wj;
    }
    if (stages) memcpy(stages + (size_t)(j - 1) * n, wjm1, sizeof(double) * n);
  }
  for (int i = 0; i < n; i++) ynew[i] = wjm1[i]; /* Eq. 21 */
  free(cf);
}

void ora_rkc_step(ora_rhs_fn f, void *ctx, int n, double t, const double *y, double h, int s,
                  double *ynew, double *stages) {
  double *work = (double *)malloc(sizeof(double) * (size_t)4 * n);
  double *f0 = work + 3 * (size_t)n;
  f(t, y, f0, ctx);
  rkc_step(f, ctx, n, t, y, f0, h, s, ynew, stages, work);
  free(work);
}

static double norm2(const double *v, int n) {
  double s = 0.0;
  for (int i = 0; i < n; i++) s += v[i] * v[i];
  return sqrt(s);
}

/* ------------------------------------------------------------------------------------------------
 * Spectral radius by a nonlinear power method (P:233 names it, gives no detail): R17/R18, DESIGN.md 4.5.
 * y, fy = f(t,y); v = previous eigenvector estimate (have_v) or scratch; on return v holds the new one.
 * Returns 1.2 * sigma; *nfe += RHS calls; *flag = ST_SIGMA if not converged in 50 iterations.
 * work: 2n doubles.
 * ---------------------------------------------------------------------------------------------- */
static double spectral_radius(ora_rhs_fn f, void *ctx, int n, double t, const double *y, const double *fy,
                              double *v, int have_v, int32_t *nfe, int *flag, double *work) {
  const double u = 2.220446049250313e-16;
  const double sqrtu = 1.4901161193847656e-08; /* 2^-26 */
  double *z = work, *g = work + n;
  if (!have_v)
    for (int i = 0; i < n; i++) v[i] = fy[i];
  const double ynrm = norm2(y, n), vnrm = norm2(v, n);
  double d;
  if (ynrm != 0.0 && vnrm != 0.0) {
    d = ynrm * sqrtu;
    for (int i = 0; i < n; i++) z[i] = y[i] + v[i] * (d / vnrm);
  } else if (ynrm != 0.0) {
    d = ynrm * sqrtu;
    for (int i = 0; i < n; i++) z[i] = y[i] * (1.0 + sqrtu);
  } else if (vnrm != 0.0) {
    d = u;
    for (int i = 0; i < n; i++) z[i] = v[i] * (d / vnrm);
  } else {
    d = u;
    for (int i = 0; i < n; i++) z[i] = d;
  }
  double sigma = 0.0;
  int converged = 0;
  for (int it = 1; it <= 50; it++) {
    f(t, z, g, ctx);
    (*nfe)++;
    double dd = 0.0;
    for (int i = 0; i < n; i++) dd += (g[i] - fy[i]) * (g[i] - fy[i]);
    dd = sqrt(dd);
    const double sigma_prev = sigma;
    sigma = dd / d;
    const double floor_ = sigma > 1e-300 ? sigma : 1e-300;
    if (it >= 2 && fabs(sigma - sigma_prev) <= 0.01 * floor_) { converged = 1; break; }
    if (dd != 0.0) {
      for (int i = 0; i < n; i++) z[i] = y[i] + (g[i] - fy[i]) * (d / dd);
    } else {
      const int i = it % n;
      z[i] = y[i] - (z[i] - y[i]);
    }
  }
  for (int i = 0; i < n; i++) v[i] = z[i] - y[i];
  if (!converged) *flag = ST_SIGMA;
  return 1.2 * sigma;
}

/* test entry */
double ora_spectral_radius(ora_rhs_fn f, void *ctx, int n, double t, const double *y, double *v,
                           int have_v, int32_t *nfe, int32_t *flag) {
  double *work = (double *)malloc(sizeof(double) * (size_t)n * 3);
  double *fy = work + 2 * (size_t)n;
  int32_t calls = 0;
  int fl = 0;
  f(t, y, fy, ctx);
  double s = spectral_radius(f, ctx, n, t, y, fy, v, have_v, &calls, &fl, work);
  if (nfe) *nfe = calls;
  if (flag) *flag = fl;
  free(work);
  return s;
}

/* ------------------------------------------------------------------------------------------------
 * RKC driver: Eq. 30-39 and P:233.  Integrates y from t0 to t1 in place.
 * stats[0]=RHS evaluations, [1]=accepted, [2]=rejected, [3]=largest stage count used.
 * ---------------------------------------------------------------------------------------------- */
static int rkc_driver(ora_rhs_fn f, void *ctx, int n, double *y, double t0, double t1, double rtol,
                      double atol, int32_t *stats, ora_trace *tr) {
  const double u = 2.220446049250313e-16;
  const double Dt = t1 - t0;
  /* R12: round-off cap on the stage count, s_max = max(2, round(sqrt(rtol/(10 u)))) */
  int s_max = (int)floor(sqrt(rtol / (10.0 * u)) + 0.5);
  if (s_max < 2) s_max = 2;
  const size_t nn = (size_t)n;
  double *buf = (double *)malloc(sizeof(double) * nn * 9);
  double *f0 = buf, *fnew = buf + nn, *ynew = buf + 2 * nn, *v = buf + 3 * nn, *pw = buf + 4 * nn,
         *sw = buf + 6 * nn;
  int32_t nfe = 0, nacc = 0, nrej = 0, smax_used = 0;
  int status = ST_OK, flag = 0;
  double t = t0;

  f(t, y, f0, ctx);
  nfe++;
  double sigma = spectral_radius(f, ctx, n, t, y, f0, v, 0, &nfe, &flag, pw);
  int sigma_fresh = 1, need_sigma = 0, since_sigma = 0;

  /* initial step: Eq. 36-38, R14 weights atol + rtol |y_0|, R15 caps at the global step */
  double h, est0;
  {
    double h0 = (sigma > 0.0 && 1.0 / sigma < Dt) ? 1.0 / sigma : Dt;      /* Eq. 36 */
    double *z = pw, *g = pw + nn;
    for (int i = 0; i < n; i++) z[i] = y[i] + h0 * f0[i];
    f(t + h0, z, g, ctx);
    nfe++;
    double acc = 0.0;
    for (int i = 0; i < n; i++) {
      double d0 = h0 * (g[i] - f0[i]);                                     /* Eq. 37 */
      double wt = atol + rtol * fabs(y[i]);
      acc += (d0 / wt) * (d0 / wt);
    }
    double est = sqrt(acc / (double)n);                                    /* Eq. 31 */
    est0 = est;
    h = Dt;
    if (est > 0.0) {
      double h1 = 0.1 * h0 / sqrt(est);                                    /* Eq. 38 */
      if (h1 < Dt) h = h1;
    }
  }

  int have_prev = 0;           /* an accepted step precedes, with no rejection since (R13) */
  double err_old = 0.0, h_old = 0.0;
  long attempts = 0;
  int saw_nonfinite = 0;
  while (1) {
    int last = 0;
    int refreshed = (attempts == 0);
    if (1.1 * h >= t1 - t) { h = t1 - t; last = 1; }                       /* R5 */
    if (need_sigma) {                                                      /* P:233, R16 */
      sigma = spectral_radius(f, ctx, n, t, y, f0, v, 1, &nfe, &flag, pw);
      sigma_fresh = 1; need_sigma = 0; since_sigma = 0;
      refreshed = 1;
    }
    int s = 1 + (int)floor(sqrt(1.0 + 1.54 * h * sigma));                  /* Eq. 39, R12 truncation */
    if (s < 2) s = 2;
    if (s > s_max) {
      s = s_max;
      h = ((double)s_max * (double)s_max - 1.0) / (1.54 * sigma);
      last = 0;
    }
    if (s > smax_used) smax_used = s;
    if (++attempts > 1000000) { status = ST_MAXSTEPS; break; }
    rkc_step(f, ctx, n, t, y, f0, h, s, ynew, NULL, sw);
    f(t + h, ynew, fnew, ctx);
    nfe += s;
    /* Eq. 30-32 */
    double acc = 0.0;
    for (int i = 0; i < n; i++) {
      double del = 0.8 * (y[i] - ynew[i]) + 0.4 * h * (f0[i] + fnew[i]);
      double ym = fabs(y[i]) > fabs(ynew[i]) ? fabs(y[i]) : fabs(ynew[i]);
      double wt = atol + rtol * ym;
      acc += (del / wt) * (del / wt);
    }
    double err = sqrt(acc / (double)n);
    trace_row(tr, t, h, err, err <= 1.0, s, refreshed, sigma, attempts == 1 ? est0 : 0.0);
    if (err <= 1.0) {                                                      /* accept */
      nacc++;
      double fac;
      if (err > 0.0) {
        double e3 = cbrt(err);
        if (have_prev) fac = 0.8 * (cbrt(err_old) / e3) * (h / h_old) * (1.0 / e3);   /* Eq. 34, R13 */
        else fac = 0.8 / e3;
      } else fac = 10.0;                                                   /* R26 */
      if (fac < 0.1) fac = 0.1;
      if (fac > 10.0) fac = 10.0;                                          /* Eq. 33 */
      for (int i = 0; i < n; i++) { y[i] = ynew[i]; f0[i] = fnew[i]; }
      err_old = err; h_old = h; have_prev = 1;
      sigma_fresh = 0;
      if (++since_sigma >= 25) need_sigma = 1;
      if (last) { t = t1; break; }
      t += h;
      h *= fac;
    } else {                                                               /* reject: Eq. 35 */
      nrej++;
      double fac;
      if (isfinite(err)) {
        fac = 0.8 / cbrt(err);
        if (fac < 0.1) fac = 0.1;
        if (fac > 10.0) fac = 10.0;
      } else { fac = 0.1; saw_nonfinite = 1; }
      h *= fac;
      have_prev = 0;
      if (!sigma_fresh) need_sigma = 1;                                    /* R16 */
      double tmax = fabs(t) > fabs(t1) ? fabs(t) : fabs(t1);
      if (!(h > 10.0 * u * tmax)) { status = saw_nonfinite ? ST_NONFINITE : ST_UNDERFLOW; break; }
    }
  }
  if (status == ST_OK && flag) status = flag;
  if (stats) { stats[0] = nfe; stats[1] = nacc; stats[2] = nrej; stats[3] = smax_used; }
  free(buf);
  return status;
}

int ora_rkc_generic(ora_rhs_fn f, void *ctx, int n, double *y, double t0, double t1, double rtol,
                    double atol, int32_t *stats) {
  return rkc_driver(f, ctx, n, y, t0, t1, rtol, atol, stats, NULL);
}

/* test entry: the same driver with the step trace (see ora_rkck_trace) */
int ora_rkc_trace(ora_rhs_fn f, void *ctx, int n, double *y, double t0, double t1, double rtol, double atol,
                  int32_t *stats, double *rows, int64_t cap, int64_t *n_rows) {
  ora_trace tr = {rows, cap, 0};
  const int st = rkc_driver(f, ctx, n, y, t0, t1, rtol, atol, stats, &tr);
  if (n_rows) *n_rows = tr.n;
  return st;
}

/* ================================================================================================
 * Chemistry: mechanism tables and the source term, Eq. 2-6, DESIGN.md 4.3
 * ============================================================================================== */
typedef struct {
  int32_t n_species, n_reactions;
  const double *mol_weight, *nasa, *arr_A, *arr_beta, *arr_E;
  const int32_t *reac_ptr, *reac_species, *reac_nu, *prod_ptr, *prod_species, *prod_nu;
  int32_t n_third_body;
  const int32_t *tb_reaction, *tb_ptr, *tb_species;
  const double *tb_eff;
} ora_mech_desc;

typedef struct ora_mech {
  int K, R;
  double *W, *nasa, *A, *beta, *E;
  int32_t *reac_ptr, *reac_sp, *reac_nu, *prod_ptr, *prod_sp, *prod_nu;
  int32_t *tb_of; /* [R] index of the reaction's third-body row, or -1 */
  double *alpha;  /* [R3][K] dense third-body efficiencies (1 where not listed) */
  int R3;
  double *nasa_hi, *T_mid; /* optional second temperature range (ora_mech_set_thermo2), else NULL */
  int32_t *fo_of;          /* optional fall-off reactions (ora_mech_set_falloff): [R] row of the reaction or -1 */
  double *fo_low, *fo_troe;/* [n_fo][3] A_0, beta_0, E_0;  [n_fo][4] a, T***, T*, T** (a = NaN: Lindemann) */
} ora_mech;

static void *dup_mem(const void *src, size_t bytes) {
  void *p = malloc(bytes ? bytes : 1);
  if (p && bytes) memcpy(p, src, bytes);
  return p;
}

void ora_mech_free(ora_mech *m) {
  if (!m) return;
  free(m->W); free(m->nasa); free(m->A); free(m->beta); free(m->E);
  free(m->reac_ptr); free(m->reac_sp); free(m->reac_nu);
  free(m->prod_ptr); free(m->prod_sp); free(m->prod_nu);
  free(m->tb_of); free(m->alpha);
  free(m->nasa_hi); free(m->T_mid);
  free(m->fo_of); free(m->fo_low); free(m->fo_troe);
  free(m);
}

/* Pressure-dependent (fall-off) reactions (P:80 refers to the Chemkin manual for the formulation;
 * reading R31, that manual's form): for a reaction listed here the Arrhenius parameters given at load are the
 * high-pressure limit k_inf, (A_0, beta_0, E_0) the low-pressure limit k_0, and
 *     P_r = k_0 [M] / k_inf,   k = k_inf (P_r / (1 + P_r)) F,   rate of progress = k prod C  (no further [M] factor),
 * [M] = sum_k alpha_k C_k with the reaction's third-body efficiencies if it is also listed as a third-body reaction,
 * else all alpha = 1.  Lindemann: F = 1.  Troe: log10 F = log10 F_cent / (1 + ((log10 P_r + c)/(n - 0.14 (log10 P_r + c)))^2),
 * c = -0.4 - 0.67 log10 F_cent, n = 0.75 - 1.27 log10 F_cent, F_cent = (1-a) exp(-T/T***) + a exp(-T/T*) + exp(-T** / T)
 * (the last term is left out where T** is not finite).  troe[i][0] = NaN marks a Lindemann reaction. */
int ora_mech_set_falloff(ora_mech *m, int32_t n_fo, const int32_t *reaction, const double *low3, const double *troe4) {
  if (!m || n_fo < 0 || (n_fo > 0 && (!reaction || !low3 || !troe4))) return ORA_EINVAL;
  free(m->fo_of); free(m->fo_low); free(m->fo_troe);
  m->fo_of = (int32_t *)malloc(sizeof(int32_t) * (size_t)(m->R ? m->R : 1));
  m->fo_low = (double *)dup_mem(low3, sizeof(double) * 3 * (size_t)n_fo);
  m->fo_troe = (double *)dup_mem(troe4, sizeof(double) * 4 * (size_t)n_fo);
  if (!m->fo_of || !m->fo_low || !m->fo_troe) return ORA_ENOMEM;
  for (int j = 0; j < m->R; j++) m->fo_of[j] = -1;
  for (int i = 0; i < n_fo; i++) {
    if (reaction[i] < 0 || reaction[i] >= m->R || m->fo_of[reaction[i]] >= 0) return ORA_EINVAL;
    m->fo_of[reaction[i]] = i;
  }
  return ORA_OK;
}

/* Two temperature ranges for the NASA fits ("thermodynamic properties are typically fitted as
 * polynomials across different temperature ranges"; reading R30, the Chemkin convention): species k uses nasa_high[k]
 * where T > T_mid[k] and the coefficients given at load (the low range) where T <= T_mid[k].  Arrays are copied. */
int ora_mech_set_thermo2(ora_mech *m, const double *nasa_high, const double *T_mid) {
  if (!m || !nasa_high || !T_mid) return ORA_EINVAL;
  free(m->nasa_hi); free(m->T_mid);
  m->nasa_hi = (double *)dup_mem(nasa_high, sizeof(double) * 7 * (size_t)m->K);
  m->T_mid = (double *)dup_mem(T_mid, sizeof(double) * (size_t)m->K);
  return (m->nasa_hi && m->T_mid) ? ORA_OK : ORA_ENOMEM;
}

int ora_mech_load(const ora_mech_desc *d, ora_mech **out) {
  if (!d || !out || d->n_species < 1 || d->n_reactions < 0) return ORA_EINVAL;
  const int K = d->n_species, R = d->n_reactions, R3 = d->n_third_body;
  for (int j = 0; j < R; j++) {
    if (d->reac_ptr[j + 1] < d->reac_ptr[j] || d->prod_ptr[j + 1] < d->prod_ptr[j]) return ORA_EINVAL;
    for (int e = d->reac_ptr[j]; e < d->reac_ptr[j + 1]; e++)
      if (d->reac_species[e] < 0 || d->reac_species[e] >= K || d->reac_nu[e] < 1) return ORA_EINVAL;
    for (int e = d->prod_ptr[j]; e < d->prod_ptr[j + 1]; e++)
      if (d->prod_species[e] < 0 || d->prod_species[e] >= K || d->prod_nu[e] < 1) return ORA_EINVAL;
  }
  ora_mech *m = (ora_mech *)calloc(1, sizeof(ora_mech));
  if (!m) return ORA_ENOMEM;
  m->K = K; m->R = R; m->R3 = R3;
  m->W = dup_mem(d->mol_weight, sizeof(double) * K);
  m->nasa = dup_mem(d->nasa, sizeof(double) * K * 7);
  m->A = dup_mem(d->arr_A, sizeof(double) * R);
  m->beta = dup_mem(d->arr_beta, sizeof(double) * R);
  m->E = dup_mem(d->arr_E, sizeof(double) * R);
  m->reac_ptr = dup_mem(d->reac_ptr, sizeof(int32_t) * (R + 1));
  m->prod_ptr = dup_mem(d->prod_ptr, sizeof(int32_t) * (R + 1));
  const int nr = R ? d->reac_ptr[R] : 0, np = R ? d->prod_ptr[R] : 0;
  m->reac_sp = dup_mem(d->reac_species, sizeof(int32_t) * nr);
  m->reac_nu = dup_mem(d->reac_nu, sizeof(int32_t) * nr);
  m->prod_sp = dup_mem(d->prod_species, sizeof(int32_t) * np);
  m->prod_nu = dup_mem(d->prod_nu, sizeof(int32_t) * np);
  m->tb_of = (int32_t *)malloc(sizeof(int32_t) * (R ? R : 1));
  m->alpha = (double *)malloc(sizeof(double) * (size_t)(R3 ? R3 : 1) * K);
  for (int j = 0; j < R; j++) m->tb_of[j] = -1;
  for (int r = 0; r < R3; r++) {
    const int j = d->tb_reaction[r];
    if (j < 0 || j >= R) { ora_mech_free(m); return ORA_EINVAL; }
    m->tb_of[j] = r;
    for (int k = 0; k < K; k++) m->alpha[(size_t)r * K + k] = 1.0;
    for (int e = d->tb_ptr[r]; e < d->tb_ptr[r + 1]; e++) {
      if (d->tb_species[e] < 0 || d->tb_species[e] >= K) { ora_mech_free(m); return ORA_EINVAL; }
      m->alpha[(size_t)r * K + d->tb_species[e]] = d->tb_eff[e];
    }
  }
  *out = m;
  return ORA_OK;
}

/* f(y): y = {T, Y_1..Y_K}.  work: 2K + R doubles.
 * cv = 0: constant pressure, p = pressure in dyn/cm^2 (Eq. 6).
 * cv = 1: constant volume (P:243 mentions the variant without equations; reading R29, the textbook form): p carries
 *         the density rho in g/cm^3, constant over the call, and the energy equation is
 *         rho c_v dT/dt = - sum_k u_k omega_k W_k  with  u_k = h_k - Ru T / W_k  and  c_v = c_p - Ru / Wbar. */
static void chem_rhs(const ora_mech *m, const double *y, double p, double *dydt, double *work, int cv) {
  const int K = m->K, R = m->R;
  const double T = y[0];
  const double *Y = y + 1;
  double *C = work, *wdot = work + K, *Omega = work + 2 * (size_t)K;
  /* R9a: ideal gas at constant pressure: rho = p Wbar/(Ru T), 1/Wbar = sum Y_k/W_k; C_k = rho Y_k / W_k */
  double Sum = 0.0;
  for (int k = 0; k < K; k++) Sum += Y[k] / m->W[k];
  const double rho = cv ? p : p / (ORA_RU * T * Sum);
  for (int k = 0; k < K; k++) C[k] = rho * Y[k] / m->W[k];
  for (int j = 0; j < R; j++) {
    const double kj = m->A[j] * pow(T, m->beta[j]) * exp(-m->E[j] / (ORA_RC * T));   /* Eq. 5, literal */
    double rate = kj;
    if (m->fo_of && m->fo_of[j] >= 0) {     /* R31: fall-off, kj is k_inf */
      const double *lo = m->fo_low + 3 * (size_t)m->fo_of[j], *tr = m->fo_troe + 4 * (size_t)m->fo_of[j];
      double M = 0.0;
      if (m->tb_of[j] >= 0) {
        const double *al = m->alpha + (size_t)m->tb_of[j] * K;
        for (int k = 0; k < K; k++) M += al[k] * C[k];
      } else {
        for (int k = 0; k < K; k++) M += C[k];
      }
      const double k0 = lo[0] * pow(T, lo[1]) * exp(-lo[2] / (ORA_RC * T));
      const double Pr = k0 * M / kj;
      double F = 1.0;                       /* Lindemann */
      if (tr[0] == tr[0]) {                 /* Troe (a is not NaN) */
        double Fcent = (1.0 - tr[0]) * exp(-T / tr[1]) + tr[0] * exp(-T / tr[2]);
        if (isfinite(tr[3])) Fcent += exp(-tr[3] / T);
        const double lF = log10(Fcent), lP = log10(Pr);
        const double c = -0.4 - 0.67 * lF, nn = 0.75 - 1.27 * lF;
        const double x = (lP + c) / (nn - 0.14 * (lP + c));
        F = pow(10.0, lF / (1.0 + x * x));
      }
      rate = kj * (Pr / (1.0 + Pr)) * F;
    } else if (m->tb_of[j] >= 0) {          /* R22: [M]_j = sum_k alpha_jk C_k */
      const double *al = m->alpha + (size_t)m->tb_of[j] * K;
      double M = 0.0;
      for (int k = 0; k < K; k++) M += al[k] * C[k];
      rate *= M;
    }
    for (int e = m->reac_ptr[j]; e < m->reac_ptr[j + 1]; e++) /* Eq. 4, integer orders; R19 no clipping */
      for (int q = 0; q < m->reac_nu[e]; q++) rate *= C[m->reac_sp[e]];
    Omega[j] = rate;
  }
  for (int k = 0; k < K; k++) wdot[k] = 0.0;
  for (int j = 0; j < R; j++) {             /* Eq. 3 */
    for (int e = m->prod_ptr[j]; e < m->prod_ptr[j + 1]; e++) wdot[m->prod_sp[e]] += m->prod_nu[e] * Omega[j];
    for (int e = m->reac_ptr[j]; e < m->reac_ptr[j + 1]; e++) wdot[m->reac_sp[e]] -= m->reac_nu[e] * Omega[j];
  }
  /* R8a: NASA 7-coefficient fits, one range */
  double cp_sum = 0.0, h_sum = 0.0;
  const double T2 = T * T, T3 = T2 * T, T4 = T3 * T;
  for (int k = 0; k < K; k++) {
    const double *a = m->nasa + 7 * (size_t)k;
    if (m->T_mid && T > m->T_mid[k]) a = m->nasa_hi + 7 * (size_t)k; /* R30: the high range above T_mid */
    const double cpR = a[0] + a[1] * T + a[2] * T2 + a[3] * T3 + a[4] * T4;
    const double hRT = a[0] + a[1] * T / 2.0 + a[2] * T2 / 3.0 + a[3] * T3 / 4.0 + a[4] * T4 / 5.0 + a[5] / T;
    cp_sum += Y[k] * cpR / m->W[k];
    h_sum += hRT * wdot[k];                 /* (h_k W_k)/(Ru T) * omega_k */
  }
  const double cp = ORA_RU * cp_sum;        /* mass-averaged c_p */
  if (cv) {                                 /* R29 */
    double w_sum = 0.0;
    for (int k = 0; k < K; k++) w_sum += wdot[k];
    const double cvm = cp - ORA_RU * Sum;   /* c_v = c_p - Ru / Wbar */
    dydt[0] = -(ORA_RU * T * (h_sum - w_sum)) / (rho * cvm);    /* sum_k (h_k/(Ru T) - 1) omega_k */
  } else {
    dydt[0] = -(ORA_RU * T * h_sum) / (rho * cp);               /* Eq. 6 */
  }
  for (int k = 0; k < K; k++) dydt[1 + k] = m->W[k] * wdot[k] / rho; /* Eq. 2 */
}

void ora_rhs(const ora_mech *m, const double *y, double p, double *dydt) {
  double *work = (double *)malloc(sizeof(double) * (2 * (size_t)m->K + (size_t)m->R + 1));
  chem_rhs(m, y, p, dydt, work, 0);
  free(work);
}

/* constant volume: rho in g/cm^3 */
void ora_rhs_cv(const ora_mech *m, const double *y, double rho, double *dydt) {
  double *work = (double *)malloc(sizeof(double) * (2 * (size_t)m->K + (size_t)m->R + 1));
  chem_rhs(m, y, rho, dydt, work, 1);
  free(work);
}

typedef struct { const ora_mech *m; double p; double *work; int cv; } chem_ctx;

static void chem_rhs_cb(double t, const double *y, double *dydt, void *ctx) {
  (void)t;                                   /* autonomous */
  chem_ctx *c = (chem_ctx *)ctx;
  chem_rhs(c->m, y, c->p, dydt, c->work, c->cv);
}

/* Batch entry mirroring the product's integrate(): states are HOST, SoA [(K+1)][ld], updated in place.
 * method 0 = RKCK, 1 = RKC.  status [N] and stats [4][N] may be NULL.  nthreads <= 0 -> OpenMP default. */
static int integrate_closure(const ora_mech *m, double *states, const double *pressure, double p_uniform, int64_t N,
                             int64_t ld, double t, double dt, double rtol, double atol, int32_t method,
                             int32_t *status, int32_t *stats, int32_t nthreads, int cv) {
  if (!m || !states || N < 0 || ld < N || (method != 0 && method != 1) || !(dt > 0.0) || !(rtol > 0.0) ||
      !(atol >= 0.0))
    return ORA_EINVAL;
  const int n = m->K + 1;
#ifdef _OPENMP
  if (nthreads <= 0) nthreads = omp_get_max_threads();
#else
  nthreads = 1;
#endif
#pragma omp parallel num_threads(nthreads)
  {
    double *y = (double *)malloc(sizeof(double) * (size_t)n);
    double *work = (double *)malloc(sizeof(double) * (2 * (size_t)m->K + (size_t)m->R + 1));
    chem_ctx ctx;
    ctx.m = m;
    ctx.work = work;
    ctx.cv = cv;
#pragma omp for schedule(dynamic, 16)
    for (int64_t i = 0; i < N; i++) {
      for (int c = 0; c < n; c++) y[c] = states[(size_t)c * ld + i];
      ctx.p = pressure ? pressure[i] : p_uniform;
      int32_t st[4];
      int code = (method == 0) ? ora_rkck_generic(chem_rhs_cb, &ctx, n, y, t, t + dt, rtol, atol, st)
                               : ora_rkc_generic(chem_rhs_cb, &ctx, n, y, t, t + dt, rtol, atol, st);
      for (int c = 0; c < n; c++) states[(size_t)c * ld + i] = y[c];
      if (status) status[i] = code;
      if (stats)
        for (int q = 0; q < 4; q++) stats[(size_t)q * N + i] = st[q];
    }
    free(y);
    free(work);
  }
  return ORA_OK;
}

int ora_integrate(const ora_mech *m, double *states, const double *pressure, double p_uniform, int64_t N,
                  int64_t ld, double t, double dt, double rtol, double atol, int32_t method,
                  int32_t *status, int32_t *stats, int32_t nthreads) {
  return integrate_closure(m, states, pressure, p_uniform, N, ld, t, dt, rtol, atol, method, status, stats, nthreads, 0);
}

/* constant volume (R29): density[] / rho_uniform in g/cm^3 in place of the pressure */
int ora_integrate_cv(const ora_mech *m, double *states, const double *density, double rho_uniform, int64_t N,
                     int64_t ld, double t, double dt, double rtol, double atol, int32_t method,
                     int32_t *status, int32_t *stats, int32_t nthreads) {
  return integrate_closure(m, states, density, rho_uniform, N, ld, t, dt, rtol, atol, method, status, stats, nthreads, 1);
}

/* ================================================================================================
 * Appendix A: reversible -> irreversible conversion.  SURVEY 8(f)-f2.
 * ============================================================================================== */

/* Eq. A.10-A.12: the reverse Arrhenius parameters (A_r, beta_r, T_ar = E_r / R) through the three points
 * (T_i, k_ri), with x_i = ln T_i and a_i = ln k_ri.  out[0] = A_r, out[1] = beta_r, out[2] = T_ar (kelvin). */
void ora_fit_reverse(const double *T, const double *kr, double *out) {
  const double T1 = T[0], T2 = T[1], T3 = T[2];
  const double x1 = log(T1), x2 = log(T2), x3 = log(T3);
  const double a1 = log(kr[0]), a2 = log(kr[1]), a3 = log(kr[2]);
  const double den = x1 * T1 * (T3 - T2) + x2 * T2 * (T1 - T3) + x3 * T3 * (T2 - T1);
  const double beta = (a1 * T1 * (T3 - T2) + a2 * T2 * (T1 - T3) + a3 * T3 * (T2 - T1)) / den;            /* A.10 */
  const double Tar = T1 * T2 * T3 * (a1 * (x2 - x3) + a2 * (x3 - x1) + a3 * (x1 - x2)) / den;              /* A.11 */
  const double lnA = (a1 * T1 * (x2 * T2 - x3 * T3) + a2 * T2 * (x3 * T3 - x1 * T1) + a3 * T3 * (x1 * T1 - x2 * T2)) / den; /* A.12 */
  out[0] = exp(lnA);
  out[1] = beta;
  out[2] = Tar;
}

/* The equilibrium constant in concentration units of reaction j of a loaded mechanism at temperature T (reading R32:
 * the paper takes "the equilibrium constants" as known, P:84 / P:461; the Chemkin form is used):
 *     K_p = exp( sum_k nu_k (s_k/R - h_k/(R T)) ),   K_c = K_p (P_atm / (Ru T))^(sum_k nu_k),   nu = nu'' - nu',
 *     s_k/R = a1 ln T + a2 T + a3 T^2/2 + a4 T^3/3 + a5 T^4/4 + a7,   h_k/(RT) = a1 + a2 T/2 + .. + a5 T^4/5 + a6/T,
 * P_atm = 1.01325e6 dyn/cm^2; the NASA range of each species is picked by R30 when the mechanism has two. */
double ora_equilibrium_constant(const ora_mech *m, int j, double T) {
  double dG = 0.0;   /* sum_k nu_k (s_k/R - h_k/RT) */
  int dnu = 0;
  for (int side = 0; side < 2; side++) {
    const int32_t *ptr = side ? m->prod_ptr : m->reac_ptr, *sp = side ? m->prod_sp : m->reac_sp,
                  *nu = side ? m->prod_nu : m->reac_nu;
    const int sign = side ? 1 : -1;
    for (int e = ptr[j]; e < ptr[j + 1]; e++) {
      const int k = sp[e];
      const double *a = m->nasa + 7 * (size_t)k;
      if (m->T_mid && T > m->T_mid[k]) a = m->nasa_hi + 7 * (size_t)k;
      const double sR = a[0] * log(T) + a[1] * T + a[2] * T * T / 2.0 + a[3] * T * T * T / 3.0 + a[4] * T * T * T * T / 4.0 + a[6];
      const double hRT = a[0] + a[1] * T / 2.0 + a[2] * T * T / 3.0 + a[3] * T * T * T / 4.0 + a[4] * T * T * T * T / 5.0 + a[5] / T;
      dG += sign * nu[e] * (sR - hRT);
      dnu += sign * nu[e];
    }
  }
  return exp(dG) * pow(1.01325e6 / (ORA_RU * T), (double)dnu);
}

/* Appendix A for reaction j: k_r = k_f / K_c at the three temperatures, then Eq. A.10-A.12.
 * out[0] = A_r, out[1] = beta_r, out[2] = E_r in cal/mol (= T_ar R_c). */
void ora_reverse_parameters(const ora_mech *m, int j, const double *T3, double *out) {
  double kr[3];
  for (int i = 0; i < 3; i++) {
    const double kf = m->A[j] * pow(T3[i], m->beta[j]) * exp(-m->E[j] / (ORA_RC * T3[i]));
    kr[i] = kf / ora_equilibrium_constant(m, j, T3[i]);
  }
  ora_fit_reverse(T3, kr, out);
  out[2] *= ORA_RC;
}

int ora_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
