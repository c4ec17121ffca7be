/*
 * ckb_device.cuh -- device code of the batched chemistry integrator (sm_100a, FP64).
 *
 * One templated "system" type maps an ODE system onto L lanes (L = 1: thread-per-ODE, the paper's
 * mapping P:255; L = 32: warp-per-ODE; L = 8/16: sub-warp).  Component c of y = {T, Y_1..Y_K}
 * lives in lane (c mod L), register slot (c div L); every stage vector of the integrators is a
 * register array double[NV] with static indexing only.  The runtime-indexed quantities of the source
 * term (concentrations C_k, third-body concentrations [M], net rates of progress q_s) live in shared
 * memory, interleaved so that thread-per-ODE access is bank-conflict free.
 *
 * Source term: Eq. 2-6.  Integrators: RKCK Eq. 7-17, RKC Eq. 18-39.
 * The readings of the paper where it is silent (R-numbers) are listed in DESIGN.md section 4.
 * Nothing here is shared with oracle/ (constants that appear in both are typed twice).
 */
#pragma once
#include <math.h>
#include <stdint.h>

#include "ckb_tables.h"

namespace ckb {

/* R20: physical constants */
#define CKB_RU 8.314462618e7 /* erg/(mol K) */

/* ------------------------------------------------------------------------------------------------
 * Sys<L, NV, CT>: one ODE system on L lanes with NV register slots per lane; tables in constant
 * memory (CT) or global/L1.
 * ---------------------------------------------------------------------------------------------- */
template <int L_, int NV_, class TAB>
struct Sys {
  static constexpr int L = L_, NV = NV_, G = 32 / L_;
  const DevMech &m;
  const TAB &tab;
  double *sC, *sM, *sQ; /* this group's shared arrays, element idx at [idx*G] */
  unsigned mask;        /* lanes of this group */
  int g;                /* lane within the group */
  int src0;             /* warp lane that holds component 0 (T) */
  double p;             /* pressure, dyn/cm^2 (R24: constant over the call) */
  int nfe;

  __device__ __forceinline__ Sys(const DevMech &m_, const TAB &tab_) : m(m_), tab(tab_) {}
  __device__ __forceinline__ unsigned long long tw(int i) const { return tab.ld(i); }
  __device__ __forceinline__ double td(int i) const { return __longlong_as_double((long long)tab.ld(i)); }

  __device__ __forceinline__ void gsync() const {
    if (L > 1) __syncwarp(mask);
  }
  __device__ __forceinline__ double gsum(double x) const {
#pragma unroll
    for (int o = L / 2; o > 0; o >>= 1) x += __shfl_xor_sync(mask, x, o);
    return x;
  }
  __device__ __forceinline__ double gmax(double x) const {
#pragma unroll
    for (int o = L / 2; o > 0; o >>= 1) x = fmax(x, __shfl_xor_sync(mask, x, o));
    return x;
  }
  __device__ __forceinline__ double bcast0(double x) const {
    if (L == 1) return x;
    return __shfl_sync(mask, x, src0);
  }
  __device__ __forceinline__ bool valid(int i) const { return g + L * i < m.n; }

  /* f(y): Eq. 2-6.  y, f: component (g + L*i) in slot i. */
  __device__ __forceinline__ void rhs(const double (&y)[NV], double (&f)[NV]) {
    nfe++;
    const int K = m.K;
    const double T = bcast0(y[0]);
    const double invT = 1.0 / T;
    const double lnT = log(T);
    double s1 = 0.0, s2 = 0.0;
    double hrt[NV], yw[NV];
#pragma unroll
    for (int i = 0; i < NV; i++) {
      const int c = g + L * i, k = c - 1;
      hrt[i] = 0.0;
      yw[i] = 0.0;
      if (c >= 1 && c <= K) {
        /* R8a: cp_k/R = a1 + a2 T + ... + a5 T^4;  h_k/(RT) = a1 + a2 T/2 + ... + a5 T^4/5 + a6/T */
        double cp = td(m.o_cp + 4 * K + k);
        double h = td(m.o_h + 4 * K + k);
#pragma unroll
        for (int q = 3; q >= 0; q--) {
          cp = fma(cp, T, td(m.o_cp + q * K + k));
          h = fma(h, T, td(m.o_h + q * K + k));
        }
        h = fma(td(m.o_h + 5 * K + k), invT, h);
        const double v = y[i] * td(m.o_invW + k); /* Y_k / W_k */
        yw[i] = v;
        hrt[i] = h;
        s1 += v;
        s2 = fma(v, cp, s2);
      }
    }
    s1 = gsum(s1);
    s2 = gsum(s2);
    /* R9a: ideal gas at constant pressure: rho = p / (Ru T sum_k Y_k/W_k), C_k = rho Y_k / W_k */
    const double ctot = p / (CKB_RU * T);
    const double rho = ctot / s1;
#pragma unroll
    for (int i = 0; i < NV; i++) {
      const int c = g + L * i;
      if (c >= 1 && c <= K) sC[(c - 1) * G] = rho * yw[i];
    }
    gsync();
    /* R22: [M] = sum_k alpha_k C_k = C_tot + sum_listed (alpha_k - 1) C_k, one value per efficiency set */
    for (int t = g; t < m.NTB; t += L) {
      const int e0 = (int)tw(m.o_tbptr + t), e1 = (int)tw(m.o_tbptr + t + 1);
      double M = ctot;
      for (int e = e0; e < e1; e++)
        M = fma(td(m.o_tbam1 + e), sC[(int)tw(m.o_tbsp + e) * G], M);
      sM[t * G] = M;
    }
    gsync();
    /* Eq. 4-5: q_s = [M] (k_f prod C_reactants - k_r prod C_products); absent molecules point at C = 1 */
#pragma unroll 2
    for (int s = g; s < m.NS; s += L) {
      const unsigned long long w = tw(m.o_idx + s);
      const double xf = fma(td(m.o_bf + s), lnT, td(m.o_lnAf + s)) -
                        td(m.o_thf + s) * invT;
      const double xr = fma(td(m.o_br + s), lnT, td(m.o_lnAr + s)) -
                        td(m.o_thr + s) * invT;
      const unsigned lo = (unsigned)w, hi = (unsigned)(w >> 32);
      const double pf = sC[(lo & 255u) * G] * sC[((lo >> 8) & 255u) * G] * sC[((lo >> 16) & 255u) * G];
      const double pr = sC[(lo >> 24) * G] * sC[(hi & 255u) * G] * sC[((hi >> 8) & 255u) * G];
      const double kf = exp(xf), kr = exp(xr);
      sQ[s * G] = (kf * pf - kr * pr) * sM[(hi >> 16) * G];
    }
    gsync();
    /* Eq. 3: omega_k = sum_s (nu''_ks - nu'_ks) q_s (gather);  Eq. 2: dY_k/dt = W_k omega_k / rho */
    const double invrho = 1.0 / rho;
    double s3 = 0.0;
#pragma unroll
    for (int i = 0; i < NV; i++) {
      const int c = g + L * i, k = c - 1;
      f[i] = 0.0;
      if (c >= 1 && c <= K) {
        const int e0 = (int)tw(m.o_gptr + k), e1 = (int)tw(m.o_gptr + k + 1);
        double acc = 0.0;
        for (int e = e0; e < e1; e++) {
          const unsigned long long w = tw(m.o_gat + e);
          const double coef = __longlong_as_double((long long)(w & ~0xFFFFull));
          acc = fma(coef, sQ[(int)(w & 0xFFFFull) * G], acc);
        }
        f[i] = td(m.o_W + k) * acc * invrho;
        s3 = fma(hrt[i], acc, s3);
      }
    }
    s3 = gsum(s3);
    /* Eq. 6: dT/dt = -(Ru T sum_k (h_k/RT) omega_k) / (rho cp), cp = Ru sum_k Y_k (cp_k/R) / W_k */
    if (g == 0) f[0] = -(T * s3) / (rho * s2);
  }
};

/* per-system status codes (mirrors ckb.h) */
#define ST_OK 0
#define ST_MAXSTEPS 1
#define ST_UNDERFLOW 2
#define ST_NONFINITE 3
#define ST_SIGMA 4

#define CKB_U 2.220446049250313e-16      /* 2^-52 */
#define CKB_SQRTU 1.4901161193847656e-08 /* 2^-26 */

/* ------------------------------------------------------------------------------------------------
 * RKCK driver: Eq. 7-17, Table 1; DESIGN.md 4.2 (R1-R7, R25).
 * ---------------------------------------------------------------------------------------------- */
template <class S>
__device__ __forceinline__ int rkck_driver(S &sys, double (&y)[S::NV], double t0, double t1, double rtol,
                                           double atol, int (&st)[4]) {
  constexpr int NV = S::NV;
  /* Table 1 (R1: Cash-Karp values) */
  constexpr double B21 = 1.0 / 5.0;
  constexpr double B31 = 3.0 / 40.0, B32 = 9.0 / 40.0;
  constexpr double B41 = 3.0 / 10.0, B42 = -9.0 / 10.0, B43 = 6.0 / 5.0;
  constexpr double B51 = -11.0 / 54.0, B52 = 5.0 / 2.0, B53 = -70.0 / 27.0, B54 = 35.0 / 27.0;
  constexpr double B61 = 1631.0 / 55296.0, B62 = 175.0 / 512.0, B63 = 575.0 / 13824.0,
                   B64 = 44275.0 / 110592.0, B65 = 253.0 / 4096.0;
  constexpr double C1 = 37.0 / 378.0, C3 = 250.0 / 621.0, C4 = 125.0 / 594.0, C6 = 512.0 / 1771.0;
  constexpr double D1 = C1 - 2825.0 / 27648.0, D3 = C3 - 18575.0 / 48384.0, D4 = C4 - 13525.0 / 55296.0,
                   D5 = -277.0 / 14336.0, D6 = C6 - 1.0 / 4.0;
  constexpr double SAFETY = 0.9;

  double k1[NV], k2[NV], k3[NV], k4[NV], k5[NV], k6[NV], yt[NV];
  int nacc = 0, nrej = 0, status = ST_OK;
  double t = t0, h = t1 - t0; /* R4: first trial step = the whole global step */
  bool have_k1 = false, saw_nonfinite = false;
  int attempts = 0;
  while (true) {
    bool last = false;
    if (1.1 * h >= t1 - t) { /* R5 */
      const double hn = t1 - t;
      if (have_k1) {
        const double r = hn / h;
#pragma unroll
        for (int i = 0; i < NV; i++) k1[i] *= r;
      }
      h = hn;
      last = true;
    }
    if (!have_k1) { /* Eq. 7 */
      sys.rhs(y, k1);
#pragma unroll
      for (int i = 0; i < NV; i++) k1[i] *= h;
      have_k1 = true;
    }
    if (++attempts > 1000000) { /* R7 */
      status = ST_MAXSTEPS;
      break;
    }
    /* Eq. 8-12 */
#pragma unroll
    for (int i = 0; i < NV; i++) yt[i] = fma(B21, k1[i], y[i]);
    sys.rhs(yt, k2);
#pragma unroll
    for (int i = 0; i < NV; i++) {
      k2[i] *= h;
      yt[i] = fma(B32, k2[i], fma(B31, k1[i], y[i]));
    }
    sys.rhs(yt, k3);
#pragma unroll
    for (int i = 0; i < NV; i++) {
      k3[i] *= h;
      yt[i] = fma(B43, k3[i], fma(B42, k2[i], fma(B41, k1[i], y[i])));
    }
    sys.rhs(yt, k4);
#pragma unroll
    for (int i = 0; i < NV; i++) {
      k4[i] *= h;
      yt[i] = fma(B54, k4[i], fma(B53, k3[i], fma(B52, k2[i], fma(B51, k1[i], y[i]))));
    }
    sys.rhs(yt, k5);
#pragma unroll
    for (int i = 0; i < NV; i++) {
      k5[i] *= h;
      yt[i] = fma(B65, k5[i], fma(B64, k4[i], fma(B63, k3[i], fma(B62, k2[i], fma(B61, k1[i], y[i])))));
    }
    sys.rhs(yt, k6);
    /* Eq. 13, 15, 16 (R2), 17 (R3) */
    double errmax = 0.0;
#pragma unroll
    for (int i = 0; i < NV; i++) {
      k6[i] *= h;
      const double yn = fma(C6, k6[i], fma(C4, k4[i], fma(C3, k3[i], fma(C1, k1[i], y[i]))));
      const double dl = fma(D6, k6[i], fma(D5, k5[i], fma(D4, k4[i], fma(D3, k3[i], D1 * k1[i]))));
      yt[i] = yn;
      if (sys.valid(i)) {
        const double d0 = fma(rtol, fabs(y[i]) + fabs(k1[i]), atol);
        double e = fabs(dl) / d0;
        if (!isfinite(yn) || isnan(e)) e = INFINITY;
        errmax = fmax(errmax, e);
      }
    }
    errmax = sys.gmax(errmax);
    if (errmax <= 1.0) { /* P:139 accept */
      nacc++;
#pragma unroll
      for (int i = 0; i < NV; i++) y[i] = yt[i];
      have_k1 = false;
      if (last) break;
      t += h;
      double fac = (errmax > 0.0) ? SAFETY * pow(errmax, -0.2) : 5.0;
      if (fac > 5.0) fac = 5.0;
      h *= fac;
    } else {
      nrej++;
      double fac;
      if (isfinite(errmax)) {
        fac = SAFETY * pow(errmax, -0.25);
        if (fac < 0.1) fac = 0.1;
      } else {
        fac = 0.1;
        saw_nonfinite = true;
      }
#pragma unroll
      for (int i = 0; i < NV; i++) k1[i] *= fac; /* R25 */
      h *= fac;
      const double tmax = fmax(fabs(t), fabs(t1));
      if (!(h > 10.0 * CKB_U * tmax)) { /* R6 */
        status = saw_nonfinite ? ST_NONFINITE : ST_UNDERFLOW;
        break;
      }
    }
  }
  st[0] = sys.nfe;
  st[1] = nacc;
  st[2] = nrej;
  st[3] = 0;
  return status;
}

/* ------------------------------------------------------------------------------------------------
 * Spectral radius by the nonlinear power method (R17/R18).
 * y, fy = f(y); v = previous eigenvector estimate (have_v) -- on return the new one.  z, gq: scratch.
 * ---------------------------------------------------------------------------------------------- */
template <class S>
__device__ __forceinline__ double spectral_radius(S &sys, const double (&y)[S::NV], const double (&fy)[S::NV],
                                                  double (&v)[S::NV], bool have_v, int &flag,
                                                  double (&z)[S::NV], double (&gq)[S::NV]) {
  constexpr int NV = S::NV;
  if (!have_v) {
#pragma unroll
    for (int i = 0; i < NV; i++) v[i] = fy[i];
  }
  double a = 0.0, b = 0.0;
#pragma unroll
  for (int i = 0; i < NV; i++) {
    a = fma(y[i], y[i], a);
    b = fma(v[i], v[i], b);
  }
  const double ynrm = sqrt(sys.gsum(a)), vnrm = sqrt(sys.gsum(b));
  double d;
  if (ynrm != 0.0 && vnrm != 0.0) {
    d = ynrm * CKB_SQRTU;
    const double r = d / vnrm;
#pragma unroll
    for (int i = 0; i < NV; i++) z[i] = fma(v[i], r, y[i]);
  } else if (ynrm != 0.0) {
    d = ynrm * CKB_SQRTU;
#pragma unroll
    for (int i = 0; i < NV; i++) z[i] = y[i] * (1.0 + CKB_SQRTU);
  } else if (vnrm != 0.0) {
    d = CKB_U;
    const double r = d / vnrm;
#pragma unroll
    for (int i = 0; i < NV; i++) z[i] = v[i] * r;
  } else {
    d = CKB_U;
#pragma unroll
    for (int i = 0; i < NV; i++) z[i] = sys.valid(i) ? d : 0.0;
  }
  double sigma = 0.0;
  bool converged = false;
  for (int it = 1; it <= 50; it++) {
    sys.rhs(z, gq);
    double dd = 0.0;
#pragma unroll
    for (int i = 0; i < NV; i++) {
      const double e = gq[i] - fy[i];
      dd = fma(e, e, dd);
    }
    dd = sqrt(sys.gsum(dd));
    const double sigma_prev = sigma;
    sigma = dd / d;
    const double fl = sigma > 1e-300 ? sigma : 1e-300;
    if (it >= 2 && fabs(sigma - sigma_prev) <= 0.01 * fl) {
      converged = true;
      break;
    }
    if (dd != 0.0) {
      const double r = d / dd;
#pragma unroll
      for (int i = 0; i < NV; i++) z[i] = fma(gq[i] - fy[i], r, y[i]);
    } else {
      const int ci = it % sys.m.n;
#pragma unroll
      for (int i = 0; i < NV; i++)
        if (sys.g + S::L * i == ci) z[i] = y[i] - (z[i] - y[i]);
    }
  }
#pragma unroll
  for (int i = 0; i < NV; i++) v[i] = z[i] - y[i];
  if (!converged) flag = ST_SIGMA;
  return 1.2 * sigma; /* R18 */
}

/* ------------------------------------------------------------------------------------------------
 * RKC driver: Eq. 18-39 and P:233; DESIGN.md 4.4 (R8-R18, R26).
 * ---------------------------------------------------------------------------------------------- */
template <class S>
__device__ __forceinline__ int rkc_driver(S &sys, double (&y)[S::NV], double t0, double t1, double rtol,
                                          double atol, int (&st)[4]) {
  constexpr int NV = S::NV;
  const double Dt = t1 - t0;
  const double nd = (double)sys.m.n;
  int s_max = (int)floor(sqrt(rtol / (10.0 * CKB_U)) + 0.5); /* R12 */
  if (s_max < 2) s_max = 2;
  double f0[NV], fj[NV], wjm1[NV], wjm2[NV], v[NV];
  int nacc = 0, nrej = 0, smax_used = 0, status = ST_OK, flag = 0;
  double t = t0;

  sys.rhs(y, f0);
  double sigma = spectral_radius(sys, y, f0, v, false, flag, wjm1, fj);
  bool sigma_fresh = true, need_sigma = false;
  int since_sigma = 0;

  /* initial step: Eq. 36-38 (R14, R15) */
  double h;
  {
    const double h0 = (sigma > 0.0 && 1.0 / sigma < Dt) ? 1.0 / sigma : Dt;
#pragma unroll
    for (int i = 0; i < NV; i++) wjm1[i] = fma(h0, f0[i], y[i]);
    sys.rhs(wjm1, fj);
    double acc = 0.0;
#pragma unroll
    for (int i = 0; i < NV; i++) {
      if (sys.valid(i)) {
        const double d0 = h0 * (fj[i] - f0[i]);
        const double wt = fma(rtol, fabs(y[i]), atol);
        const double q = d0 / wt;
        acc = fma(q, q, acc);
      }
    }
    const double est = sqrt(sys.gsum(acc) / nd);
    h = Dt;
    if (est > 0.0) {
      const double h1 = 0.1 * h0 / sqrt(est);
      if (h1 < Dt) h = h1;
    }
  }

  bool have_prev = false, saw_nonfinite = false;
  double err_old = 0.0, h_old = 0.0;
  int attempts = 0;
  while (true) {
    bool last = false;
    if (1.1 * h >= t1 - t) { /* R5 */
      h = t1 - t;
      last = true;
    }
    if (need_sigma) { /* P:233, R16 */
      sigma = spectral_radius(sys, y, f0, v, true, flag, wjm1, fj);
      sigma_fresh = true;
      need_sigma = false;
      since_sigma = 0;
    }
    int s = 1 + (int)floor(sqrt(fma(1.54 * h, sigma, 1.0))); /* Eq. 39, R12 */
    if (s < 2) s = 2;
    if (s > s_max) {
      s = s_max;
      h = ((double)s_max * (double)s_max - 1.0) / (1.54 * sigma);
      last = false;
    }
    if (s > smax_used) smax_used = s;
    if (++attempts > 1000000) {
      status = ST_MAXSTEPS;
      break;
    }
    /* coefficients, Eq. 22-26: w0 (R8), then w1 = T_s'(w0)/T_s''(w0) by a scalar pre-pass */
    const double w0 = 1.0 + (2.0 / 13.0) / ((double)s * (double)s);
    double w1;
    {
      double Tm2 = 1.0, Tm1 = w0, dm2 = 0.0, dm1 = 1.0, em2 = 0.0, em1 = 0.0;
      for (int j = 2; j <= s; j++) {
        const double Tj = 2.0 * w0 * Tm1 - Tm2;
        const double dj = 2.0 * Tm1 + 2.0 * w0 * dm1 - dm2;
        const double ej = 4.0 * dm1 + 2.0 * w0 * em1 - em2;
        Tm2 = Tm1; Tm1 = Tj; dm2 = dm1; dm1 = dj; em2 = em1; em1 = ej;
      }
      w1 = dm1 / em1;
    }
    /* Eq. 18-21 */
    {
      /* j = 2 values: T_2 = 2 w0^2 - 1, T_2' = 4 w0, T_2'' = 4 */
      double Tm2 = 1.0, Tm1 = w0, dm2 = 0.0, dm1 = 1.0, em2 = 0.0, em1 = 0.0;
      const double T2 = 2.0 * w0 * Tm1 - Tm2, d2 = 2.0 * Tm1 + 2.0 * w0 * dm1 - dm2, e2 = 4.0 * dm1;
      const double b2 = e2 / (d2 * d2);
      double bjm2 = b2, bjm1 = b2;           /* R10: b_0 = b_1 = b_2 */
      double ajm1 = 1.0 - bjm1 * w0;         /* R9: a_1 = 1 - b_1 T_1(w0) */
      const double mut1 = bjm1 * w1;         /* Eq. 22 */
#pragma unroll
      for (int i = 0; i < NV; i++) {
        wjm2[i] = y[i];
        wjm1[i] = fma(mut1 * h, f0[i], y[i]); /* Eq. 19 */
      }
      for (int j = 2; j <= s; j++) {
        double Tj, dj, ej;
        if (j == 2) { Tj = T2; dj = d2; ej = e2; }
        else {
          Tj = 2.0 * w0 * Tm1 - Tm2;
          dj = 2.0 * Tm1 + 2.0 * w0 * dm1 - dm2;
          ej = 4.0 * dm1 + 2.0 * w0 * em1 - em2;
        }
        const double bj = ej / (dj * dj);                 /* Eq. 24 */
        const double mu = 2.0 * bj * w0 / bjm1;           /* Eq. 23 */
        const double nu = -bj / bjm2;
        const double mut = 2.0 * bj * w1 / bjm1;
        const double gamt = -ajm1 * mut;
        sys.rhs(wjm1, fj);
        const double c0 = 1.0 - mu - nu, mh = mut * h, gh = gamt * h;
#pragma unroll
        for (int i = 0; i < NV; i++) {                    /* Eq. 20 */
          const double wj = fma(gh, f0[i], fma(mh, fj[i], fma(nu, wjm2[i], fma(mu, wjm1[i], c0 * y[i]))));
          wjm2[i] = wjm1[i];
          wjm1[i] = wj;
        }
        ajm1 = 1.0 - bj * Tj;
        bjm2 = bjm1; bjm1 = bj;
        Tm2 = Tm1; Tm1 = Tj; dm2 = dm1; dm1 = dj; em2 = em1; em1 = ej;
      }
    }
    sys.rhs(wjm1, fj); /* f(y_{n+1}) */
    /* Eq. 30-32 */
    double acc = 0.0;
#pragma unroll
    for (int i = 0; i < NV; i++) {
      if (sys.valid(i)) {
        const double del = fma(0.8, y[i] - wjm1[i], 0.4 * h * (f0[i] + fj[i]));
        const double wt = fma(rtol, fmax(fabs(y[i]), fabs(wjm1[i])), atol);
        const double q = del / wt;
        acc = fma(q, q, acc);
      }
    }
    const double err = sqrt(sys.gsum(acc) / nd);
    if (err <= 1.0) { /* accept */
      nacc++;
      double fac;
      if (err > 0.0) {
        const double e3 = cbrt(err);
        if (have_prev) fac = 0.8 * (cbrt(err_old) / e3) * (h / h_old) * (1.0 / e3); /* Eq. 34, R13 */
        else fac = 0.8 / e3;
      } else fac = 10.0; /* R26 */
      fac = fmin(10.0, fmax(0.1, fac)); /* Eq. 33 */
#pragma unroll
      for (int i = 0; i < NV; i++) {
        y[i] = wjm1[i];
        f0[i] = fj[i];
      }
      err_old = err;
      h_old = h;
      have_prev = true;
      sigma_fresh = false;
      if (++since_sigma >= 25) need_sigma = true;
      if (last) break;
      t += h;
      h *= fac;
    } else { /* reject: Eq. 35 */
      nrej++;
      double fac;
      if (isfinite(err)) fac = fmin(10.0, fmax(0.1, 0.8 / cbrt(err)));
      else {
        fac = 0.1;
        saw_nonfinite = true;
      }
      h *= fac;
      have_prev = false;
      if (!sigma_fresh) need_sigma = true; /* R16 */
      const double tmax = fmax(fabs(t), fabs(t1));
      if (!(h > 10.0 * CKB_U * tmax)) {
        status = saw_nonfinite ? ST_NONFINITE : ST_UNDERFLOW;
        break;
      }
    }
  }
  if (status == ST_OK && flag) status = flag;
  st[0] = sys.nfe;
  st[1] = nacc;
  st[2] = nrej;
  st[3] = smax_used;
  return status;
}

/* ------------------------------------------------------------------------------------------------
 * Kernels.  Block = CKB_BLOCK threads; a warp holds G = 32/L systems.
 * Shared memory per warp: (K+1 + NTB+1 + NS) * G doubles.
 * ---------------------------------------------------------------------------------------------- */
#define CKB_BLOCK 128

template <class S>
__device__ __forceinline__ bool sys_setup(S &sys, const DevMech &m, double *smem, long long N, long long &ode) {
  constexpr int L = S::L, G = S::G;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int grp = lane / L;
  sys.g = lane % L;
  sys.src0 = grp * L;
  sys.mask = (L == 32) ? 0xffffffffu : (((1u << L) - 1u) << (grp * L));
  ode = ((long long)blockIdx.x * (CKB_BLOCK / 32) + warp) * G + grp;
  const int per_warp = (m.K + 1 + m.NTB + 1 + m.NS) * G;
  double *base = smem + (size_t)warp * per_warp + grp;
  sys.sC = base;
  sys.sM = base + (m.K + 1) * G;
  sys.sQ = base + (m.K + 1 + m.NTB + 1) * G;
  sys.nfe = 0;
  if (ode >= N) return false;
  if (sys.g == 0) {
    sys.sC[m.K * G] = 1.0;   /* "absent molecule" concentration */
    sys.sM[m.NTB * G] = 1.0; /* "no third body" */
  }
  sys.gsync();
  return true;
}

template <int L, int NV, class TAB, int METHOD>
__global__ void __launch_bounds__(CKB_BLOCK)
integrate_kernel(const __grid_constant__ DevMech m, const __grid_constant__ TAB tab, double *__restrict__ states, const double *__restrict__ pressure,
                 double p_uniform, long long N, long long ld, double t0, double dt, double rtol, double atol,
                 int *__restrict__ status, int *__restrict__ stats) {
  extern __shared__ double smem[];
  Sys<L, NV, TAB> sys(m, tab);
  long long ode;
  if (!sys_setup(sys, m, smem, N, ode)) return;
  sys.p = pressure ? pressure[ode] : p_uniform;
  double y[NV];
#pragma unroll
  for (int i = 0; i < NV; i++) {
    const int c = sys.g + L * i;
    y[i] = (c < m.n) ? states[(size_t)c * ld + ode] : 0.0;
  }
  int st[4];
  int code;
  if (METHOD == 0) code = rkck_driver(sys, y, t0, t0 + dt, rtol, atol, st);
  else code = rkc_driver(sys, y, t0, t0 + dt, rtol, atol, st);
#pragma unroll
  for (int i = 0; i < NV; i++) {
    const int c = sys.g + L * i;
    if (c < m.n) states[(size_t)c * ld + ode] = y[i];
  }
  if (sys.g == 0) {
    if (status) status[ode] = code;
    if (stats) {
#pragma unroll
      for (int q = 0; q < 4; q++) stats[(size_t)q * N + ode] = st[q];
    }
  }
}

template <int L, int NV, class TAB>
__global__ void __launch_bounds__(CKB_BLOCK)
rhs_kernel(const __grid_constant__ DevMech m, const __grid_constant__ TAB tab, const double *__restrict__ states, const double *__restrict__ pressure,
           double p_uniform, long long N, long long ld, double *__restrict__ dydt, int repeat) {
  extern __shared__ double smem[];
  Sys<L, NV, TAB> sys(m, tab);
  long long ode;
  if (!sys_setup(sys, m, smem, N, ode)) return;
  sys.p = pressure ? pressure[ode] : p_uniform;
  double y[NV], f[NV];
#pragma unroll
  for (int i = 0; i < NV; i++) {
    const int c = sys.g + L * i;
    y[i] = (c < m.n) ? states[(size_t)c * ld + ode] : 0.0;
  }
  for (int r = 0; r < repeat; r++) {
    sys.rhs(y, f);
    if (r + 1 < repeat) {
      /* keep the repeats from being folded: feed a zero-weight dependence on f back into y */
#pragma unroll
      for (int i = 0; i < NV; i++) y[i] = fma(f[i], 0.0, y[i]);
    }
  }
#pragma unroll
  for (int i = 0; i < NV; i++) {
    const int c = sys.g + L * i;
    if (c < m.n) dydt[(size_t)c * ld + ode] = f[i];
  }
}

} /* namespace ckb */
