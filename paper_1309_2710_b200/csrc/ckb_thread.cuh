/*
 * ckb_thread.cuh -- thread-per-ODE (the paper's mapping) for mechanisms with MORE than 16 unknowns:
 * table-driven source term, stage vectors in a global-memory workspace (as the paper's kernels kept them, P:255:
 * "global memory"; here the workspace of a resident grid fits the 126 MB L2), concentrations and production
 * rates in shared memory.  DESIGN.md 6.8.
 *
 * Why it exists beside the warp-per-ODE kernels (ckb_device.cuh): with one system per LANE every table word,
 * every index and every loop counter of f(y) is warp-uniform.  The reaction-slot stream is read through the
 * constant bank (kernel parameter) or as broadcast loads, indices are decoded once per warp instead of once per
 * lane, Eq. 3 is a scatter into the lane's own accumulators (no gather schedule, no padding), and the once-per-
 * evaluation work (log, divisions, reductions -> plain sums) is amortised over 32 systems.  Per evaluation of f(y) a
 * warp issues ~1/3 of the instructions of the lane-distributed mapping.
 *
 * Data layout per warp in shared memory (doubles, element e of lane l at [e*32 + l]: conflict free):
 *   C[0..n)   C[1+k] = concentration of species k (C[0] unused)
 *   F[0..n)   during f(y): F[1+k] accumulates omega_k (Eq. 3);  afterwards F[c] = f_c(y), F[0] = dT/dt
 * Stage vectors: ws[(v*n + c)*NT + gtid], v = physical vector, c = component, NT = threads of the grid.
 *
 * Source term: Eq. 2-6; integrators: the same controller logic, constant for constant, as Rkck / Rkc in
 * ckb_device.cuh (readings R1-R31) with the vectors in memory instead of registers.
 */
#pragma once
#include "ckb_device.cuh"

namespace ckbt {

using ckb::ExpConst;
using ckb::ckb_exp;

/* all shared-memory accesses go through this symbol with 32-bit byte offsets, so that they compile to LDS / STS (a
 * pointer kept in a struct degrades to generic loads with 64-bit address arithmetic) */
extern __shared__ double ckbt_smem[];

#ifndef CKBT_LOCKSTEP
#define CKBT_LOCKSTEP 1 /* the warps of a block enter f(y) together (one instruction stream per SM) */
#endif
#ifndef CKBT_U
#define CKBT_U 3    /* reaction slots per trip of a class loop (2U exponential chains in lock step) */
#endif
#ifndef CKBT_U_TB
#define CKBT_U_TB 2 /* the same for the classes with a third body */
#endif

/* R31: blending factor of a fall-off reaction from its [M] (same arithmetic as ckb_device.cuh); a free function that
 * takes scalars only: nothing of the caller's state escapes into memory */
static __device__ __noinline__ double falloff_factor(const unsigned long long *__restrict__ aux, double Mc, int fb,
                                                     double T, double invT, double lnT) {
  const ExpConst<false> fec;
  auto ad = [&](int i) { return __longlong_as_double((long long)__ldg(aux + i)); };
  const int kind = (int)ad(fb);
  const double Pr = Mc * ckb_exp(fma(-ad(fb + 3), invT, fma(ad(fb + 2), lnT, ad(fb + 1))), fec);
  double B = Pr / (1.0 + Pr);
  if (kind >= 2) { /* Troe */
    const double a = ad(fb + 4);
    double Fc = (1.0 - a) * ckb_exp(-T * ad(fb + 5), fec) + a * ckb_exp(-T * ad(fb + 6), fec);
    if (kind == 2) Fc += ckb_exp(-ad(fb + 7) * invT, fec);
    const double lF = log10(Fc), lP = log10(Pr);
    const double c = -0.4 - 0.67 * lF, nn = 0.75 - 1.27 * lF;
    const double x = (lP + c) / (nn - 0.14 * (lP + c));
    B *= exp(2.302585092994046 * (lF / (1.0 + x * x)));
  }
  return B;
}

template <class STAB, int CV_>
struct TSys {
  static constexpr bool CV = CV_ != 0;
  const DevThread &m;
  const STAB &st;
  const unsigned long long *__restrict__ aux;
  unsigned cC, cF;   /* byte offsets in ckbt_smem of this lane's column of the warp's C and F regions */
  double *__restrict__ ws; /* this thread's column of the workspace */
  size_t NT;
  double pR, Rp;
  int n;

  __device__ __forceinline__ TSys(const DevThread &m_, const STAB &st_, const unsigned long long *aux_)
      : m(m_), st(st_), aux(aux_) {}
  __device__ __forceinline__ double ad(int i) const { return __longlong_as_double((long long)__ldg(aux + i)); }
  __device__ __forceinline__ unsigned long long aw(int i) const { return __ldg(aux + i); }
  __device__ __forceinline__ double sd(int i) const { return __longlong_as_double((long long)st.ld(i)); }
  __device__ __forceinline__ double td(int i) const { return ad(i); } /* RKC coefficient table (Rkc::take_step idiom) */
  __device__ __forceinline__ void set_pressure(double p) {
    if (CV) { pR = p; Rp = 1.0 / p; } else { pR = p / CKB_RU; Rp = CKB_RU / p; }
  }
  /* stage-vector accesses go to L2 directly (ld/st.global.cg): they have no reuse in L1, and the few KB of L1 that the
   * shared regions leave stay with the species / coefficient tables */
  /* a load the compiler keeps where it is written (it would otherwise sink every load of a batch down to its first use
   * and run the batch at one memory latency per component) */
  __device__ __forceinline__ static double ld_pinned(const double *p) {
    double x;
    asm volatile("ld.global.cg.f64 %0, [%1];" : "=d"(x) : "l"(p) : "memory");
    return x;
  }
  struct VRef {
    double *p;
    __device__ __forceinline__ operator double() const { return __ldcg(p); }
    __device__ __forceinline__ double pinned() const { return ld_pinned(p); }
    __device__ __forceinline__ void operator=(double x) const { __stcg(p, x); }
    __device__ __forceinline__ void operator*=(double x) const { __stcg(p, __ldcg(p) * x); }
  };
  __device__ __forceinline__ VRef V(int vec, int c) const { return VRef{ws + ((size_t)vec * n + c) * NT}; }
  __device__ __forceinline__ static double &sm(unsigned byte_off) {
    return *reinterpret_cast<double *>(reinterpret_cast<char *>(ckbt_smem) + byte_off);
  }
  __device__ __forceinline__ double &C(unsigned off) const { return sm(cC + off); }   /* off = component * 256 */
  __device__ __forceinline__ double &Fo(unsigned off) const { return sm(cF + off); }
  __device__ __forceinline__ double &F(int c) const { return sm(cF + (unsigned)c * 256u); }

  /* One pass over the components: body(i, x, f) with x[q] = component i of vector vin[q] and f = F(i).  The inputs of
   * CKBT_VB components are loaded before the first store of the batch. */
  template <int NIN, class Body>
  __device__ __forceinline__ void vloop(const int (&vin)[NIN], Body body) const {
    for (int i0 = 0; i0 < n; i0 += CKBT_VB) {
      double x[CKBT_VB][NIN];
#pragma unroll
      for (int u = 0; u < CKBT_VB; u++) {
        const int i = min(i0 + u, n - 1);
#pragma unroll
        for (int q = 0; q < NIN; q++) x[u][q] = V(vin[q], i).pinned();
      }
#pragma unroll
      for (int u = 0; u < CKBT_VB; u++)
        if (i0 + u < n) body(i0 + u, x[u], F(i0 + u));
    }
  }

  /* R22: [M]_t = C_tot + sum_listed (alpha - 1) C, evaluated where it is used; R31: replaced by the blending factor */
  __device__ __forceinline__ double third_body(int t, double ctot, double T, double invT, double lnT) const {
    const unsigned long long d0 = aw(m.o_set + 2 * t), d1 = aw(m.o_set + 2 * t + 1);
    int b = (int)d0;
    const int cnt = (int)(unsigned)d1, fb = (int)(d1 >> 32);
    double Mc = ctot;
    for (int e = 0; e < cnt; e++, b += 2) Mc = fma(ad(b), C((unsigned)aw(b + 1)), Mc);
    if (m.has_fo && fb) Mc = falloff_factor(aux, Mc, fb, T, invT, lnT);
    return Mc;
  }

  /* One class of regular slots: NA reactant molecules, NB product molecules, TB third body.  U slots per trip: their 2U
   * exponentials are advanced in lock step (2U independent dependency chains: a warp alone keeps the FP64 pipe fed), the
   * table words of the NEXT trip are fetched at the top of this one (an indexed constant-bank load takes ~90 cycles),
   * and Eq. 3 of the PREVIOUS trip's slots is applied while this trip's chains are in flight (slot by slot: two slots of
   * a trip may share a species).  Trips past the end of the class re-read its last slot and contribute q = 0. */
  template <int NA, int NB, int TB, int U>
  __device__ __forceinline__ void slot_loop(int base, int count, double ctot, double T, double invT, double lnT) const {
    const ExpConst<false> ec;
    const int last = base + (count - 1) * CKBT_SLOT_WORDS;
    unsigned long long w[U][CKBT_SLOT_WORDS];
#pragma unroll
    for (int u = 0; u < U; u++) {
      const int bs = min(base + u * CKBT_SLOT_WORDS, last);
#pragma unroll
      for (int x = 0; x < CKBT_SLOT_WORDS; x++) w[u][x] = st.ld(bs + x);
    }
    double qp[U];
    unsigned pa[U][3], pb[U][3]; /* offsets of the previous trip's slots; the first trip adds 0 to F[0] */
#pragma unroll
    for (int u = 0; u < U; u++) {
      qp[u] = 0.0;
#pragma unroll
      for (int q = 0; q < 3; q++) pa[u][q] = pb[u][q] = 0;
    }
    for (int r = 0; r < count; r += U) {
      /* this trip's words are in w; fetch the next trip's */
      unsigned long long wn[U][CKBT_SLOT_WORDS];
#pragma unroll
      for (int u = 0; u < U; u++) {
        const int bs = min(base + (r + U + u) * CKBT_SLOT_WORDS, last);
#pragma unroll
        for (int x = 0; x < CKBT_SLOT_WORDS; x++) wn[u][x] = st.ld(bs + x);
      }
      unsigned a[U][3], b[U][3];
      double pf[U], pr[U], xs[2 * U], ks[2 * U];
#pragma unroll
      for (int u = 0; u < U; u++) {
#pragma unroll
        for (int q = 0; q < 3; q++) {
          a[u][q] = (unsigned)(w[u][CKB_SL_IDXA] >> (16 * q)) & 0xFFFFu;
          b[u][q] = (unsigned)(w[u][CKB_SL_IDXB] >> (16 * q)) & 0xFFFFu;
        }
        pf[u] = C(a[u][0]);
        pr[u] = C(b[u][0]);
#pragma unroll
        for (int q = 1; q < NA; q++) pf[u] *= C(a[u][q]);
#pragma unroll
        for (int q = 1; q < NB; q++) pr[u] *= C(b[u][q]);
#define CKBT_WD(x) __longlong_as_double((long long)w[u][x])
        xs[2 * u] = fma(-CKBT_WD(CKB_SL_THF), invT, fma(CKBT_WD(CKB_SL_BF), lnT, CKBT_WD(CKB_SL_LNAF)));
        xs[2 * u + 1] = fma(-CKBT_WD(CKB_SL_THR), invT, fma(CKBT_WD(CKB_SL_BR), lnT, CKBT_WD(CKB_SL_LNAR)));
#undef CKBT_WD
      }
      double Mt[U];
#pragma unroll
      for (int u = 0; u < U; u++) Mt[u] = TB ? third_body((int)(w[u][CKB_SL_IDXA] >> 48), ctot, T, invT, lnT) : 1.0;
      ckb::ckb_exp_n<2 * U>(xs, ks, ec);
      /* Eq. 3 of the previous trip */
#pragma unroll
      for (int u = 0; u < U; u++) {
        double oa[3], ob[3];
#pragma unroll
        for (int q = 0; q < NA; q++) oa[q] = Fo(pa[u][q]);
#pragma unroll
        for (int q = 0; q < NB; q++) ob[q] = Fo(pb[u][q]);
#pragma unroll
        for (int q = 0; q < NA; q++) Fo(pa[u][q]) = oa[q] - qp[u];
#pragma unroll
        for (int q = 0; q < NB; q++) Fo(pb[u][q]) = ob[q] + qp[u];
      }
#pragma unroll
      for (int u = 0; u < U; u++) {
        double q = fma(ks[2 * u], pf[u], -(ks[2 * u + 1] * pr[u])); /* Eq. 4-5, net rate of the pair */
        if (TB) q *= Mt[u];
        qp[u] = (r + u < count) ? q : 0.0;
#pragma unroll
        for (int x = 0; x < 3; x++) { pa[u][x] = a[u][x]; pb[u][x] = b[u][x]; }
#pragma unroll
        for (int x = 0; x < CKBT_SLOT_WORDS; x++) w[u][x] = wn[u][x];
      }
    }
#pragma unroll
    for (int u = 0; u < U; u++) {
#pragma unroll
      for (int q = 0; q < NA; q++) Fo(pa[u][q]) -= qp[u];
#pragma unroll
      for (int q = 0; q < NB; q++) Fo(pb[u][q]) += qp[u];
    }
  }

  /* slots with a repeated species: molecule counts and an explicit net-coefficient list (rare) */
  __device__ __forceinline__ void irregular_loop(int base, int count, double ctot, double T, double invT, double lnT) const {
    const ExpConst<false> ec;
    for (int r = 0; r < count; r++, base += CKBT_IRR_WORDS) {
      const unsigned long long wa = st.ld(base + CKB_SL_IDXA), wb = st.ld(base + CKB_SL_IDXB);
      const unsigned fl = (unsigned)(wb >> 48);
      const int na = fl & 3, nb = (fl >> 2) & 3;
      double pf = 1.0, pr = 1.0;
      for (int q = 0; q < na; q++) pf *= C((unsigned)(wa >> (16 * q)) & 0xFFFFu);
      for (int q = 0; q < nb; q++) pr *= C((unsigned)(wb >> (16 * q)) & 0xFFFFu);
      const double xf = fma(-sd(base + CKB_SL_THF), invT, fma(sd(base + CKB_SL_BF), lnT, sd(base + CKB_SL_LNAF)));
      const double xr = fma(-sd(base + CKB_SL_THR), invT, fma(sd(base + CKB_SL_BR), lnT, sd(base + CKB_SL_LNAR)));
      double q = fma(ckb_exp(xf, ec), pf, -(ckb_exp(xr, ec) * pr));
      if (fl & 16) q *= third_body((int)(wa >> 48), ctot, T, invT, lnT);
      for (int w = 0; w < 4; w++) {
        const unsigned long long e2 = st.ld(base + 8 + w);
#pragma unroll
        for (int h = 0; h < 2; h++) {
          const unsigned e = (unsigned)(e2 >> (32 * h));
          const int coef = (int)e >> 16; /* arithmetic shift: signed */
          if (coef != 0) Fo(e & 0xFFFFu) = fma((double)coef, q, Fo(e & 0xFFFFu));
        }
      }
    }
  }

  /* f(y) of the vector stored at physical slot `vec`; on return F[c] = f_c */
  __device__ __forceinline__ void rhs(int vec) const {
    const int K = m.K;
    const double T = V(vec, 0);
    const double invT = 1.0 / T, lnT = log(T);
    double s1 = 0.0, s2 = 0.0;
    /* R8a: cp_k/R = a1 + a2 T + .. + a5 T^4;  R30: the high range where T > T_mid (per lane: a select of the row) */
    for (int k0 = 0; k0 < K; k0 += CKBT_VB) {
      double Yb[CKBT_VB];
#pragma unroll
      for (int u = 0; u < CKBT_VB; u++) Yb[u] = V(vec, 1 + min(k0 + u, K - 1)).pinned();
#pragma unroll
      for (int u = 0; u < CKBT_VB; u++) {
      const int k = min(k0 + u, K - 1); /* past the end: the last species again, contributing nothing */
      const bool live = k0 + u < K;
      const int b = m.o_sp + k * CKB_SP_WORDS;
      int bt = b;
      if (m.o_sp2) {
        const int b2 = m.o_sp2 + k * CKB_SP_WORDS;
        if (T > ad(b2 + CKB_SP_INVW)) bt = b2;
      }
      double cp = ad(bt + CKB_SP_CP + 4);
#pragma unroll
      for (int q = 3; q >= 0; q--) cp = fma(cp, T, ad(bt + CKB_SP_CP + q));
      const double v = live ? Yb[u] * ad(b + CKB_SP_INVW) : 0.0; /* Y_k / W_k */
      if (live) C((1 + k) * 256u) = v;
      s1 += v;
      s2 = fma(v, cp, s2);
      }
    }
    /* R9a: rho = p / (Ru T sum_k Y_k/W_k), C_k = rho Y_k / W_k;  R29: rho given, C_tot = rho sum_k Y_k/W_k */
    const double ctot = CV ? pR * s1 : pR * invT;
    const double rho = CV ? pR : ctot * (1.0 / s1);
    const double invrho = CV ? Rp : s1 * T * Rp;
#pragma unroll 4
    for (int k = 1; k <= K; k++) {
      C(k * 256u) *= rho;
      F(k) = 0.0;
    }
    F(0) = 0.0;
    /* Eq. 3-5, class by class (every lane runs the same class loop on its own system) */
    for (int c = 0; c < m.ncls; c++) {
      const unsigned long long d0 = st.ld(m.o_cls + 2 * c);
      const int kind = (int)(unsigned)d0, count = (int)(d0 >> 32), base = (int)st.ld(m.o_cls + 2 * c + 1);
      switch (kind) {
#define CKBT_CASE(NA, NB, TB) \
  case ((NA - 1) * 6 + (NB - 1) * 2 + TB): slot_loop<NA, NB, TB, (TB ? CKBT_U_TB : CKBT_U)>(base, count, ctot, T, invT, lnT); break;
        CKBT_CASE(1, 1, 0) CKBT_CASE(1, 1, 1) CKBT_CASE(1, 2, 0) CKBT_CASE(1, 2, 1) CKBT_CASE(1, 3, 0) CKBT_CASE(1, 3, 1)
        CKBT_CASE(2, 1, 0) CKBT_CASE(2, 1, 1) CKBT_CASE(2, 2, 0) CKBT_CASE(2, 2, 1) CKBT_CASE(2, 3, 0) CKBT_CASE(2, 3, 1)
        CKBT_CASE(3, 1, 0) CKBT_CASE(3, 1, 1) CKBT_CASE(3, 2, 0) CKBT_CASE(3, 2, 1) CKBT_CASE(3, 3, 0) CKBT_CASE(3, 3, 1)
#undef CKBT_CASE
        default: irregular_loop(base, count, ctot, T, invT, lnT); break;
      }
    }
    /* Eq. 2: dY_k/dt = W_k omega_k / rho;  Eq. 6 / R29: dT/dt from sum_k (h_k/RT [- 1]) omega_k */
    double s3 = 0.0;
#pragma unroll 6
    for (int k = 0; k < K; k++) {
      const int b = m.o_sp + k * CKB_SP_WORDS;
      int bt = b;
      if (m.o_sp2) {
        const int b2 = m.o_sp2 + k * CKB_SP_WORDS;
        if (T > ad(b2 + CKB_SP_INVW)) bt = b2;
      }
      double h = ad(bt + CKB_SP_H + 4);
#pragma unroll
      for (int q = 3; q >= 0; q--) h = fma(h, T, ad(bt + CKB_SP_H + q));
      h = fma(ad(bt + CKB_SP_H + 5), invT, h);
      if (CV) h -= 1.0;
      const double om = F(1 + k);
      s3 = fma(h, om, s3);
      F(1 + k) = ad(b + CKB_SP_W) * om * invrho;
    }
    F(0) = -(T * s3 * invrho) / (CV ? s2 - s1 : s2);
  }
};

/* ================================================================================================
 * Integrators with memory-resident vectors.  Same state machines, same decisions, same constants as ckb::Rkck /
 * ckb::Rkc (one call site of f(y) per loop trip); norms are plain sums over the components (the
 * oracle's order).  The argument of the next f(y) is the vector at physical slot arg().
 * Every pass over the components goes through TSys::vloop: the inputs of CKBT_VB components are loaded before the
 * first store of the batch, so that a thread has CKBT_VB x (number of input vectors) loads in flight (the stores of a
 * batch may alias the loads of the next one as far as the compiler can tell, so a plain loop runs at one memory
 * latency per component).
 * ============================================================================================== */
template <class S>
struct RkckMem {
  typedef ckb::Rkck<ckb::Sys<1, 1, ckb::ParamTab>> Tab; /* Table 1 constants (R1) */
  enum { Y = 0, K1 = 1, K2 = 2, K3 = 3, K4 = 4, K5 = 5, W = 6 };
  double t, h, t1, rtol, atol;
  int stage, nfe, nacc, nrej, attempts, status, iy, iw;
  bool last, saw_nonfinite;

  __device__ __forceinline__ int arg() const { return iw; }
  __device__ __forceinline__ int yvec() const { return iy; }

  __device__ __forceinline__ void begin_attempt(const S &sys, bool have_k1) {
    last = false;
    double r = 1.0;
    if (1.1 * h >= t1 - t) { /* R5 */
      const double hn = t1 - t;
      if (have_k1) r = hn / h;
      h = hn;
      last = true;
    }
    if (!have_k1) {
      stage = 1;
      const int out = iw;
      sys.template vloop<1>({iy}, [&](int i, const double(&x)[1], double) { sys.V(out, i) = x[0]; });
    } else {
      start_stages(sys, r);
    }
  }
  /* k1 <- r k1 (R5 clip / R25 rescale; r = 1: untouched) and the argument of stage 2 */
  __device__ __forceinline__ void start_stages(const S &sys, double r) {
    if (++attempts > 1000000) { /* R7 */
      status = ST_MAXSTEPS;
      stage = 0;
      return;
    }
    stage = 2;
    const int out = iw;
    const bool scale = r != 1.0;
    sys.template vloop<2>({K1, iy}, [&](int i, const double(&x)[2], double) {
      double k1 = x[0];
      if (scale) {
        k1 *= r;
        sys.V(K1, i) = k1;
      }
      sys.V(out, i) = fma(Tab::B21, k1, x[1]);
    });
  }
  /* the initial state has been stored at physical slot 0 */
  __device__ __forceinline__ void start(const S &sys, double t0_, double t1_, double rtol_, double atol_) {
    iy = Y; iw = W;
    t = t0_; t1 = t1_; rtol = rtol_; atol = atol_;
    h = t1_ - t0_; /* R4 */
    nfe = nacc = nrej = attempts = 0;
    status = ST_OK;
    saw_nonfinite = false;
    begin_attempt(sys, false);
  }

  __device__ __forceinline__ bool advance(const S &sys) {
    nfe++;
    const int out = iw;
    const double hh = h;
    switch (stage) {
      case 1: { /* Eq. 7, then the argument of stage 2 */
        if (++attempts > 1000000) { /* R7 */
          status = ST_MAXSTEPS;
          stage = 0;
          return true;
        }
        sys.template vloop<1>({iy}, [&](int i, const double(&x)[1], double f) {
          const double k1 = hh * f;
          sys.V(K1, i) = k1;
          sys.V(out, i) = fma(Tab::B21, k1, x[0]);
        });
        stage = 2;
        return false;
      }
      case 2:
        sys.template vloop<2>({K1, iy}, [&](int i, const double(&x)[2], double f) {
          const double k2 = hh * f;
          sys.V(K2, i) = k2;
          sys.V(out, i) = fma(Tab::B32, k2, fma(Tab::B31, x[0], x[1]));
        });
        stage = 3;
        return false;
      case 3:
        sys.template vloop<3>({K1, K2, iy}, [&](int i, const double(&x)[3], double f) {
          const double k3 = hh * f;
          sys.V(K3, i) = k3;
          sys.V(out, i) = fma(Tab::B43, k3, fma(Tab::B42, x[1], fma(Tab::B41, x[0], x[2])));
        });
        stage = 4;
        return false;
      case 4:
        sys.template vloop<4>({K1, K2, K3, iy}, [&](int i, const double(&x)[4], double f) {
          const double k4 = hh * f;
          sys.V(K4, i) = k4;
          sys.V(out, i) = fma(Tab::B54, k4, fma(Tab::B53, x[2], fma(Tab::B52, x[1], fma(Tab::B51, x[0], x[3]))));
        });
        stage = 5;
        return false;
      case 5:
        sys.template vloop<5>({K1, K2, K3, K4, iy}, [&](int i, const double(&x)[5], double f) {
          const double k5 = hh * f;
          sys.V(K5, i) = k5;
          sys.V(out, i) = fma(Tab::B65, k5, fma(Tab::B64, x[3], fma(Tab::B63, x[2], fma(Tab::B62, x[1], fma(Tab::B61, x[0], x[4])))));
        });
        stage = 6;
        return false;
      default:
        break;
    }
    /* stage 6: Eq. 13, 15, 16 (R2), 17 (R3) */
    double errmax = 0.0;
    const double rt = rtol, at = atol;
    sys.template vloop<5>({K1, K3, K4, K5, iy}, [&](int i, const double(&x)[5], double f) {
      const double k6 = hh * f;
      const double k1 = x[0], k3 = x[1], k4 = x[2], k5 = x[3], yi = x[4];
      const double yn = fma(Tab::C6, k6, fma(Tab::C4, k4, fma(Tab::C3, k3, fma(Tab::C1, k1, yi))));
      const double dl = fma(Tab::D6, k6, fma(Tab::D5, k5, fma(Tab::D4, k4, fma(Tab::D3, k3, Tab::D1 * k1))));
      sys.V(out, i) = yn;
      const double d0 = fma(rt, fabs(yi) + fabs(k1), at);
      double e = fabs(dl) / d0;
      if (!isfinite(yn) || isnan(e)) e = __longlong_as_double(0x7ff0000000000000LL);
      errmax = fmax(errmax, e);
    });
    if (errmax <= 1.0) { /* P:139 accept: y <- w by exchanging the two physical vectors */
      nacc++;
      const int o = iy; iy = iw; iw = o;
      if (last) return true;
      t += h;
      double fac = (errmax > 0.0) ? Tab::SAFETY * pow(errmax, -0.2) : 5.0;
      if (fac > 5.0) fac = 5.0;
      h *= fac;
      begin_attempt(sys, false);
      return false;
    }
    nrej++;
    double fac;
    if (isfinite(errmax)) {
      fac = Tab::SAFETY * pow(errmax, -0.25);
      if (fac < 0.1) fac = 0.1;
    } else {
      fac = 0.1;
      saw_nonfinite = true;
    }
    h *= fac;
    const double tmax = fmax(fabs(t), fabs(t1));
    if (!(h > 10.0 * CKB_U * tmax)) { /* R6 */
      status = saw_nonfinite ? ST_NONFINITE : ST_UNDERFLOW;
      return true;
    }
    /* R25: k1 rescaled, not re-evaluated; then R5.  Two scalings in the register-resident kernels (k1 *= fac, then
     * k1 *= hn/h at a clip) are two roundings there and here */
    last = false;
    double r2 = 1.0;
    if (1.1 * h >= t1 - t) {
      const double hn = t1 - t;
      r2 = hn / h;
      h = hn;
      last = true;
    }
    if (++attempts > 1000000) {
      status = ST_MAXSTEPS;
      stage = 0;
      return true;
    }
    stage = 2;
    const bool clip = last;
    sys.template vloop<2>({K1, iy}, [&](int i, const double(&x)[2], double) {
      double k1 = x[0] * fac;
      if (clip) k1 *= r2;
      sys.V(K1, i) = k1;
      sys.V(out, i) = fma(Tab::B21, k1, x[1]);
    });
    return false;
  }
  __device__ __forceinline__ int phase() const { return stage; }
  __device__ __forceinline__ void result(int (&st)[4]) const { st[0] = nfe; st[1] = nacc; st[2] = nrej; st[3] = 0; }
};

template <class S>
struct RkcMem {
  enum { S_F0 = 1, S_PM = 2, S_H0 = 3, S_STAGE = 4, S_FINAL = 5 };
  double t, h, t1, Dt, rtol, atol, nd;
  double sigma, err_old, h_old, pm_d, pm_sigma;
  int state, j, s, s_max, pm_it, cbase;
  int nfe, nacc, nrej, smax_used, attempts, since_sigma, status, flag;
  int iy, if0, iv, iw, iwm2; /* physical vectors of y, f0, v, w (= w_{j-1}), w_{j-2} (may be y itself) */
  bool last, have_prev, saw_nonfinite, sigma_fresh, need_sigma, pm_initial;

  __device__ __forceinline__ int arg() const { return iw; }
  __device__ __forceinline__ int yvec() const { return iy; }
  __device__ __forceinline__ int free_vec() const {
    const unsigned used = (1u << iy) | (1u << if0) | (1u << iv) | (1u << iw) | (1u << iwm2);
    return __ffs((int)(~used & ((1u << CKBT_VECS) - 1u))) - 1;
  }

  __device__ __forceinline__ void start(const S &sys, double t0_, double t1_, double rtol_, double atol_) {
    iy = 0; iw = 1; if0 = 2; iv = 3; iwm2 = 0;
    sys.template vloop<1>({0}, [&](int i, const double(&x)[1], double) { sys.V(1, i) = x[0]; });
    t = t0_; t1 = t1_; Dt = t1_ - t0_; rtol = rtol_; atol = atol_; nd = (double)sys.n;
    s_max = (int)floor(sqrt(rtol_ / (10.0 * CKB_U)) + 0.5); /* R12 */
    if (s_max < 2) s_max = 2;
    nfe = nacc = nrej = smax_used = attempts = since_sigma = 0;
    status = ST_OK; flag = 0;
    have_prev = saw_nonfinite = need_sigma = false;
    sigma_fresh = true;
    err_old = h_old = 0.0;
    state = S_F0;
  }

  /* power method set-up (R17 step 2): z at distance d from y along v; copy_f0 = first call, v <- f0 <- F */
  __device__ __forceinline__ void pm_begin(const S &sys, bool copy_f0, bool initial) {
    double a = 0.0, b = 0.0;
    const int of0 = if0, ov = iv, out = iw;
    if (copy_f0) {
      sys.template vloop<1>({iy}, [&](int i, const double(&x)[1], double f) {
        sys.V(of0, i) = f;
        sys.V(ov, i) = f;
        a = fma(x[0], x[0], a);
        b = fma(f, f, b);
      });
    } else {
      sys.template vloop<2>({iy, iv}, [&](int i, const double(&x)[2], double) {
        a = fma(x[0], x[0], a);
        b = fma(x[1], x[1], b);
      });
    }
    const double ynrm = sqrt(a), vnrm = sqrt(b);
    if (ynrm != 0.0 && vnrm != 0.0) {
      pm_d = ynrm * CKB_SQRTU;
      const double r = pm_d / vnrm;
      sys.template vloop<2>({iy, iv}, [&](int i, const double(&x)[2], double) { sys.V(out, i) = fma(x[1], r, x[0]); });
    } else if (ynrm != 0.0) {
      pm_d = ynrm * CKB_SQRTU;
      sys.template vloop<1>({iy}, [&](int i, const double(&x)[1], double) { sys.V(out, i) = x[0] * (1.0 + CKB_SQRTU); });
    } else if (vnrm != 0.0) {
      pm_d = CKB_U;
      const double r = pm_d / vnrm;
      sys.template vloop<1>({iv}, [&](int i, const double(&x)[1], double) { sys.V(out, i) = x[0] * r; });
    } else {
      pm_d = CKB_U;
      for (int i = 0; i < sys.n; i++) sys.V(out, i) = pm_d;
    }
    pm_sigma = 0.0;
    pm_it = 1;
    pm_initial = initial;
    state = S_PM;
  }

  __device__ __forceinline__ bool begin_step(const S &sys) {
    last = false;
    if (1.1 * h >= t1 - t) { /* R5 */
      h = t1 - t;
      last = true;
    }
    if (need_sigma) { /* R16 */
      pm_begin(sys, false, false);
      return false;
    }
    return take_step(sys);
  }

  /* Eq. 39 (R12), first stage Eq. 19; true = failed */
  __device__ __forceinline__ bool take_step(const S &sys) {
    s = 1 + (int)floor(sqrt(fma(1.54 * h, sigma, 1.0)));
    if (s < 2) s = 2;
    if (s > s_max) {
      s = s_max;
      h = ((double)s_max * (double)s_max - 1.0) / (1.54 * sigma);
      last = false;
    }
    if (s > smax_used) smax_used = s;
    if (++attempts > 1000000) {
      status = ST_MAXSTEPS;
      return true;
    }
    double mut1; /* Eq. 22 */
    if (s <= sys.m.s_tab) {
      mut1 = sys.td(sys.m.o_rkc + (s - 2));
      cbase = sys.m.o_rkcs + 4 * ((s - 2) * (s - 1) / 2);
    } else {
      double mu, nu, mut, gamt;
      ckb::rkc_coefficients(s, 2, mut1, mu, nu, mut, gamt);
      cbase = -1;
    }
    const double mh = mut1 * h;
    iwm2 = iy; /* w_0 = y: no copy */
    const int out = iw;
    sys.template vloop<2>({if0, iy}, [&](int i, const double(&x)[2], double) { sys.V(out, i) = fma(mh, x[0], x[1]); }); /* Eq. 19 */
    j = 2;
    state = S_STAGE;
    return false;
  }

  __device__ __forceinline__ void pm_next_z(const S &sys, double dd) {
    const int out = iw;
    if (dd != 0.0) {
      const double r = pm_d / dd;
      sys.template vloop<2>({if0, iy}, [&](int i, const double(&x)[2], double f) { sys.V(out, i) = fma(f - x[0], r, x[1]); });
    } else {
      const int ci = pm_it % sys.n;
      const double yi = sys.V(iy, ci);
      sys.V(out, ci) = yi - (sys.V(out, ci) - yi);
    }
  }

  __device__ __forceinline__ bool advance(const S &sys) {
    nfe++;
    switch (state) {
      case S_F0:
        pm_begin(sys, true, true);
        return false;
      case S_PM: { /* R17 steps 3-5 */
        double dd = 0.0;
        sys.template vloop<1>({if0}, [&](int, const double(&x)[1], double f) {
          const double e = f - x[0];
          dd = fma(e, e, dd);
        });
        dd = sqrt(dd);
        const double sigma_prev = pm_sigma;
        pm_sigma = dd / pm_d;
        const double fl = pm_sigma > 1e-300 ? pm_sigma : 1e-300;
        const bool conv = pm_it >= 2 && fabs(pm_sigma - sigma_prev) <= 0.01 * fl;
        if (!conv && pm_it < 50) {
          pm_next_z(sys, dd);
          pm_it++;
          return false;
        }
        if (!conv) {
          flag = ST_SIGMA;
          pm_next_z(sys, dd); /* R17: z is updated once more after the 50th evaluation before v is saved */
        }
        sigma = 1.2 * pm_sigma; /* R18 */
        sigma_fresh = true;
        need_sigma = false;
        since_sigma = 0;
        const int ov = iv, out = iw;
        if (!pm_initial) {
          sys.template vloop<2>({iw, iy}, [&](int i, const double(&x)[2], double) { sys.V(ov, i) = x[0] - x[1]; });
          return take_step(sys);
        }
        h_old = (sigma > 0.0 && 1.0 / sigma < Dt) ? 1.0 / sigma : Dt; /* Eq. 36: h0, parked in h_old */
        const double h0 = h_old;
        sys.template vloop<3>({iw, iy, if0}, [&](int i, const double(&x)[3], double) {
          sys.V(ov, i) = x[0] - x[1];
          sys.V(out, i) = fma(h0, x[2], x[1]);
        });
        state = S_H0;
        return false;
      }
      case S_H0: { /* Eq. 37-38 (R14, R15) */
        const double h0 = h_old, rt = rtol, at = atol;
        double acc = 0.0;
        sys.template vloop<2>({if0, iy}, [&](int, const double(&x)[2], double f) {
          const double d0 = h0 * (f - x[0]);
          const double wt = fma(rt, fabs(x[1]), at);
          const double q = d0 / wt;
          acc = fma(q, q, acc);
        });
        const double est = sqrt(acc / nd);
        h = Dt;
        if (est > 0.0) {
          const double h1 = 0.1 * h0 / sqrt(est);
          if (h1 < Dt) h = h1;
        }
        h_old = 0.0;
        return begin_step(sys);
      }
      case S_STAGE: { /* Eq. 20, 23-24, 26 */
        double mu, nu, mut, gamt;
        if (cbase >= 0) {
          const int b = cbase + 4 * (j - 2);
          mu = sys.td(b); nu = sys.td(b + 1); mut = sys.td(b + 2); gamt = sys.td(b + 3);
        } else {
          double mut1;
          ckb::rkc_coefficients(s, j, mut1, mu, nu, mut, gamt);
        }
        const double c0 = 1.0 - mu - nu, mh = mut * h, gh = gamt * h;
        const int iout = free_vec();
        if (iwm2 == iy) { /* j = 2: w_0 is y itself */
          sys.template vloop<3>({if0, iw, iy}, [&](int i, const double(&x)[3], double f) {
            sys.V(iout, i) = fma(gh, x[0], fma(mh, f, fma(nu, x[2], fma(mu, x[1], c0 * x[2]))));
          });
        } else {
          sys.template vloop<4>({if0, iwm2, iw, iy}, [&](int i, const double(&x)[4], double f) {
            sys.V(iout, i) = fma(gh, x[0], fma(mh, f, fma(nu, x[1], fma(mu, x[2], c0 * x[3]))));
          });
        }
        iwm2 = iw;
        iw = iout;
        if (++j > s) state = S_FINAL;
        return false;
      }
      default:
        break;
    }
    /* S_FINAL: F = f(y_{n+1}), y_{n+1} = w.  Eq. 30-35 */
    double acc = 0.0;
    {
      const double hh = h, rt = rtol, at = atol;
      sys.template vloop<3>({iy, iw, if0}, [&](int, const double(&x)[3], double f) {
        const double del = fma(0.8, x[0] - x[1], 0.4 * hh * (x[2] + f));
        const double wt = fma(rt, fmax(fabs(x[0]), fabs(x[1])), at);
        const double q = del / wt;
        acc = fma(q, q, acc);
      });
    }
    const double err = sqrt(acc / nd);
    if (err <= 1.0) {
      nacc++;
      double fac;
      if (err > 0.0) {
        const double e3 = cbrt(err);
        if (have_prev) fac = 0.8 * (cbrt(err_old) / e3) * (h / h_old) * (1.0 / e3); /* Eq. 34, R13 */
        else fac = 0.8 / e3;
      } else fac = 10.0; /* R26 */
      fac = fmin(10.0, fmax(0.1, fac)); /* Eq. 33 */
      const int o = iy; iy = iw; iw = o; /* y <- w by exchanging the physical vectors */
      iwm2 = iy;
      err_old = err;
      h_old = h;
      have_prev = true;
      sigma_fresh = false;
      if (++since_sigma >= 25) need_sigma = true;
      const int of0 = if0;
      if (last) {
        return true; /* f0 is not needed any more */
      }
      t += h;
      h *= fac;
      /* f0 <- F, then the next step (begin_step); when no sigma refresh is due the copy rides on the first-stage pass */
      last = false;
      if (1.1 * h >= t1 - t) { /* R5 */
        h = t1 - t;
        last = true;
      }
      if (need_sigma) {
        for (int i = 0; i < sys.n; i++) sys.V(of0, i) = sys.F(i);
        pm_begin(sys, false, false);
        return false;
      }
      s = 1 + (int)floor(sqrt(fma(1.54 * h, sigma, 1.0)));
      if (s < 2) s = 2;
      if (s > s_max) {
        s = s_max;
        h = ((double)s_max * (double)s_max - 1.0) / (1.54 * sigma);
        last = false;
      }
      if (s > smax_used) smax_used = s;
      if (++attempts > 1000000) {
        status = ST_MAXSTEPS;
        return true;
      }
      double mut1;
      if (s <= sys.m.s_tab) {
        mut1 = sys.td(sys.m.o_rkc + (s - 2));
        cbase = sys.m.o_rkcs + 4 * ((s - 2) * (s - 1) / 2);
      } else {
        double mu, nu, mut, gamt;
        ckb::rkc_coefficients(s, 2, mut1, mu, nu, mut, gamt);
        cbase = -1;
      }
      const double mh = mut1 * h;
      const int out = iw;
      sys.template vloop<1>({iy}, [&](int i, const double(&x)[1], double f) {
        sys.V(of0, i) = f;
        sys.V(out, i) = fma(mh, f, x[0]); /* Eq. 19 */
      });
      j = 2;
      state = S_STAGE;
      return false;
    }
    nrej++;
    double fac;
    if (isfinite(err)) fac = fmin(10.0, fmax(0.1, 0.8 / cbrt(err))); /* Eq. 35 */
    else {
      fac = 0.1;
      saw_nonfinite = true;
    }
    h *= fac;
    have_prev = false;
    iwm2 = iy;
    if (!sigma_fresh) need_sigma = true; /* R16 */
    const double tmax = fmax(fabs(t), fabs(t1));
    if (!(h > 10.0 * CKB_U * tmax)) {
      status = saw_nonfinite ? ST_NONFINITE : ST_UNDERFLOW;
      return true;
    }
    return begin_step(sys);
  }

  /* 3 = error estimate, 2 = last stage of a step, 1 = earlier stage, 0 = other */
  __device__ __forceinline__ int phase() const { return state == S_FINAL ? 3 : state == S_STAGE ? (j == s ? 2 : 1) : 0; }
  __device__ __forceinline__ void result(int (&st)[4]) {
    if (status == ST_OK && flag) status = flag;
    st[0] = nfe; st[1] = nacc; st[2] = nrej; st[3] = smax_used;
  }
};

template <class S, int METHOD>
struct MemIntegratorOf { typedef RkckMem<S> type; };
template <class S>
struct MemIntegratorOf<S, 1> { typedef RkcMem<S> type; };

#define CKBT_MAX_BLOCK 256

template <class S>
__device__ __forceinline__ void tsys_setup(S &sys, const DevThread &m, double *ws, size_t NT) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  sys.n = m.n;
  sys.cC = (unsigned)((warp * 2 * m.n * 32 + lane) * 8);
  sys.cF = sys.cC + (unsigned)(m.n * 256);
  sys.NT = NT;
  sys.ws = ws + (size_t)blockIdx.x * blockDim.x + threadIdx.x;
}

/* Persistent grid, one block per SM; every LANE pulls system indices from the work queue (lane refill)
 * and the lanes of a warp are kept in the same stage where that costs one idle evaluation (stage alignment). */
template <class STAB, int METHOD, int CV>
__global__ void __launch_bounds__(CKBT_MAX_BLOCK, 1)
integrate_thread_kernel(const __grid_constant__ DevThread m, const __grid_constant__ STAB st,
                        const unsigned long long *__restrict__ aux, double *__restrict__ ws, double *__restrict__ states,
                        const double *__restrict__ pressure, double p_uniform, long long N, long long ld, double t0,
                        double dt, double rtol, double atol, int *__restrict__ status, int *__restrict__ stats,
                        unsigned long long *__restrict__ counter, const int *__restrict__ order) {
  typedef TSys<STAB, CV> S;
  S sys(m, st, aux);
  const size_t NT = (size_t)gridDim.x * blockDim.x;
  tsys_setup(sys, m, ws, NT);
  const int n = m.n;
  const long long n_static = (long long)NT;
  typename MemIntegratorOf<S, METHOD>::type integ;
  long long qi = (long long)blockIdx.x * blockDim.x + threadIdx.x, ode = 0;
  bool need_load = true, active = true, held_last = false;
#if CKBT_LOCKSTEP
  __shared__ unsigned ls_ph[64];
  unsigned ls_iter = 0;
#endif
  sys.set_pressure(1.0);
  integ.iw = 0;
  for (int i = 0; i < n; i++) sys.V(0, i) = 1.0; /* finite argument for a lane that never gets a system */
  while (true) {
    if (need_load && active) {
      if (qi >= N) {
        active = false; /* queue exhausted: the lane idles on its last argument */
      } else {
        ode = order ? (long long)order[qi] : qi;
        sys.set_pressure(pressure ? pressure[ode] : p_uniform);
        for (int i = 0; i < n; i++) sys.V(0, i) = states[(size_t)i * ld + ode];
        integ.start(sys, t0, t0 + dt, rtol, atol);
        need_load = false;
      }
    }
    /* the warps of the block enter f(y) together: one instruction stream per SM through the instruction caches (the
     * code of one trip is several times the 32 KB L1.5); a warp that has run out of systems only keeps the barrier */
    const bool warp_any = __any_sync(0xffffffffu, active);
#if CKBT_LOCKSTEP
    int b_last = 0, b_final = 0;
    if constexpr (METHOD == 1) { /* this warp's lanes in their last stage / at the error estimate, for the block-wide vote */
      const int ph = active ? integ.phase() : 0;
      const unsigned w_last = __popc(__ballot_sync(0xffffffffu, ph == 2)), w_final = __popc(__ballot_sync(0xffffffffu, ph == 3));
      if ((threadIdx.x & 31) == 0) ls_ph[(ls_iter & 1) * 32 + (threadIdx.x >> 5)] = w_last | (w_final << 16);
    }
    if (!__syncthreads_or(warp_any)) break;
    if constexpr (METHOD == 1) {
      const int lane = threadIdx.x & 31;
      const unsigned v = __reduce_add_sync(0xffffffffu, lane < (int)(blockDim.x >> 5) ? ls_ph[(ls_iter & 1) * 32 + lane] : 0u);
      b_last = (int)(v & 0xFFFFu);
      b_final = (int)(v >> 16);
      ls_iter++; /* double buffer: a warp writes its next counts while a slower one may still read these */
    }
    if (!warp_any) continue;
#else
    if (!warp_any) break;
#endif
    bool hold = false;
    if constexpr (METHOD == 0) { /* RKCK: stage-2 lanes sit out an evaluation that some lane needs as stage 1 (R25) */
      const bool s1 = active && integ.stage == 1;
      const bool any1 = __any_sync(0xffffffffu, s1);
      hold = active && !s1 && any1;
    } else { /* RKC: last-stage and error-estimate evaluations line up (never held twice in a row) */
      const int ph = active ? integ.phase() : 0;
#if CKBT_LOCKSTEP /* the vote is taken over the block: its warps reach the error estimate, the long path of advance(), together */
      const int n_last = b_last, n_final = b_final;
#else
      const int n_last = __popc(__ballot_sync(0xffffffffu, ph == 2)), n_final = __popc(__ballot_sync(0xffffffffu, ph == 3));
#endif
      hold = !held_last && ((ph == 3 && n_last > 0 && n_last >= n_final) || (ph == 2 && n_final > n_last));
      held_last = hold;
    }
    sys.rhs(integ.arg());
    if (active && !hold && integ.advance(sys)) {
      int st4[4];
      integ.result(st4);
      const int iy = integ.yvec();
      for (int i = 0; i < n; i++) states[(size_t)i * ld + ode] = sys.V(iy, i);
      if (status) status[ode] = integ.status;
      if (stats) {
#pragma unroll
        for (int k = 0; k < 4; k++) stats[(size_t)k * N + ode] = st4[k];
      }
      qi = n_static + (long long)atomicAdd(counter, 1ull);
      need_load = true;
    }
  }
}

/* f(y) only (source-term parity test, ckb_rhs): one system per thread, workspace vector 0 holds the argument */
template <class STAB, int CV>
__global__ void __launch_bounds__(CKBT_MAX_BLOCK, 1)
rhs_thread_kernel(const __grid_constant__ DevThread m, const __grid_constant__ STAB st,
                  const unsigned long long *__restrict__ aux, double *__restrict__ ws, const double *__restrict__ states,
                  const double *__restrict__ pressure, double p_uniform, long long N, long long ld,
                  double *__restrict__ dydt, int repeat) {
  typedef TSys<STAB, CV> S;
  S sys(m, st, aux);
  const size_t NT = (size_t)gridDim.x * blockDim.x;
  tsys_setup(sys, m, ws, NT);
  const int n = m.n;
  for (long long ode = (long long)blockIdx.x * blockDim.x + threadIdx.x; __any_sync(0xffffffffu, ode < N); ode += (long long)NT) {
    const bool mine = ode < N;
    sys.set_pressure(mine ? (pressure ? pressure[ode] : p_uniform) : 1.0);
    for (int i = 0; i < n; i++) sys.V(0, i) = mine ? states[(size_t)i * ld + ode] : 1.0;
    for (int r = 0; r < repeat; r++) sys.rhs(0);
    if (mine)
      for (int i = 0; i < n; i++) dydt[(size_t)i * ld + ode] = sys.F(i);
  }
}

} /* namespace ckbt */
