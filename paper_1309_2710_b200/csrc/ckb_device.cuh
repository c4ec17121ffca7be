/*
 * ckb_device.cuh -- device code of the batched chemistry integrator (sm_100a, FP64).
 *
 * One templated "system" type maps an ODE system onto L lanes (L = 1: thread-per-ODE, the paper's
 * mapping P:255; L = 32: warp-per-ODE; L = 8/16: sub-warp).  Component c of the (renumbered, see
 * ckb_tables.h) unknowns {T, Y_1..Y_K} lives in lane (c mod L), register slot (c div L); every
 * stage vector of the integrators is a register array double[NV] with static indexing only.  The
 * runtime-indexed quantities of the source term (concentrations C_c, third-body concentrations [M], net
 * rates of progress q_s) live in shared memory, interleaved so that thread-per-ODE access is
 * bank-conflict free.
 *
 * Source term: Eq. 2-6.  Integrators: RKCK Eq. 7-17, RKC Eq. 18-39.
 * The readings of the paper where it is silent (R-numbers) are listed in DESIGN.md section 4.
 * Nothing here is shared with the CPU checker (constants that appear in both are typed twice).
 */
#pragma once
#ifndef __CUDACC_RTC__ /* the runtime compiler has the math functions built in and no host headers */
#include <math.h>
#include <stdint.h>
#endif

#include "ckb_tables.h"

namespace ckb {

/* R20: physical constants */
#define CKB_RU 8.314462618e7 /* erg/(mol K) */

#ifndef CKB_XS_RKCK_K12
#define CKB_XS_RKCK_K12 0 /* thread-per-ODE RKCK: 1 = k1, k2 live in the shared scratch too */
#endif
#ifndef CKB_XS_RKC_F0
#define CKB_XS_RKC_F0 0 /* thread-per-ODE RKC: 1 = f0 and w_{j-2} live in the shared scratch too */
#endif
#ifndef CKB_RKC_BLOCK_ALIGN
#define CKB_RKC_BLOCK_ALIGN 1 /* ... and, in a lock-step block, over the warps of the block */
#endif
#ifndef CKB_BLOCK_LOCKSTEP
#define CKB_BLOCK_LOCKSTEP 0
#endif
#ifndef CKB_XS_RKC_Y
#define CKB_XS_RKC_Y 0 /* ... and y as well */
#endif
#ifndef CKB_RKCK_ALIGN
#define CKB_RKCK_ALIGN 1 /* thread-per-ODE RKCK: the lanes of a warp stay in the same stage (integrate_kernel): +35 % */
#endif
#ifndef CKB_RKC_ALIGN
#define CKB_RKC_ALIGN 1 /* RKC, several systems per warp: they line up on stage / error-estimate evaluations */
#endif
#ifndef CKB_EXP_TABLE
#define CKB_EXP_TABLE 0
#endif
#ifndef CKB_UNROLL_SLOTS
#define CKB_UNROLL_SLOTS 1 /* reaction slots in flight per lane: 2 slots = 4 independent exp chains */
#endif

/* exp(x) for the Arrhenius coefficients (Eq. 5): x = k ln2 + r, |r| <= ln2/2; e^r = 1 + r + r^2 q(r) with
 * q of degree 9 fitted at Chebyshev nodes (truncation 1.7e-17 relative); 2^k by exponent arithmetic with k
 * clamped to the normal range, so x << -708 gives ~1e-308 (not 0, not NaN) and the code has no branch.
 * The coefficients sit in the constant bank so that every DFMA takes its addend as a c[][] operand. */
static __constant__ double c_expq[10] = {
    0.5000000000000001,    0.16666666666666669,   0.041666666666623824,  0.008333333333330039,
    0.0013888888917367081, 0.00019841269863171557, 2.4801521057868204e-05, 2.7557268276905696e-06,
    2.7620201591031547e-07, 2.5100472505694996e-08};

/* The constants of ckb_exp: either operands from the constant bank (PIN = false; thread-per-ODE, where registers
 * are scarce) or pinned in registers for the duration of the slot loop (PIN = true; otherwise the compiler
 * re-materialises them with ~12 extra instructions per reaction slot). */
template <bool PIN>
struct ExpConst {
  double log2e, ln2hi, ln2lo, q[10];
  __device__ __forceinline__ ExpConst() {
    log2e = 1.4426950408889634;
    ln2hi = -0.6931471805599453;
    ln2lo = -2.3190468138462996e-17;
#pragma unroll
    for (int i = 0; i < 10; i++) q[i] = c_expq[i];
    if (PIN) {
      asm volatile("" : "+d"(log2e), "+d"(ln2hi), "+d"(ln2lo));
#pragma unroll
      for (int i = 0; i < 10; i++) asm volatile("" : "+d"(q[i]));
    }
  }
};

#if CKB_EXP_TABLE
/* Table variant: x = (64 k + j) ln2/64 + r, |r| <= ln2/128, e^x = 2^k 2^(j/64) p(r) with p of degree 5 (truncation
 * r^6/720 <= 3.5e-17) and 2^(j/64) from a 64-entry table in shared memory: 12 FP64 instructions instead of 17 and a
 * dependency chain of 9 instead of 14.  CKB_EXP_TABLE_REPL copies of the table, entry j of copy c at [j * REPL + c]:
 * with 16 copies lane l reads copy (l mod 16), i.e. always its own bank pair -- conflict free whatever j is (the
 * lane-distributed kernels, whose shared-memory pipe is busy); one copy where that pipe is idle (thread-per-ODE). */
#ifndef CKB_EXP_TABLE_REPL
#define CKB_EXP_TABLE_REPL 1
#endif
__device__ __forceinline__ double *ckb_exp_table() {
  __shared__ double tab[64 * CKB_EXP_TABLE_REPL];
  return tab;
}
__device__ __forceinline__ void ckb_exp_table_init() {
  for (int i = threadIdx.x; i < 64 * CKB_EXP_TABLE_REPL; i += blockDim.x)
    ckb_exp_table()[i] = exp2((double)(i / CKB_EXP_TABLE_REPL) * 0.015625);
  __syncthreads();
}
__device__ __forceinline__ double ckb_exp_table_at(int kj) {
  if (CKB_EXP_TABLE_REPL == 1) return ckb_exp_table()[kj & 63];
  return ckb_exp_table()[(kj & 63) * CKB_EXP_TABLE_REPL + (threadIdx.x & (CKB_EXP_TABLE_REPL - 1))];
}
static __constant__ double c_expt[6] = {92.332482616893657 /* 64 / ln 2 */, -0.6931471805599453 * 0.015625,
                                        -2.3190468138462996e-17 * 0.015625, 1.0 / 120.0, 1.0 / 24.0, 1.0 / 6.0};
template <bool PIN>
__device__ __forceinline__ double ckb_exp(double x, const ExpConst<PIN> &) {
  /* literal constants: the compiler picks immediates / constant-bank operands itself (measured on the specialised
   * thread-per-ODE kernels: 2 % faster than reading them from c_expt) */
  const double t = fma(x, 92.332482616893657, 6755399441055744.0); /* 64 / ln 2 */
  const double kd = t - 6755399441055744.0;
  double r = fma(kd, -0.6931471805599453 * 0.015625, x);
  r = fma(kd, -2.3190468138462996e-17 * 0.015625, r);
  const int kj = __double2loint(t);
  const double tv = ckb_exp_table_at(kj);
  double p = 1.0 / 120.0;
  p = fma(p, r, 1.0 / 24.0);
  p = fma(p, r, 1.0 / 6.0);
  p = fma(p, r, 0.5);
  p = fma(p, r, 1.0);
  p = fma(p, r, 1.0);
  p *= tv;
  int k = kj >> 6;
  k = max(-1022, min(1022, k));
  return __hiloint2double(__double2hiint(p) + (k << 20), __double2loint(p));
}
#else
template <bool PIN>
__device__ __forceinline__ double ckb_exp(double x, const ExpConst<PIN> &c) {
  const double t = fma(x, c.log2e, 6755399441055744.0); /* 1.5 * 2^52: round to nearest integer */
  const double kd = t - 6755399441055744.0;
  double r = fma(kd, c.ln2hi, x);
  r = fma(kd, c.ln2lo, r);
  double p = c.q[9];
#pragma unroll
  for (int i = 8; i >= 0; i--) p = fma(p, r, c.q[i]);
  p = fma(p, r, 1.0);
  p = fma(p, r, 1.0);
  int k = __double2loint(t);
  k = max(-1022, min(1023, k));
  return __hiloint2double(__double2hiint(p) + (k << 20), __double2loint(p));
}
#endif

/* N exponentials advanced in lock step (same arithmetic per chain as ckb_exp, non-table form): the N dependency
 * chains are emitted interleaved, step by step, so that a warp has N DFMAs in flight instead of one (the compiler
 * keeps the emission order; left to itself it runs the chains one after the other). */
#if CKB_EXP_TABLE
template <int N, bool PIN>
__device__ __forceinline__ void ckb_exp_n(const double (&x)[N], double (&out)[N], const ExpConst<PIN> &) {
  double t[N], r[N], p[N], tv[N];
  double a0 = c_expt[0], a1 = c_expt[1], a2 = c_expt[2];
  if (PIN) asm volatile("" : "+d"(a0), "+d"(a1), "+d"(a2));
#pragma unroll
  for (int u = 0; u < N; u++) t[u] = fma(x[u], a0, 6755399441055744.0);
#pragma unroll
  for (int u = 0; u < N; u++) tv[u] = ckb_exp_table_at(__double2loint(t[u]));
#pragma unroll
  for (int u = 0; u < N; u++) r[u] = fma(t[u] - 6755399441055744.0, a1, x[u]);
#pragma unroll
  for (int u = 0; u < N; u++) r[u] = fma(t[u] - 6755399441055744.0, a2, r[u]);
#pragma unroll
  for (int u = 0; u < N; u++) p[u] = fma(c_expt[3], r[u], c_expt[4]);
#pragma unroll
  for (int u = 0; u < N; u++) p[u] = fma(p[u], r[u], c_expt[5]);
#pragma unroll
  for (int u = 0; u < N; u++) p[u] = fma(p[u], r[u], 0.5);
#pragma unroll
  for (int u = 0; u < N; u++) p[u] = fma(p[u], r[u], 1.0);
#pragma unroll
  for (int u = 0; u < N; u++) p[u] = fma(p[u], r[u], 1.0);
#pragma unroll
  for (int u = 0; u < N; u++) {
    p[u] *= tv[u];
    int k = __double2loint(t[u]) >> 6;
    k = max(-1022, min(1022, k));
    out[u] = __hiloint2double(__double2hiint(p[u]) + (k << 20), __double2loint(p[u]));
  }
}
#else
template <int N, bool PIN>
__device__ __forceinline__ void ckb_exp_n(const double (&x)[N], double (&out)[N], const ExpConst<PIN> &c) {
  double t[N], r[N], p[N];
#pragma unroll
  for (int u = 0; u < N; u++) t[u] = fma(x[u], c.log2e, 6755399441055744.0);
#pragma unroll
  for (int u = 0; u < N; u++) r[u] = fma(t[u] - 6755399441055744.0, c.ln2hi, x[u]);
#pragma unroll
  for (int u = 0; u < N; u++) r[u] = fma(t[u] - 6755399441055744.0, c.ln2lo, r[u]);
#pragma unroll
  for (int u = 0; u < N; u++) p[u] = c.q[9];
#pragma unroll
  for (int i = 8; i >= 0; i--) {
#pragma unroll
    for (int u = 0; u < N; u++) p[u] = fma(p[u], r[u], c.q[i]);
  }
#pragma unroll
  for (int u = 0; u < N; u++) p[u] = fma(p[u], r[u], 1.0);
#pragma unroll
  for (int u = 0; u < N; u++) p[u] = fma(p[u], r[u], 1.0);
#pragma unroll
  for (int u = 0; u < N; u++) {
    int k = __double2loint(t[u]);
    k = max(-1022, min(1023, k));
    out[u] = __hiloint2double(__double2hiint(p[u]) + (k << 20), __double2loint(p[u]));
  }
}
#endif

#ifndef CKB_TMEM
#define CKB_TMEM 0 /* warp-per-ODE integrate kernels: 1 = the reaction-slot table is read from tensor memory */
#endif
#if CKB_TMEM
/* Tensor memory as a table store.  The warp-per-ODE kernels are bound by the L1/shared data pipe
 * (ncu: LSU wavefronts at 82 % of peak), and half of those wavefronts are the coalesced loads of the slot table --
 * the same 8 words per lane every evaluation of f(y).  TMEM (512 columns x 128 lanes x 32 bit per SM) is read with
 * tcgen05.ld over its own datapath: lane g of warp w owns TMEM lane 32 (w mod 4) + g, and the 8 table words of slot
 * round r sit in 16 consecutive columns -- ONE tcgen05.ld.32x32b.x16 per slot instead of 8 LDG.64. */
#define CKB_TMEM_COLS 512
__device__ __forceinline__ void tm_alloc(unsigned *holder_smem) {
  const unsigned dst = (unsigned)__cvta_generic_to_shared(holder_smem);
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(dst), "r"(CKB_TMEM_COLS) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tm_dealloc(unsigned base) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(base), "r"(CKB_TMEM_COLS) : "memory");
}
__device__ __forceinline__ void tm_fence_sync_fence() {
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
}
__device__ __forceinline__ void tm_st16(unsigned addr, const unsigned (&v)[16]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
               ::"r"(addr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]),
               "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]) : "memory");
}
__device__ __forceinline__ void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tm_ld16(unsigned addr, unsigned (&v)[16]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
               : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
                 "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
               : "r"(addr) : "memory");
}
__device__ __forceinline__ void tm_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
#ifndef CKB_TMEM_SLOTS
#define CKB_TMEM_SLOTS 1 /* reaction slots in flight per lane in the TMEM slot loop (2 slots = 4 exp chains in lock step:
                            measured slower, the registers they take cost more than the overlap gives) */
#endif
#endif

/* ------------------------------------------------------------------------------------------------
 * Sys<L, NV, TAB>: one ODE system on L lanes with NV register slots per lane; tables from the kernel
 * parameter bank (ParamTab) or global/L1 (GlobalTab).
 * ---------------------------------------------------------------------------------------------- */
template <int L_, int NV_, class TAB, int M_ = 1, int CV_ = 0>
struct Sys {
  /* closure (compile time, so that the constant-pressure kernels carry none of it): false = constant pressure
   * (Eq. 6), true = constant volume (R29: the "pressure" argument carries the density rho) */
  static constexpr bool CV = CV_ != 0;
  /* M systems share the lanes of a group and are evaluated together: every table word is loaded and decoded
   * once for all of them, and their (independent) dependency chains interleave -- DESIGN.md 7.4. */
  static constexpr int L = L_, NV = NV_, G = 32 / L_, M = M_;
  /* shared-memory interleave: thread-per-ODE interleaves the 32 systems of a warp element by element (conflict
   * free: all lanes read the same element); lane-distributed mappings give every system a contiguous region */
  static constexpr int GI = (L_ == 1) ? 32 : 1;
  const DevMech &m;
  const TAB &tab;
  double *sR;      /* shared region of system 0 of this group (ckb_tables.h), element e at sR[e*G]; system q at + q*RS */
  int RS;          /* doubles between the regions of two systems of the group */
  int qoff;        /* (n + NTB + 1) * GI: start of the q region */
  double *sX;      /* scratch of the integrator behind the region (XVec), same interleave */
  double *sH;      /* thread-per-ODE: h_k/(RT) parked here between the two halves of f(y) instead of in registers */
#ifdef CKB_GEN_RHS
  static constexpr int HDOUBLES = 0;
#else
  static constexpr int HDOUBLES = (L_ == 1) ? NV_ : 0;
#endif
  unsigned mask;   /* lanes of this group */
  int g;           /* lane within the group */
  int src0;        /* warp lane that holds component 0 (T) */
  double pR[M], Rp[M]; /* p / Ru and Ru / p (R24: pressure constant over the call) */
#if CKB_TMEM
  bool tm_on = false;  /* slot table resident in tensor memory (set by integrate_kernel) */
  unsigned tm_addr = 0;/* TMEM address of this warp's lane quarter, column of slot round 0 */
#endif

  __device__ __forceinline__ Sys(const DevMech &m_, const TAB &tab_) : m(m_), tab(tab_) {}
  __device__ __forceinline__ unsigned long long tw(int i) const { return tab.ld(i); }
  __device__ __forceinline__ double td(int i) const { return __longlong_as_double((long long)tab.ld(i)); }
  __device__ __forceinline__ void set_pressure(int q, double p) {
    if (CV) { /* R29, constant volume: p carries the density rho (constant over the call) */
      pR[q] = p;
      Rp[q] = 1.0 / p;
    } else {
      pR[q] = p / CKB_RU;
      Rp[q] = CKB_RU / p;
    }
  }

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

  /* f(y): Eq. 2-6 for the M systems of the group.  y, f: [system][slot], component (g + L*i) in slot i. */
  /* Y(q, i): slot i of the argument of system q (read in place from the integrators' registers) */
  template <class GetY>
  __device__ __forceinline__ void rhs(GetY Y, double (&f)[M][NV]) {
#ifdef CKB_GEN_RHS
    /* mechanism-specialised translation unit (ckb_gen.cu): straight-line f(y) generated from the mechanism,
     * every table value a literal, C_k, [M] and q_s in registers -- no shared region, no table reads */
    if constexpr (L == 1 && M == 1) {
#include CKB_GEN_RHS
      return;
    }
#endif
    const int n = m.n;
    double T[M], invT[M], lnT[M], s1[M], s2[M];
    double hrt[M][L == 1 ? 1 : NV], yw[M][L == 1 ? 1 : NV];
#pragma unroll
    for (int q = 0; q < M; q++) {
      T[q] = bcast0(Y(q, 0));
      invT[q] = 1.0 / T[q];
      lnT[q] = log(T[q]);
      s1[q] = 0.0;
      s2[q] = 0.0;
    }
    /* species table rows of T and of padding components are all zero: no branch needed */
#pragma unroll
    for (int i = 0; i < NV; i++) {
      const int b = m.o_sp + i * CKB_SP_WORDS * L + g;
      /* R8a: cp_k/R = a1 + a2 T + ... + a5 T^4;  h_k/(RT) = a1 + a2 T/2 + ... + a5 T^4/5 + a6/T */
      double cc[5], hc[6];
      /* R30 (two temperature ranges, ckb_mech_load2): this lane's species takes its coefficients from the second
       * species table where T > T_mid -- a select between two table rows, per species and per evaluation */
      int bt = b;
      if (m.o_sp2) { /* launch-uniform */
        const int b2 = m.o_sp2 + i * CKB_SP_WORDS * L + g;
        if (T[0] > td(b2 + CKB_SP_INVW * L)) bt = b2;
      }
#pragma unroll
      for (int k = 0; k < 5; k++) cc[k] = td(bt + (CKB_SP_CP + k) * L);
#pragma unroll
      for (int k = 0; k < 6; k++) hc[k] = td(bt + (CKB_SP_H + k) * L);
      const double iw = td(b + CKB_SP_INVW * L);
#pragma unroll
      for (int q = 0; q < M; q++) {
        double cp = cc[4], h = hc[4];
#pragma unroll
        for (int k = 3; k >= 0; k--) {
          cp = fma(cp, T[q], cc[k]);
          h = fma(h, T[q], hc[k]);
        }
        h = fma(hc[5], invT[q], h);
        if (CV) h -= 1.0; /* R29: u_k W_k/(Ru T) = h_k W_k/(Ru T) - 1 */
        const double v = Y(q, i) * iw; /* Y_k / W_k */
        if (L == 1) {
          sH[i * GI] = h;
        } else {
          yw[q][i] = v;
          hrt[q][i] = h;
        }
        s1[q] += v;
        s2[q] = fma(v, cp, s2[q]);
      }
    }
#pragma unroll
    for (int o = L / 2; o > 0; o >>= 1) {
#pragma unroll
      for (int q = 0; q < M; q++) {
        s1[q] += __shfl_xor_sync(mask, s1[q], o);
        s2[q] += __shfl_xor_sync(mask, s2[q], o);
      }
    }
    /* R9a: ideal gas at constant pressure: rho = p / (Ru T sum_k Y_k/W_k), C_k = rho Y_k / W_k;
     * R29: constant volume: rho given, C_tot = rho sum_k Y_k/W_k */
    double ctot[M], invrho[M], rcp_c[M];
#pragma unroll
    for (int q = 0; q < M; q++) {
      /* 1 / cp (1 / c_v) for Eq. 6 now, off the critical path, instead of a division at the very end of f(y) (lane-distributed
       * mappings: a warp waits out every dependent instruction; thread-per-ODE keeps the division: registers) */
      rcp_c[q] = (L > 1) ? 1.0 / (CV ? s2[q] - s1[q] : s2[q]) : 0.0;
      ctot[q] = CV ? pR[q] * s1[q] : pR[q] * invT[q];
      const double rho = CV ? pR[q] : ctot[q] * (1.0 / s1[q]);
      invrho[q] = CV ? Rp[q] : s1[q] * T[q] * Rp[q];
#pragma unroll
      for (int i = 0; i < NV; i++) {
        const int c = g + L * i;
        if (c >= 1 && c < n)
          sR[q * RS + c * GI] = rho * (L == 1 ? Y(q, i) * td(m.o_sp + i * CKB_SP_WORDS * L + g + CKB_SP_INVW * L) : yw[q][i]);
      }
    }
    gsync();
    /* R22: [M] = sum_k alpha_k C_k = C_tot + sum_listed (alpha_k - 1) C_k, one value per efficiency set */
    for (int r = 0; r < m.NTBR; r++) {
      double Mc[M];
#pragma unroll
      for (int q = 0; q < M; q++) Mc[q] = ctot[q];
      int b = m.o_tb + r * m.TBE * 2 * L + g;
      for (int e = 0; e < m.TBE; e++, b += 2 * L) {
        const double am1 = td(b);
        const unsigned off = (unsigned)tw(b + L); /* byte offset */
#pragma unroll
        for (int q = 0; q < M; q++)
          Mc[q] = fma(am1, *reinterpret_cast<const double *>(reinterpret_cast<const char *>(sR + q * RS) + off), Mc[q]);
      }
      const int t = r * L + g;
      if (t < m.NTB) {
#pragma unroll
        for (int q = 0; q < M; q++) sR[q * RS + (n + t) * GI] = Mc[q];
      }
    }
    if (m.o_fo) { /* launch-uniform: the mechanism has fall-off reactions (R31).  A second pass, so that mechanisms without
                     them keep the loop above as it was: the set of a fall-off reaction has its [M] replaced by
                     P_r/(1+P_r) F (k_j stays k_inf); each lane revisits the sets it wrote itself */
      for (int r = 0; r < m.NTBR; r++) {
        const int t = r * L + g, fb = m.o_fo + r * 8 * L + g;
        const int kind = (int)td(fb);
        if (kind > 0 && t < m.NTB) {
          const ExpConst<false> fec;
          const double dlnA = td(fb + L), dbeta = td(fb + 2 * L), dtheta = td(fb + 3 * L);
#pragma unroll
          for (int q = 0; q < M; q++) {
            const double Pr = sR[q * RS + (n + t) * GI] * ckb_exp(fma(-dtheta, invT[q], fma(dbeta, lnT[q], dlnA)), fec);
            double B = Pr / (1.0 + Pr);
            if (kind >= 2) { /* Troe */
              const double a = td(fb + 4 * L);
              double Fc = (1.0 - a) * ckb_exp(-T[q] * td(fb + 5 * L), fec) + a * ckb_exp(-T[q] * td(fb + 6 * L), fec);
              if (kind == 2) Fc += ckb_exp(-td(fb + 7 * L) * invT[q], fec);
              const double lF = log10(Fc), lP = log10(Pr);
              const double c = -0.4 - 0.67 * lF, nn = 0.75 - 1.27 * lF;
              const double x = (lP + c) / (nn - 0.14 * (lP + c));
              B *= exp(2.302585092994046 * (lF / (1.0 + x * x)));
            }
            sR[q * RS + (n + t) * GI] = B;
          }
        }
      }
    }
    gsync();
    /* Eq. 4-5: q_s = [M] (k_f prod C_reactants - k_r prod C_products); absent molecules point at C_0 = 1, an
     * absent third body at a 1.0.  The 16-bit fields are BYTE offsets into the system's region. */
#if CKB_TMEM
    if (L == 32 && M == 1 && tm_on) { /* warp-uniform: slot table in tensor memory, U slots per lane in flight */
      constexpr int U = CKB_TMEM_SLOTS;
      const ExpConst<true> ec;
      double *qp = sR + qoff + g;
      const char *c = reinterpret_cast<const char *>(sR);
      const int last = m.NSR - 1, nq = m.NSR * L; /* -q_s sits NSR*L doubles behind q_s */
      for (int r = 0; r < m.NSR; r += U, qp += U * L) {
        unsigned v[U][16];
#pragma unroll
        for (int u = 0; u < U; u++) tm_ld16(tm_addr + (unsigned)(r + u < last ? r + u : last) * 16u, v[u]);
        tm_wait_ld();
        double xf[U], xr[U], pf[U], pr[U], mt[U];
#pragma unroll
        for (int u = 0; u < U; u++) {
#define CKB_TD(x) __hiloint2double((int)v[u][2 * (x) + 1], (int)v[u][2 * (x)])
          xf[u] = fma(-CKB_TD(CKB_SL_THF), invT[0], fma(CKB_TD(CKB_SL_BF), lnT[0], CKB_TD(CKB_SL_LNAF)));
          xr[u] = fma(-CKB_TD(CKB_SL_THR), invT[0], fma(CKB_TD(CKB_SL_BR), lnT[0], CKB_TD(CKB_SL_LNAR)));
#undef CKB_TD
          const unsigned alo = v[u][2 * CKB_SL_IDXA], ahi = v[u][2 * CKB_SL_IDXA + 1];
          const unsigned blo = v[u][2 * CKB_SL_IDXB], bhi = v[u][2 * CKB_SL_IDXB + 1];
#define CKB_AT(off) (*reinterpret_cast<const double *>(c + (off)))
          pf[u] = CKB_AT(alo & 0xFFFFu) * CKB_AT(alo >> 16) * CKB_AT(ahi & 0xFFFFu);
          pr[u] = CKB_AT(blo & 0xFFFFu) * CKB_AT(blo >> 16) * CKB_AT(bhi & 0xFFFFu);
          mt[u] = CKB_AT(ahi >> 16);
#undef CKB_AT
        }
        double xs[2 * U], ks[2 * U], res[U];
#pragma unroll
        for (int u = 0; u < U; u++) { xs[2 * u] = xf[u]; xs[2 * u + 1] = xr[u]; }
        ckb_exp_n<2 * U>(xs, ks, ec);
#pragma unroll
        for (int u = 0; u < U; u++) res[u] = (ks[2 * u] * pf[u] - ks[2 * u + 1] * pr[u]) * mt[u];
#pragma unroll
        for (int u = 0; u < U; u++)
          if (u == 0 || r + u <= last) {
            qp[u * L] = res[u];
            qp[nq + u * L] = -res[u];
          }
      }
    } else
#endif
    {
      constexpr int US = CKB_UNROLL_SLOTS;
      const ExpConst<(L > 1)> ec;
      int b = m.o_sl + g;
      double *qp = sR + qoff + g * GI;
#pragma unroll US
      for (int r = 0; r < m.NSR; r++, b += CKB_SL_WORDS * L, qp += L * GI) {
        double lnAf, bf, thf, lnAr, br, thr;
        unsigned long long wa, wb;
        {
          lnAf = td(b + CKB_SL_LNAF * L), bf = td(b + CKB_SL_BF * L), thf = td(b + CKB_SL_THF * L);
          lnAr = td(b + CKB_SL_LNAR * L), br = td(b + CKB_SL_BR * L), thr = td(b + CKB_SL_THR * L);
          wa = tw(b + CKB_SL_IDXA * L), wb = tw(b + CKB_SL_IDXB * L);
        }
        const unsigned alo = (unsigned)wa, ahi = (unsigned)(wa >> 32), blo = (unsigned)wb, bhi = (unsigned)(wb >> 32);
        const unsigned a0 = alo & 0xFFFFu, a1 = alo >> 16, a2 = ahi & 0xFFFFu, tb = ahi >> 16;
        const unsigned b0 = blo & 0xFFFFu, b1 = blo >> 16, b2 = bhi & 0xFFFFu;
#pragma unroll
        for (int q = 0; q < M; q++) {
          const char *c = reinterpret_cast<const char *>(sR + q * RS);
#define CKB_AT(off) (*reinterpret_cast<const double *>(c + (off)))
          const double xf = fma(-thf, invT[q], fma(bf, lnT[q], lnAf));
          const double xr = fma(-thr, invT[q], fma(br, lnT[q], lnAr));
          const double pf = CKB_AT(a0) * CKB_AT(a1) * CKB_AT(a2);
          const double pr = CKB_AT(b0) * CKB_AT(b1) * CKB_AT(b2);
          const double kf = ckb_exp(xf, ec), kr = ckb_exp(xr, ec);
          const double qs = (kf * pf - kr * pr) * CKB_AT(tb);
          qp[q * RS] = qs;
          if (L == CKB_NEGQ_L) qp[q * RS + m.NSR * L] = -qs; /* the gather reads -q_s where the coefficient is -1 */
#undef CKB_AT
        }
      }
    }
    gsync();
    /* Eq. 3: omega_c = sum_s (nu''_cs - nu'_cs) q_s (gather);  Eq. 2: dY_k/dt = W_k omega_k / rho */
    double s3[M];
#pragma unroll
    for (int q = 0; q < M; q++) s3[q] = 0.0;
    int gp = m.o_gat + g;
    const double *sQ = sR + qoff;
    double om[M][NV]; /* Eq. 3 per register slot */
#pragma unroll
    for (int i = 0; i < NV; i++) {
      const int len = (int)tw(m.o_glen + i);
      double acc0[M], acc1[M];
#pragma unroll
      for (int q = 0; q < M; q++) acc0[q] = acc1[q] = 0.0;
      if (L == 1) { /* one entry per word: double coefficient, low 16 mantissa bits = q offset (a constant-bank operand) */
        for (int t = 0; t < len; t++, gp += L) {
          const unsigned long long w = tw(gp);
          const double coef = __longlong_as_double((long long)(w & ~0xFFFFull));
          const unsigned o = (unsigned)w & 0xFFFFu;
#pragma unroll
          for (int q = 0; q < M; q++)
            acc0[q] = fma(coef, *reinterpret_cast<const double *>(reinterpret_cast<const char *>(sQ + q * RS) + o), acc0[q]);
        }
      } else if (L < CKB_NEGQ_L) { /* two entries per word: (sign of the coefficient in bit 31) | q offset; the sign is
                  XOR-ed into q (exactly fma(+-1, q, acc)); |nu| > 1 is entered |nu| times, an idle entry reads a 0.0 slot */
        for (int t = 0; t < len; t++, gp += L) {
          const unsigned long long w = tw(gp);
          const unsigned lo = (unsigned)w, hi = (unsigned)(w >> 32);
          const unsigned o0 = lo & 0xFFFFu, o1 = hi & 0xFFFFu;
#pragma unroll
          for (int q = 0; q < M; q++) {
            const char *qb = reinterpret_cast<const char *>(sQ + q * RS);
            const double q0 = *reinterpret_cast<const double *>(qb + o0), q1 = *reinterpret_cast<const double *>(qb + o1);
            acc0[q] += __hiloint2double(__double2hiint(q0) ^ (int)(lo & 0x80000000u), __double2loint(q0));
            acc1[q] += __hiloint2double(__double2hiint(q1) ^ (int)(hi & 0x80000000u), __double2loint(q1));
          }
        }
      } else { /* four entries per word, each the byte offset of q_s (coefficient +1), of -q_s (coefficient -1: the slot
                  loop stores both) or of one of the 0.0 slots behind them (idle entry): an extract, a shared read and
                  an add per entry; |nu| > 1 is entered |nu| times */
        double acc2[M], acc3[M];
#pragma unroll
        for (int q = 0; q < M; q++) acc2[q] = acc3[q] = 0.0;
        for (int t = 0; t < len; t++, gp += L) {
          const unsigned long long w = tw(gp);
          const unsigned lo = (unsigned)w, hi = (unsigned)(w >> 32);
#pragma unroll
          for (int q = 0; q < M; q++) {
            const char *qb = reinterpret_cast<const char *>(sQ + q * RS);
            acc0[q] += *reinterpret_cast<const double *>(qb + (lo & 0xFFFFu));
            acc1[q] += *reinterpret_cast<const double *>(qb + (lo >> 16));
            acc2[q] += *reinterpret_cast<const double *>(qb + (hi & 0xFFFFu));
            acc3[q] += *reinterpret_cast<const double *>(qb + (hi >> 16));
          }
        }
#pragma unroll
        for (int q = 0; q < M; q++) {
          acc0[q] += acc2[q];
          acc1[q] += acc3[q];
        }
      }
#pragma unroll
      for (int q = 0; q < M; q++) om[q][i] = acc0[q] + acc1[q];
    }
    if (L > 1 && m.o_split) { /* launch-uniform: the tails of the longest rows were summed in the last level's spare slots
                                 (ckb_pack.cu); a component takes its tail from the lane that holds it */
      double tail[M][NV];
#pragma unroll
      for (int i = 0; i < NV; i++) {
        const int src = (int)tw(m.o_split + i * L + g);
#pragma unroll
        for (int q = 0; q < M; q++) {
          const double t = __shfl_sync(mask, om[q][NV - 1], src < 0 ? src0 : src0 + src);
          tail[q][i] = src < 0 ? 0.0 : t;
        }
      }
#pragma unroll
      for (int i = 0; i < NV; i++)
#pragma unroll
        for (int q = 0; q < M; q++) om[q][i] += tail[q][i];
      if (g + L * (NV - 1) >= n) { /* a spare slot has handed its sum over: it is no component (its h - 1 is not 0 at constant volume) */
#pragma unroll
        for (int q = 0; q < M; q++) om[q][NV - 1] = 0.0;
      }
    }
#pragma unroll
    for (int i = 0; i < NV; i++) {
      const double W = td(m.o_sp + i * CKB_SP_WORDS * L + g + CKB_SP_W * L);
#pragma unroll
      for (int q = 0; q < M; q++) {
        f[q][i] = W * om[q][i] * invrho[q];
        s3[q] = fma(L == 1 ? sH[i * GI] : hrt[q][i], om[q][i], s3[q]);
      }
    }
#pragma unroll
    for (int o = L / 2; o > 0; o >>= 1) {
#pragma unroll
      for (int q = 0; q < M; q++) s3[q] += __shfl_xor_sync(mask, s3[q], o);
    }
    /* Eq. 6: dT/dt = -(Ru T sum_k (h_k/RT) omega_k) / (rho cp), cp = Ru sum_k Y_k (cp_k/R) / W_k;
     * R29: dT/dt = -(Ru T sum_k (h_k/RT - 1) omega_k) / (rho c_v), c_v = cp - Ru sum_k Y_k / W_k */
    if (g == 0) {
#pragma unroll
      for (int q = 0; q < M; q++)
        f[q][0] = (L > 1) ? -(T[q] * s3[q] * invrho[q]) * rcp_c[q] : -(T[q] * s3[q] * invrho[q]) / (CV ? s2[q] - s1[q] : s2[q]);
    }
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

/* ================================================================================================
 * Integrators as state machines with ONE call site of f(y).
 *
 * Each integrator object holds the whole per-system controller state in registers.  The kernel loop is
 *     while (work) { f = rhs(integ.w);  done = integ.advance(f); }
 * so that (a) the source term -- > 90 % of the instructions -- is inlined once, and (b) in the
 * thread-per-ODE mapping all lanes of a warp evaluate f(y) together whatever sub-step, stage or
 * power-method iteration each of them is in: divergence is confined to the short vector updates
 * between two evaluations (the paper's divergence sources, made harmless).
 * The arithmetic and the order of the controller decisions follow DESIGN.md section 4 step by step.
 * ============================================================================================== */

/* A stage vector that lives in registers, or -- for thread-per-ODE, where registers per thread are what limits
 * the resident warps -- in the system's shared scratch area sX (interleaved like the region: conflict free). */
template <class S, int SLOT, bool IN_SMEM>
struct XVec {
  double r[IN_SMEM ? 1 : S::NV];
  __device__ __forceinline__ double get(const S &sys, int i) const {
    if (IN_SMEM) return sys.sX[(SLOT * S::NV + i) * S::GI];
    return r[IN_SMEM ? 0 : i];
  }
  __device__ __forceinline__ void set(const S &sys, int i, double x) {
    if (IN_SMEM) sys.sX[(SLOT * S::NV + i) * S::GI] = x;
    else r[IN_SMEM ? 0 : i] = x;
  }
};

/* RKCK: Eq. 7-17, Table 1; R1-R7, R25. */
template <class S>
struct Rkck {
  static constexpr int NV = S::NV;
  /* Table 1 (R1: Cash-Karp values) */
  static constexpr double B21 = 1.0 / 5.0;
  static constexpr double B31 = 3.0 / 40.0, B32 = 9.0 / 40.0;
  static constexpr double B41 = 3.0 / 10.0, B42 = -9.0 / 10.0, B43 = 6.0 / 5.0;
  static constexpr double B51 = -11.0 / 54.0, B52 = 5.0 / 2.0, B53 = -70.0 / 27.0, B54 = 35.0 / 27.0;
  static constexpr double B61 = 1631.0 / 55296.0, B62 = 175.0 / 512.0, B63 = 575.0 / 13824.0,
                          B64 = 44275.0 / 110592.0, B65 = 253.0 / 4096.0;
  static constexpr double C1 = 37.0 / 378.0, C3 = 250.0 / 621.0, C4 = 125.0 / 594.0, C6 = 512.0 / 1771.0;
  static constexpr double D1 = C1 - 2825.0 / 27648.0, D3 = C3 - 18575.0 / 48384.0,
                          D4 = C4 - 13525.0 / 55296.0, D5 = -277.0 / 14336.0, D6 = C6 - 1.0 / 4.0;
  static constexpr double SAFETY = 0.9;

  double w[NV];                 /* the next argument of f */
  static constexpr bool XS = (S::L == 1); /* k3..k5 in shared scratch */
  static constexpr bool XS12 = XS && (CKB_XS_RKCK_K12 != 0); /* k1, k2 as well (specialised kernels: 4 blocks per SM) */
  static constexpr int XDOUBLES = XS ? (XS12 ? 5 : 3) * NV : 0;
  double y[NV];
  XVec<S, 3, XS12> k1;
  XVec<S, 4, XS12> k2;
  XVec<S, 0, XS> k3;
  XVec<S, 1, XS> k4;
  XVec<S, 2, XS> k5;
  double t, h, t1, rtol, atol;
  int stage, nfe, nacc, nrej, attempts, status;
  bool last, saw_nonfinite;

  /* R5 clip, then either evaluate k1 (stage 1) or go on with the stages (k1 kept and rescaled, R25) */
  __device__ __forceinline__ void begin_attempt(const S &sys, bool have_k1) {
    last = false;
    if (1.1 * h >= t1 - t) {
      const double hn = t1 - t;
      if (have_k1) {
        const double r = hn / h;
#pragma unroll
        for (int i = 0; i < NV; i++) k1.set(sys, i, k1.get(sys, i) * r);
      }
      h = hn;
      last = true;
    }
    if (!have_k1) {
      stage = 1;
#pragma unroll
      for (int i = 0; i < NV; i++) w[i] = y[i];
    } else {
      start_stages(sys);
    }
  }
  __device__ __forceinline__ void start_stages(const S &sys) {
    if (++attempts > 1000000) { /* R7 */
      status = ST_MAXSTEPS;
      stage = 0;
      return;
    }
    stage = 2;
#pragma unroll
    for (int i = 0; i < NV; i++) w[i] = fma(B21, k1.get(sys, i), y[i]);
  }

  __device__ __forceinline__ void start(const S &sys, const double (&y0)[NV], double t0_, double t1_, double rtol_,
                                        double atol_, int /*n*/) {
#pragma unroll
    for (int i = 0; i < NV; i++) y[i] = y0[i];
    t = t0_; t1 = t1_; rtol = rtol_; atol = atol_;
    h = t1_ - t0_; /* R4 */
    nfe = nacc = nrej = attempts = 0;
    status = ST_OK;
    saw_nonfinite = false;
    begin_attempt(sys, false);
  }

  /* consume f = f(w); returns true when the system has reached t1 (or failed) */
  __device__ __forceinline__ bool advance(const S &sys, const double (&f)[NV]) {
    nfe++;
    switch (stage) {
      case 1: /* Eq. 7 */
#pragma unroll
        for (int i = 0; i < NV; i++) k1.set(sys, i, h * f[i]);
        start_stages(sys);
        return stage == 0;
      case 2:
#pragma unroll
        for (int i = 0; i < NV; i++) {
          const double k2i = h * f[i];
          k2.set(sys, i, k2i);
          w[i] = fma(B32, k2i, fma(B31, k1.get(sys, i), y[i]));
        }
        stage = 3;
        return false;
      case 3:
#pragma unroll
        for (int i = 0; i < NV; i++) {
          const double k3i = h * f[i];
          k3.set(sys, i, k3i);
          w[i] = fma(B43, k3i, fma(B42, k2.get(sys, i), fma(B41, k1.get(sys, i), y[i])));
        }
        stage = 4;
        return false;
      case 4:
#pragma unroll
        for (int i = 0; i < NV; i++) {
          const double k4i = h * f[i], k3i = k3.get(sys, i);
          k4.set(sys, i, k4i);
          w[i] = fma(B54, k4i, fma(B53, k3i, fma(B52, k2.get(sys, i), fma(B51, k1.get(sys, i), y[i]))));
        }
        stage = 5;
        return false;
      case 5:
#pragma unroll
        for (int i = 0; i < NV; i++) {
          const double k5i = h * f[i], k3i = k3.get(sys, i), k4i = k4.get(sys, i);
          k5.set(sys, i, k5i);
          w[i] = fma(B65, k5i, fma(B64, k4i, fma(B63, k3i, fma(B62, k2.get(sys, i), fma(B61, k1.get(sys, i), y[i])))));
        }
        stage = 6;
        return false;
      default:
        break;
    }
    /* stage 6: Eq. 13, 15, 16 (R2), 17 (R3) */
    double errmax = 0.0;
#pragma unroll
    for (int i = 0; i < NV; i++) {
      const double k6 = h * f[i];
      const double k3i = k3.get(sys, i), k4i = k4.get(sys, i), k5i = k5.get(sys, i);
      const double k1i = k1.get(sys, i);
      const double yn = fma(C6, k6, fma(C4, k4i, fma(C3, k3i, fma(C1, k1i, y[i]))));
      const double dl = fma(D6, k6, fma(D5, k5i, fma(D4, k4i, fma(D3, k3i, D1 * k1i))));
      w[i] = yn;
      if (sys.valid(i)) {
        const double d0 = fma(rtol, fabs(y[i]) + fabs(k1i), atol);
        double e = fabs(dl) / d0;
        if (!isfinite(yn) || isnan(e)) e = __longlong_as_double(0x7ff0000000000000LL); /* +inf */
        errmax = fmax(errmax, e);
      }
    }
    errmax = sys.gmax(errmax);
    if (errmax <= 1.0) { /* P:139 accept */
      nacc++;
#pragma unroll
      for (int i = 0; i < NV; i++) y[i] = w[i];
      if (last) return true;
      t += h;
      double fac = (errmax > 0.0) ? SAFETY * pow(errmax, -0.2) : 5.0;
      if (fac > 5.0) fac = 5.0;
      h *= fac;
      begin_attempt(sys, false);
      return false;
    }
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
    for (int i = 0; i < NV; i++) k1.set(sys, i, k1.get(sys, i) * fac); /* R25 */
    h *= fac;
    const double tmax = fmax(fabs(t), fabs(t1));
    if (!(h > 10.0 * CKB_U * tmax)) { /* R6 */
      status = saw_nonfinite ? ST_NONFINITE : ST_UNDERFLOW;
      return true;
    }
    begin_attempt(sys, true);
    return stage == 0;
  }

  __device__ __forceinline__ double y_at(const S &, int i) const { return y[i]; }
  __device__ __forceinline__ void result(int (&st)[4]) const {
    st[0] = nfe; st[1] = nacc; st[2] = nrej; st[3] = 0;
  }
};

/* RKC coefficients of stage j (2 <= j <= s) of an s-stage step, Eq. 22-26 with R8-R10, computed from scratch
 * (O(s) scalar work; used only above the precomputed table, s > s_tab, where f(y) costs far more). */
static __device__ __noinline__ void rkc_coefficients(int s, int j, double &mut1, double &mu, double &nu, double &mut,
                                              double &gamt) {
  const double w0 = 1.0 + (2.0 / 13.0) / ((double)s * (double)s);
  double Tm2 = 1.0, Tm1 = w0, dm2 = 0.0, dm1 = 1.0, em2 = 0.0, em1 = 0.0;
  double b2 = 0.0, bj = 0.0, bjm1 = 0.0, bjm2 = 0.0, Tjm1 = w0;
  for (int q = 2; q <= s; q++) {
    const double Tq = 2.0 * w0 * Tm1 - Tm2;
    const double dq = 2.0 * Tm1 + 2.0 * w0 * dm1 - dm2;
    const double eq = 4.0 * dm1 + 2.0 * w0 * em1 - em2;
    if (q == 2) b2 = eq / (dq * dq);
    if (q == j - 2) bjm2 = eq / (dq * dq);
    if (q == j - 1) { bjm1 = eq / (dq * dq); Tjm1 = Tq; }
    if (q == j) bj = eq / (dq * dq);
    Tm2 = Tm1; Tm1 = Tq; dm2 = dm1; dm1 = dq; em2 = em1; em1 = eq;
  }
  const double w1 = dm1 / em1; /* Eq. 25 */
  if (j - 2 < 2) bjm2 = b2;    /* R10: b_0 = b_1 = b_2 */
  if (j - 1 < 2) { bjm1 = b2; Tjm1 = w0; }
  const double ajm1 = 1.0 - bjm1 * Tjm1; /* R9 */
  mut1 = b2 * w1;
  mu = 2.0 * bj * w0 / bjm1;
  nu = -bj / bjm2;
  mut = 2.0 * bj * w1 / bjm1;
  gamt = -ajm1 * mut;
}

/* RKC: Eq. 18-39 and P:233; R8-R18, R26.  Spectral radius by the nonlinear power method (R17/R18). */
template <class S>
struct Rkc {
  static constexpr int NV = S::NV;
  enum { S_F0 = 1, S_PM = 2, S_H0 = 3, S_STAGE = 4, S_FINAL = 5 };

  double w[NV];                                   /* the next argument of f: y, z (power method), w_{j-1} */
  static constexpr bool XS = (S::L == 1); /* eigenvector estimate v in shared scratch */
  static constexpr bool XSF = XS && (CKB_XS_RKC_F0 != 0); /* f0 and w_{j-2} as well (specialised kernels) */
  static constexpr bool XSY = XSF && (CKB_XS_RKC_Y != 0); /* and y */
  static constexpr int XDOUBLES = XS ? (XSY ? 4 : XSF ? 3 : 1) * NV : 0;
  XVec<S, 3, XSY> y;
  XVec<S, 1, XSF> f0;
  XVec<S, 2, XSF> wjm2;
  XVec<S, 0, XS> v;
  double t, h, t1, Dt, rtol, atol, nd;
  double sigma, err_old, h_old;                   /* err_old: CUBE ROOT of the previous accepted step's error norm */
  double pm_d, pm_sigma;                          /* power method: displacement size, last estimate */
  int state, j, s, s_max, pm_it, cbase;           /* cbase: this step's rows of the coefficient table */
  int nfe, nacc, nrej, smax_used, attempts, since_sigma, status, flag;
  bool last, have_prev, saw_nonfinite, sigma_fresh, need_sigma, pm_initial;

  __device__ __forceinline__ void start(const S &sys, const double (&y0)[NV], double t0_, double t1_, double rtol_,
                                        double atol_, int n) {
#pragma unroll
    for (int i = 0; i < NV; i++) {
      y.set(sys, i, y0[i]);
      w[i] = y0[i];
    }
    t = t0_; t1 = t1_; Dt = t1_ - t0_; rtol = rtol_; atol = atol_; nd = (double)n;
    s_max = (int)floor(sqrt(rtol_ / (10.0 * CKB_U)) + 0.5); /* R12 */
    if (s_max < 2) s_max = 2;
    nfe = nacc = nrej = smax_used = attempts = since_sigma = 0;
    status = ST_OK; flag = 0;
    have_prev = saw_nonfinite = need_sigma = false;
    sigma_fresh = true;
    err_old = h_old = 0.0;
    state = S_F0;
  }

  /* power method set-up: place z at distance d from y along v (R17 step 2) */
  __device__ __forceinline__ void pm_begin(const S &sys, bool have_v, bool initial) {
    if (!have_v) {
#pragma unroll
      for (int i = 0; i < NV; i++) v.set(sys, i, f0.get(sys, i));
    }
    double a = 0.0, b = 0.0;
#pragma unroll
    for (int i = 0; i < NV; i++) {
      a = fma(y.get(sys, i), y.get(sys, i), a);
      const double vi = v.get(sys, i);
      b = fma(vi, vi, b);
    }
    const double ynrm = sqrt(sys.gsum(a)), vnrm = sqrt(sys.gsum(b));
    if (ynrm != 0.0 && vnrm != 0.0) {
      pm_d = ynrm * CKB_SQRTU;
      const double r = pm_d / vnrm;
#pragma unroll
      for (int i = 0; i < NV; i++) w[i] = fma(v.get(sys, i), r, y.get(sys, i));
    } else if (ynrm != 0.0) {
      pm_d = ynrm * CKB_SQRTU;
#pragma unroll
      for (int i = 0; i < NV; i++) w[i] = y.get(sys, i) * (1.0 + CKB_SQRTU);
    } else if (vnrm != 0.0) {
      pm_d = CKB_U;
      const double r = pm_d / vnrm;
#pragma unroll
      for (int i = 0; i < NV; i++) w[i] = v.get(sys, i) * r;
    } else {
      pm_d = CKB_U;
#pragma unroll
      for (int i = 0; i < NV; i++) w[i] = sys.valid(i) ? pm_d : 0.0;
    }
    pm_sigma = 0.0;
    pm_it = 1;
    pm_initial = initial;
    state = S_PM;
  }

  /* R5 clip, R16 refresh check (the clip is not redone after a refresh) */
  __device__ __forceinline__ bool begin_step(const S &sys) {
    last = false;
    if (1.1 * h >= t1 - t) {
      h = t1 - t;
      last = true;
    }
    if (need_sigma) {
      pm_begin(sys, true, false);
      return false;
    }
    return take_step(sys);
  }

  /* Eq. 39 (R12), coefficients for j = 1, 2 (Eq. 22-26, R8-R10), first stage Eq. 19; true = failed */
  __device__ __forceinline__ bool take_step(const S &sys) {
    {
      const double x39 = fma(1.54 * h, sigma, 1.0);
      /* x < 4 (and NaN: the cast of NaN is 0): floor(sqrt(x)) <= 1, so s = 2 without the square root */
      s = (x39 >= 4.0) ? 1 + (int)floor(sqrt(x39)) : 2;
    }
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
      rkc_coefficients(s, 2, mut1, mu, nu, mut, gamt);
      cbase = -1;
    }
    const double mh = mut1 * h;
#pragma unroll
    for (int i = 0; i < NV; i++) {
      wjm2.set(sys, i, y.get(sys, i));
      w[i] = fma(mh, f0.get(sys, i), y.get(sys, i)); /* Eq. 19 */
    }
    j = 2;
    state = S_STAGE;
    return false;
  }

  __device__ __forceinline__ bool advance(const S &sys, const double (&f)[NV]) {
    nfe++;
    switch (state) {
      case S_F0: {
#pragma unroll
        for (int i = 0; i < NV; i++) f0.set(sys, i, f[i]);
        pm_begin(sys, false, true);
        return false;
      }
      case S_PM: { /* R17 step 3-5 */
        double dd = 0.0;
#pragma unroll
        for (int i = 0; i < NV; i++) {
          const double e = f[i] - f0.get(sys, i);
          dd = fma(e, e, dd);
        }
        dd = sqrt(sys.gsum(dd));
        const double sigma_prev = pm_sigma;
        pm_sigma = dd / pm_d;
        const double fl = pm_sigma > 1e-300 ? pm_sigma : 1e-300;
        const bool conv = pm_it >= 2 && fabs(pm_sigma - sigma_prev) <= 0.01 * fl;
        if (!conv && pm_it < 50) {
          if (dd != 0.0) {
            const double r = pm_d / dd;
#pragma unroll
            for (int i = 0; i < NV; i++) w[i] = fma(f[i] - f0.get(sys, i), r, y.get(sys, i));
          } else {
            const int ci = pm_it % (int)nd; /* an ORIGINAL state row (0 = T, 1 + species), as in the oracle */
#pragma unroll
            for (int i = 0; i < NV; i++)
              if (sys.valid(i) && (int)sys.tw(sys.m.o_perm + sys.g + S::L * i) == ci) w[i] = y.get(sys, i) - (w[i] - y.get(sys, i));
          }
          pm_it++;
          return false;
        }
        if (!conv) {
          flag = ST_SIGMA;
          /* R17: z is updated once more after the 50th evaluation before v is saved */
          if (dd != 0.0) {
            const double r = pm_d / dd;
#pragma unroll
            for (int i = 0; i < NV; i++) w[i] = fma(f[i] - f0.get(sys, i), r, y.get(sys, i));
          } else {
            const int ci = pm_it % (int)nd; /* an ORIGINAL state row (0 = T, 1 + species), as in the oracle */
#pragma unroll
            for (int i = 0; i < NV; i++)
              if (sys.valid(i) && (int)sys.tw(sys.m.o_perm + sys.g + S::L * i) == ci) w[i] = y.get(sys, i) - (w[i] - y.get(sys, i));
          }
        }
#pragma unroll
        for (int i = 0; i < NV; i++) v.set(sys, i, w[i] - y.get(sys, i));
        sigma = 1.2 * pm_sigma; /* R18 */
        sigma_fresh = true;
        need_sigma = false;
        since_sigma = 0;
        if (!pm_initial) return take_step(sys);
        /* initial step, Eq. 36-37 (R14, R15): probe f(y + h0 f0) */
        h_old = (sigma > 0.0 && 1.0 / sigma < Dt) ? 1.0 / sigma : Dt; /* h0, parked in h_old */
#pragma unroll
        for (int i = 0; i < NV; i++) w[i] = fma(h_old, f0.get(sys, i), y.get(sys, i));
        state = S_H0;
        return false;
      }
      case S_H0: { /* Eq. 37-38 */
        const double h0 = h_old;
        double acc = 0.0;
#pragma unroll
        for (int i = 0; i < NV; i++) {
          if (sys.valid(i)) {
            const double d0 = h0 * (f[i] - f0.get(sys, i));
            const double wt = fma(rtol, fabs(y.get(sys, i)), atol);
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
          rkc_coefficients(s, j, mut1, mu, nu, mut, gamt);
        }
        const double c0 = 1.0 - mu - nu, mh = mut * h, gh = gamt * h;
#pragma unroll
        for (int i = 0; i < NV; i++) {
          const double wj = fma(gh, f0.get(sys, i), fma(mh, f[i], fma(nu, wjm2.get(sys, i), fma(mu, w[i], c0 * y.get(sys, i)))));
          wjm2.set(sys, i, w[i]);
          w[i] = wj;
        }
        if (++j > s) state = S_FINAL;
        return false;
      }
      default:
        break;
    }
    /* S_FINAL: f = f(y_{n+1}), y_{n+1} = w.  Eq. 30-35 */
    double acc = 0.0;
#pragma unroll
    for (int i = 0; i < NV; i++) {
      if (sys.valid(i)) {
        const double del = fma(0.8, y.get(sys, i) - w[i], 0.4 * h * (f0.get(sys, i) + f[i]));
        const double wt = fma(rtol, fmax(fabs(y.get(sys, i)), fabs(w[i])), atol);
        const double q = del / wt;
        acc = fma(q, q, acc);
      }
    }
    const double err = sqrt(sys.gsum(acc) / nd);
    if (err <= 1.0) {
      nacc++;
      double fac;
      double e3 = 0.0;
      if (err > 0.0) {
        e3 = cbrt(err);
        if (have_prev) fac = (0.8 * err_old * h) / (e3 * e3 * h_old); /* Eq. 34, R13 (err_old = cbrt of that error): one division */
        else fac = 0.8 / e3;
      } else fac = 10.0; /* R26 */
      fac = fmin(10.0, fmax(0.1, fac)); /* Eq. 33 */
#pragma unroll
      for (int i = 0; i < NV; i++) {
        y.set(sys, i, w[i]);
        f0.set(sys, i, f[i]);
      }
      err_old = e3; /* the cube root is what Eq. 34 needs next time (cbrt(0) = 0 as well) */
      h_old = h;
      have_prev = true;
      sigma_fresh = false;
      if (++since_sigma >= 25) need_sigma = true;
      if (last) return true;
      t += h;
      h *= fac;
      return begin_step(sys);
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
    if (!sigma_fresh) need_sigma = true; /* R16 */
    const double tmax = fmax(fabs(t), fabs(t1));
    if (!(h > 10.0 * CKB_U * tmax)) {
      status = saw_nonfinite ? ST_NONFINITE : ST_UNDERFLOW;
      return true;
    }
    return begin_step(sys);
  }

  __device__ __forceinline__ double y_at(const S &sys, int i) const { return y.get(sys, i); }
  /* what the next advance() will do: 3 = error estimate, 2 = last stage of a step, 1 = earlier stage, 0 = other */
  __device__ __forceinline__ int phase() const {
    return state == S_FINAL ? 3 : state == S_STAGE ? (j == s ? 2 : 1) : 0;
  }
  __device__ __forceinline__ void result(int (&st)[4]) {
    if (status == ST_OK && flag) status = flag;
    st[0] = nfe; st[1] = nacc; st[2] = nrej; st[3] = smax_used;
  }
};

/* ------------------------------------------------------------------------------------------------
 * Kernels.  Block = CKB_BLOCK threads; a warp holds G = 32/L systems at a time.
 * Shared memory per warp: (region_doubles(m) + scratch) * G * M doubles (ckb_tables.h).
 *
 * integrate_kernel is persistent: the grid is sized to the resident capacity of the GPU (a multiple of the
 * SM count) and every group of L lanes pulls system indices -- first its own global group index, then
 * from an atomic counter -- until the batch is exhausted.  In the thread-per-ODE mapping this is "lane
 * refill": a lane whose system has finished fetches the next one while its warp neighbours are still
 * sub-stepping, so finished lanes never idle behind a slow neighbour (divergence control).
 * ---------------------------------------------------------------------------------------------- */
#ifndef CKB_BLOCK
#define CKB_BLOCK 128
#endif
#ifndef CKB_MINB
#define CKB_MINB 1 /* resident blocks per SM the register allocation must allow (set per instantiation) */
#endif
#ifndef CKB_MINB_RKC
#define CKB_MINB_RKC CKB_MINB /* the same for the RKC kernels (more controller state) */
#endif

template <class S>
__device__ __forceinline__ void sys_setup(S &sys, const DevMech &m, double *smem, int xdoubles) {
  constexpr int L = S::L, G = S::G, M = S::M;
  /* a one-warp block (CKB_BLOCK == 32) has its shared region at a compile-time address: every runtime-indexed
   * shared read is then [offset + immediate], without the add of a per-warp base */
  const int lane = threadIdx.x & 31, warp = (CKB_BLOCK == 32) ? 0 : (threadIdx.x >> 5);
  const int grp = lane / L;
  sys.g = lane % L;
  sys.src0 = grp * L;
  sys.mask = (L == 32) ? 0xffffffffu : (((1u << L) - 1u) << (grp * L));
  constexpr int GI = S::GI;
#if CKB_EXP_TABLE
  ckb_exp_table_init();
#endif
#ifdef CKB_GEN_RHS
  const int region = 0; /* generated f(y): only the integrator's scratch lives in shared memory */
#else
  const int region = region_doubles(m);
#endif
  sys.RS = (region + xdoubles) * GI;
  sys.qoff = (m.n + m.NTB + 1) * GI;
  /* per warp: G groups x M systems x (region + scratch); interleaved by lane (GI = 32) or one after the other */
  sys.sR = smem + (size_t)warp * (region + xdoubles) * G * M + (GI == 1 ? grp * sys.RS * M : grp);
  sys.sX = sys.sR + region * GI;
  sys.sH = sys.sX + (xdoubles - S::HDOUBLES) * GI;
#ifndef CKB_GEN_RHS
  if (sys.g == 0) {
#pragma unroll
    for (int q = 0; q < M; q++) {
      sys.sR[q * sys.RS] = 1.0;                          /* "absent molecule" concentration */
      sys.sR[q * sys.RS + (m.n + m.NTB) * GI] = 1.0;     /* "no third body" */
    }
  }
  if (L > 1 && sys.g < CKB_ZERO_SLOTS) { /* the operands of idle gather entries (a group has >= 2 lanes: loop) */
    for (int z = sys.g; z < CKB_ZERO_SLOTS; z += L) {
#pragma unroll
      for (int q = 0; q < M; q++) sys.sR[q * sys.RS + sys.qoff + (L == CKB_NEGQ_L ? 2 : 1) * m.NSR * L + z] = 0.0;
    }
  }
#endif
  sys.gsync();
}

template <class S, int METHOD>
struct IntegratorOf { typedef Rkck<S> type; };
template <class S>
struct IntegratorOf<S, 1> { typedef Rkc<S> type; };

#ifndef CKB_TMEM_BLOCK
#define CKB_TMEM_BLOCK 512 /* TM = 1: one block per SM owns the SM's tensor memory; 512 threads x 128 registers */
#endif

/* TM = 1 (only where the object is compiled with CKB_TMEM): the slot table is read from tensor memory. */
template <int L, int NV, class TAB, int METHOD, int M, int CV = 0, int TM = 0>
__global__ void __launch_bounds__(TM ? CKB_TMEM_BLOCK : CKB_BLOCK, TM ? 1 : (METHOD == 0 ? CKB_MINB : CKB_MINB_RKC))
integrate_kernel(const __grid_constant__ DevMech m, const __grid_constant__ TAB tab, double *__restrict__ states,
                 const double *__restrict__ pressure, double p_uniform, long long N, long long ld, double t0,
                 double dt, double rtol, double atol, int *__restrict__ status, int *__restrict__ stats,
                 unsigned long long *__restrict__ counter, const int *__restrict__ order) {
  extern __shared__ double smem[];
  typedef Sys<L, NV, TAB, M, CV> S;
  S sys(m, tab);
  sys_setup(sys, m, smem, IntegratorOf<S, METHOD>::type::XDOUBLES + S::HDOUBLES);
  constexpr int G = S::G;
  constexpr int BLOCK = TM ? CKB_TMEM_BLOCK : CKB_BLOCK;
#if CKB_TMEM
  /* slot table -> tensor memory: warp 0 allocates the SM's 512 columns (one block per SM: the launch bounds fill the
   * register file), warps 0..3 copy the table into their lane quarter, every warp then reads its own quarter */
  __shared__ unsigned tm_holder;
  unsigned tm_base = 0;
  sys.tm_on = (TM != 0) && (L == 32) && m.NSR * 16 <= CKB_TMEM_COLS;
  if (sys.tm_on) {
    const int warp = threadIdx.x >> 5;
    if (warp == 0) tm_alloc(&tm_holder);
    tm_fence_sync_fence();
    tm_base = *reinterpret_cast<volatile unsigned *>(&tm_holder);
    sys.tm_addr = tm_base + ((unsigned)((warp & 3) * 32) << 16);
    if (warp < 4) {
      for (int r = 0; r < m.NSR; r++) {
        unsigned v[16];
#pragma unroll
        for (int x = 0; x < CKB_SL_WORDS; x++) {
          const unsigned long long w = sys.tw(m.o_sl + (r * CKB_SL_WORDS + x) * L + sys.g);
          v[2 * x] = (unsigned)w;
          v[2 * x + 1] = (unsigned)(w >> 32);
        }
        tm_st16(sys.tm_addr + (unsigned)r * 16u, v);
      }
      tm_wait_st();
    }
    tm_fence_sync_fence();
  }
#endif
  /* queue positions: every group starts with one of its own, then pulls from the counter.  One system per group (M = 1):
   * the loop state is kept in scalars -- as arrays indexed by the system of the group it stayed in local memory (flags,
   * counters and a pointer were re-read from the stack on every evaluation of f(y): ~5 % of the stall samples). */
  static_assert(M == 1, "integrate_kernel handles one system per group");
  const long long n_static = (long long)gridDim.x * (BLOCK / 32) * G;
  typename IntegratorOf<S, METHOD>::type integ;
  long long qi = ((long long)blockIdx.x * (BLOCK / 32) + (threadIdx.x >> 5)) * G + (threadIdx.x & 31) / L, ode = 0;
  bool need_load = true, active = true;
  double f[1][NV];
  sys.set_pressure(0, 1.0);
#pragma unroll
  for (int i = 0; i < NV; i++) integ.w[i] = 1.0; /* finite argument for a group that never gets a system */
  bool held_last = false;
  constexpr bool BALIGN = CKB_BLOCK_LOCKSTEP != 0 && METHOD == 1 && L < 32 && CKB_RKC_ALIGN != 0 && CKB_RKC_BLOCK_ALIGN != 0;
#if CKB_BLOCK_LOCKSTEP
  __shared__ unsigned ls_ph[64];
  unsigned ls_iter = 0;
#endif
  while (true) {
    if (need_load && active) {
      if (qi >= N) {
        active = false; /* queue exhausted: this group idles (its f(y) input stays at the last finite state) */
      } else {
        ode = order ? (long long)order[qi] : qi; /* queue position -> system */
        sys.set_pressure(0, pressure ? pressure[ode] : p_uniform);
        double y0[NV];
#pragma unroll
        for (int i = 0; i < NV; i++) {
          const int c = sys.g + L * i;
          y0[i] = (c < m.n) ? states[(size_t)sys.tw(m.o_perm + c) * ld + ode] : 0.0;
        }
        integ.start(sys, y0, t0, t0 + dt, rtol, atol, m.n);
        need_load = false;
      }
    }
    bool any = active;
    int b_last = 0, b_final = 0;
#if CKB_BLOCK_LOCKSTEP
    /* RKC: the warps of a block enter f(y) together (one instruction stream per block through the instruction caches:
     * the generated straight-line f(y) is larger than the 32 KB L1.5 I-cache) and leave the loop together.  RKCK runs
     * its warps independently: with the lanes of a warp stage-aligned its advance() is a few vector updates, and the
     * barrier cost more than the shared instruction stream saved (configs[1]: 9.32e8 -> 1.03e9 ODE/s without it; lock
     * step in 2, 3, 4, 6 groups of warps was measured in between; RKC loses 16 % with two groups already). */
    if constexpr (METHOD == 1) {
      const bool mine = any;
      if constexpr (BALIGN) { /* this warp's lanes in their last stage / at the error estimate, for the block-wide vote below */
        const int ph = active ? integ.phase() : 0;
        const unsigned w_last = __popc(__ballot_sync(0xffffffffu, ph == 2)), w_final = __popc(__ballot_sync(0xffffffffu, ph == 3));
        if ((threadIdx.x & 31) == 0) ls_ph[(ls_iter & 1) * 32 + (threadIdx.x >> 5)] = w_last | (w_final << 16);
      }
      any = __syncthreads_or(any);
      if constexpr (BALIGN) {
        const int lane = threadIdx.x & 31;
        const unsigned v = __reduce_add_sync(0xffffffffu, lane < BLOCK / 32 ? ls_ph[(ls_iter & 1) * 32 + lane] : 0u);
        b_last = (int)(v & 0xFFFFu);
        b_final = (int)(v >> 16);
        ls_iter++; /* double buffer: a warp writes its next counts while a slower one may still read these */
      }
      /* a warp that has run out of systems only keeps the barrier: the stragglers of the block get its issue slots */
      if (any && !__any_sync(0xffffffffu, mine)) continue;
    }
#endif
    if (!any) break;
    /* RKCK with several systems per warp (L < 32): keep the lanes of a warp in the same stage, so that the stage switch of advance() is
     * warp-uniform instead of up to six serialised paths.  Lanes only fall out of step at an attempt boundary:
     * after an accepted step (or a refill) the next evaluation is stage 1 (k1 = f(y)), after a rejection it is
     * stage 2 (k1 rescaled, R25).  When some lane needs stage 1, the stage-2 lanes sit that evaluation out (their
     * argument is evaluated again next time: same values, not counted). */
    bool hold = false;
    if constexpr (METHOD == 0 && L < 32 && CKB_RKCK_ALIGN != 0) {
      const bool s1 = active && integ.stage == 1;
      const bool any1 = __any_sync(0xffffffffu, s1); /* every lane votes */
      hold = active && !s1 && any1;
    }
    /* RKC with several systems per warp: a step with s stages is s - 1 stage evaluations (S_STAGE) and the evaluation of the error
     * estimate (S_FINAL); with lane refill and the occasional power-method excursion the lanes of a warp drift
     * into both at once, and advance() then runs both paths one after the other.  A lane in the minority sits one
     * evaluation out when that lines it up with the majority: S_FINAL lanes wait for lanes that are in their last
     * stage, last-stage lanes wait for S_FINAL lanes (which start their next step's stages afterwards).  Never
     * twice in a row, so no lane starves. */
    if constexpr (METHOD == 1 && L < 32 && CKB_RKC_ALIGN != 0) {
      const int ph = active ? integ.phase() : 0;
      /* block lock step: the vote is taken over the block, so that its warps reach the error estimate -- the long path of
       * advance(), which every warp waits for at the barrier -- on the same evaluations */
      const int n_last = BALIGN ? b_last : __popc(__ballot_sync(0xffffffffu, ph == 2));
      const int n_final = BALIGN ? b_final : __popc(__ballot_sync(0xffffffffu, ph == 3));
      hold = !held_last && ((ph == 3 && n_last > 0 && n_last >= n_final) || (ph == 2 && n_final > n_last));
      held_last = hold;
    }
    /* an idle group (queue exhausted) keeps evaluating its last argument: harmless, never stored */
    sys.rhs([&](int, int i) -> double { return integ.w[i]; }, f);
    if (active && !hold && integ.advance(sys, f[0])) {
      int st[4];
      integ.result(st);
#pragma unroll
      for (int i = 0; i < NV; i++) {
        const int c = sys.g + L * i;
        if (c < m.n) states[(size_t)sys.tw(m.o_perm + c) * ld + ode] = integ.y_at(sys, i);
      }
      if (sys.g == 0) {
        if (status) status[ode] = integ.status;
        if (stats) {
#pragma unroll
          for (int k = 0; k < 4; k++) stats[(size_t)k * N + ode] = st[k];
        }
      }
      /* next system: lane refill (L = 1) / group refill */
      unsigned long long nx = 0;
      if (sys.g == 0) nx = atomicAdd(counter, 1ull);
      if (L > 1) nx = __shfl_sync(sys.mask, nx, sys.src0);
      qi = n_static + (long long)nx;
      need_load = true;
    }
  }
#if CKB_TMEM
  if (sys.tm_on) {
    tm_fence_sync_fence(); /* every warp has left the loop */
    if ((threadIdx.x >> 5) == 0) tm_dealloc(tm_base);
  }
#endif
}

template <int L, int NV, class TAB, int CV = 0>
__global__ void __launch_bounds__(CKB_BLOCK)
rhs_kernel(const __grid_constant__ DevMech m, const __grid_constant__ TAB tab, const double *__restrict__ states,
           const double *__restrict__ pressure, double p_uniform, long long N, long long ld,
           double *__restrict__ dydt, int repeat) {
  extern __shared__ double smem[];
  typedef Sys<L, NV, TAB, 1, CV> S;
  S sys(m, tab);
  sys_setup(sys, m, smem, S::HDOUBLES);
  const long long ode = ((long long)blockIdx.x * (CKB_BLOCK / 32) + (threadIdx.x >> 5)) * S::G + (threadIdx.x & 31) / L;
  if (ode >= N) return;
  sys.set_pressure(0, pressure ? pressure[ode] : p_uniform);
  double y[1][NV], f[1][NV];
#pragma unroll
  for (int i = 0; i < NV; i++) {
    const int c = sys.g + L * i;
    y[0][i] = (c < m.n) ? states[(size_t)sys.tw(m.o_perm + c) * ld + ode] : 0.0;
  }
  for (int r = 0; r < repeat; r++) {
    sys.rhs([&](int, int i) -> double { return y[0][i]; }, f);
    if (r + 1 < repeat) {
      /* keep the repeats from being folded: feed a zero-weight dependence on f back into y */
#pragma unroll
      for (int i = 0; i < NV; i++) y[0][i] = fma(f[0][i], 0.0, y[0][i]);
    }
  }
#pragma unroll
  for (int i = 0; i < NV; i++) {
    const int c = sys.g + L * i;
    if (c < m.n) dydt[(size_t)sys.tw(m.o_perm + c) * ld + ode] = f[0][i];
  }
}

/* Cost proxy for the work-queue order of the thread-per-ODE RKC kernel: the number of sub-steps
 * an accuracy-limited RKC integration needs grows with the size of y'' = J f, so
 *     key_i = || (f(y + h f(y)) - f(y)) / (h wt) ||_rms,   wt = atol + rtol |y|
 * (two evaluations of f, a fraction of a percent of the integration) orders the queue far better than T does
 * (rank correlation with the true cost 0.79 against 0.27 on configs[2]). */
template <int L, int NV, class TAB, int CV = 0>
__global__ void __launch_bounds__(CKB_BLOCK)
cost_proxy_kernel(const __grid_constant__ DevMech m, const __grid_constant__ TAB tab,
                  const double *__restrict__ states, const double *__restrict__ pressure, double p_uniform,
                  long long N, long long ld, double h, double rtol, double atol, double *__restrict__ key) {
  extern __shared__ double smem[];
  typedef Sys<L, NV, TAB, 1, CV> S;
  S sys(m, tab);
  sys_setup(sys, m, smem, S::HDOUBLES);
  const long long ode = ((long long)blockIdx.x * (CKB_BLOCK / 32) + (threadIdx.x >> 5)) * S::G + (threadIdx.x & 31) / L;
  if (ode >= N) return;
  sys.set_pressure(0, pressure ? pressure[ode] : p_uniform);
  double y[NV], y1[NV], f0[1][NV], f1[1][NV];
#pragma unroll
  for (int i = 0; i < NV; i++) {
    const int c = sys.g + L * i;
    y[i] = (c < m.n) ? states[(size_t)sys.tw(m.o_perm + c) * ld + ode] : 0.0;
  }
  sys.rhs([&](int, int i) -> double { return y[i]; }, f0);
#pragma unroll
  for (int i = 0; i < NV; i++) y1[i] = fma(h, f0[0][i], y[i]);
  sys.rhs([&](int, int i) -> double { return y1[i]; }, f1);
  double acc = 0.0;
#pragma unroll
  for (int i = 0; i < NV; i++) {
    if (sys.valid(i)) {
      const double q = (f1[0][i] - f0[0][i]) / (h * fma(rtol, fabs(y[i]), atol));
      acc = fma(q, q, acc);
    }
  }
  acc = sys.gsum(acc);
  if (sys.g == 0) key[ode] = sqrt(acc / (double)m.n);
}

} /* namespace ckb */
