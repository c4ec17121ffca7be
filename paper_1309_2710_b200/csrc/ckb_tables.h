/*
 * ckb_tables.h -- layout of the packed mechanism, seen by the packer and the kernels.
 *
 * The mechanism is packed once per lanes-per-system value L (1, 8, 16, 32) because every table is
 * "blocked SoA with block L": entry x of item (r*L + g) sits at word (r*X + x)*L + g, so that the L lanes
 * of a group read X consecutive runs of L words with ONE address register and immediate offsets -- fully
 * coalesced for L = 32, a broadcast for L = 1 (kernel-parameter / constant bank).
 *
 * Components are renumbered: c = 0 is T, c = 1..K are the species sorted by the length of their gather
 * row (longest first), so that the rows handled in one gather level have similar lengths.
 * Shared-memory region of one system (in doubles; thread-per-ODE interleaves the 32 systems of a warp, element
 * e of lane l at [e*32 + l]; the lane-distributed mappings keep each system's region contiguous):
 *   [0, n)            C_c, concentration of component c; C_0 = 1.0 stands for "no molecule"
 *   [n, n+NTB+1)      [M]_t per third-body efficiency set; the last one = 1.0 stands for "no third body"
 *   [n+NTB+1, +NSR*L) q_s, net rate of progress of reaction slot s
 *   L = 32: then NSR*L doubles -q_s (so that the Eq. 3 gather applies a coefficient of +1 / -1 by WHERE it reads)
 *   L > 1: then 16 doubles of 0.0 (one per bank pair), the operand of an idle entry of the gather
 */
#pragma once
#ifndef __CUDACC__
#define __device__
#define __host__
#define __forceinline__ inline
#endif

namespace ckb {

/* Table sources.  ParamTab: the whole packed mechanism travels as a __grid_constant__ kernel parameter
 * (constant bank, broadcast reads; used by thread-per-ODE where every lane reads the same entry).
 * GlobalTab: device blob read through L1 (used when lanes read different entries). */
#define CKB_PARAM_WORDS 3072 /* 24 KB of kernel-parameter space */
struct ParamTab {
  unsigned long long w[CKB_PARAM_WORDS];
  __device__ __forceinline__ unsigned long long ld(int i) const { return w[i]; }
};
struct GlobalTab {
  const unsigned long long *p;
  __device__ __forceinline__ unsigned long long ld(int i) const {
#ifdef __CUDA_ARCH__
    return __ldg(p + i);
#else
    return p[i];
#endif
  }
};

/* species table: 13 words per component */
#define CKB_SP_INVW 0 /* 1/W                                   */
#define CKB_SP_W 1    /* W                                     */
#define CKB_SP_CP 2   /* 5 words: a1..a5 (cp/R)                */
#define CKB_SP_H 7    /* 6 words: a1, a2/2, .., a5/5, a6 (h/RT) */
#define CKB_SP_WORDS 13
/* slot table: 8 words per reaction slot */
#define CKB_SL_LNAF 0
#define CKB_SL_BF 1
#define CKB_SL_THF 2
#define CKB_SL_LNAR 3 /* -inf when the slot has no reverse reaction */
#define CKB_SL_BR 4
#define CKB_SL_THR 5
#define CKB_SL_IDXA 6 /* 16-bit fields: region BYTE offsets (x G) of reactant molecules 0,1,2 and of [M] */
#define CKB_SL_IDXB 7 /* 16-bit fields: product molecules 0,1,2; field 3 unused                              */
#define CKB_SL_WORDS 8

struct DevMech {
  int K, n;          /* species, unknowns (K+1)                                                           */
  int L;             /* lanes per system this packing is for                                              */
  int NV;            /* gather levels = ceil(n / L)                                                       */
  int NS, NSR;       /* reaction slots (fused forward/reverse pairs), slot rounds = ceil(NS / L)          */
  int NTB, NTBR, TBE;/* third-body sets, set rounds = ceil(NTB / L), listed entries per set (padded)      */
  int o_sp;          /* [NV][13][L]        species table                                                  */
  int o_sl;          /* [NSR][8][L]        slot table                                                     */
  int o_rflag;       /* [NSR]              round flags: 1 = a third molecule is read, 2 = a third body is read   */
  int o_tb;          /* [NTBR][TBE][2][L]  (alpha-1, region byte offset of the species)                        */
  int o_glen;        /* [NV]               64-bit words per lane of gather level i (uniform over lanes)   */
  int o_gat;         /* [sum glen][L]      gather entries.  L = 32: four per word, each the 16-bit BYTE offset inside
                                           the q region of q_s (coefficient +1), of -q_s (coefficient -1) or of a 0.0
                                           slot (idle).  1 < L < 32 (shared memory is what limits those mappings: no
                                           -q copies): two per word, (sign of the coefficient in bit 31) | BYTE offset
                                           of q_s.  |nu| > 1 is entered nu times.  L = 1: one per word, double
                                           coefficient with the offset in its low 16 bits */
  int o_rkc;         /* RKC coefficients for s = 2..s_tab: [s-2] -> mu~_1; stages at o_rkcs               */
  int o_rkcs;        /* [(s-2)(s-1)/2 + (j-2)][4] = mu_j, nu_j, mu~_j, gamma~_j, j = 2..s                  */
  int s_tab;
  int words;
  int o_perm;        /* [n] original state row (0 = T, 1 + species index) of component c                    */
  int o_fo;          /* [NTBR][8][L] fall-off description of efficiency set t (R31): kind (0 none, 1 Lindemann,
                        2 Troe, 3 Troe without T**), ln A_0 - ln A_inf, beta_0 - beta_inf, (E_0 - E_inf)/R_c,
                        a, 1/T***, 1/T*, T**; 0 = the mechanism has no fall-off reaction                     */
  int o_split;       /* [NV][L] L > 1: lane whose LAST gather level holds the second part of this component's Eq. 3 row, or
                        -1 (ckb_pack.cu: the NV*L - n register slots without a component take the tails of the longest
                        rows, so that no row is longer than the (NV*L - n + 1)-th longest); 0 = no row is split    */
  int o_sp2;         /* [NV][13][L] second species table: the high temperature range of the NASA fits, with
                        T_mid in the CKB_SP_INVW word (W word unused); 0 = the mechanism has one range       */
};

/* doubles of shared memory per system: C region, [M] region, q region */
#define CKB_ZERO_SLOTS 16 /* L > 1: 0.0 in every bank pair behind the q region, read by idle gather entries */
#define CKB_NEGQ_L 32     /* the mapping whose slot loop stores -q_s beside q_s (warp-per-ODE) */
__host__ __device__ __forceinline__ int region_doubles(const DevMech &m) {
  return m.n + m.NTB + 1 + m.NSR * m.L + (m.L == CKB_NEGQ_L ? m.NSR * m.L : 0) + (m.L > 1 ? CKB_ZERO_SLOTS : 0);
}

}  // namespace ckb

/* ------------------------------------------------------------------------------------------------
 * Thread-per-ODE for mechanisms with more than 16 unknowns (ckb_thread.cuh)
 * ---------------------------------------------------------------------------------------------- */
namespace ckbt {

/* slot tables: 64-bit words read with a warp-uniform index */
#define CKBT_PARAM_WORDS 3840 /* 30 KB of the 32 764-byte kernel-parameter space */
struct SlotParamTab {
  unsigned long long w[CKBT_PARAM_WORDS];
  __device__ __forceinline__ unsigned long long ld(int i) const { return w[i]; }
};
typedef ckb::GlobalTab SlotGlobalTab;

/* a regular slot: 8 words (ckb_tables.h CKB_SL_*): ln A_f, beta_f, theta_f, ln A_r, beta_r, theta_r,
 *   idx A = byte offsets (component * 256) of the reactant molecules in fields 0..2, efficiency-set index in field 3
 *   idx B = byte offsets of the product molecules in fields 0..2
 * Every molecule of a regular slot is a different species (reactants AND products), so Eq. 3 is -q on the reactant
 * offsets and +q on the product offsets, read-modify-write with all reads first.
 * An irregular slot (a species twice on one side, or on both sides): 12 words = the 8 above with the molecule counts in
 * field 3 of idx B (nA | nB << 2 | has_tb << 4), then 4 words holding up to 8 scatter entries
 * (int16 net coefficient << 16 | byte offset), unused entries 0. */
#define CKBT_SLOT_WORDS 8
#define CKBT_IRR_WORDS 12
#define CKBT_KIND_IRREGULAR 18 /* kinds 0..17: (nA-1)*6 + (nB-1)*2 + tb */

struct DevThread {
  int K, n;
  int ncls;      /* class directory in the slot table: [ncls][2] = (kind | count << 32, first word) */
  int o_cls;
  /* in the aux blob (global memory, broadcast loads): */
  int o_sp;      /* [K][13] species table (CKB_SP_*), species order = state row order */
  int o_sp2;     /* [K][13] high temperature range, T_mid in the CKB_SP_INVW word; 0 = one range (R30) */
  int o_set;     /* [NTB][2]: (first word of the entries, count | fo word << 32); entries (alpha-1, byte offset) */
  int o_rkc, o_rkcs, s_tab;
  int NS, NTB;
  int has_fo;
};

#define CKBT_VECS 8 /* physical stage vectors per thread in the workspace */
#define CKBT_VB 9   /* components per batch of a pass over a stage vector (loads in flight per input vector) */

}  // namespace ckbt
