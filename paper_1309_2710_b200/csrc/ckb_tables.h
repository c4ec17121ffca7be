/*
 * ckb_tables.h -- layout of the packed mechanism, seen by the packer and the kernels.
 */
#pragma once
#ifndef __CUDACC__
#define __device__
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

/* Packed mechanism: one blob of 8-byte words, offsets in words. */
struct DevMech {
  int K, n, NS, NTB;
  int o_invW, o_W;          /* [K] 1/W_k, W_k                                                    */
  int o_cp, o_h;            /* [5][K] cp/R coefficients; [6][K] h/(RT) coefficients (a_i/i, a6)  */
  int o_lnAf, o_bf, o_thf;  /* [NS] forward ln A, beta, E/R_c                                    */
  int o_lnAr, o_br, o_thr;  /* [NS] reverse (ln A = -inf when the slot has no reverse reaction)  */
  int o_idx;                /* [NS] bytes 0-2 side-A species, 3-5 side-B species, bits 48-63 third-body set */
  int o_tbptr, o_tbsp, o_tbam1; /* [NTB+1], [nnz], [nnz]: listed species and (alpha - 1)         */
  int o_gptr, o_gat;        /* [K+1], [nnz]: species-major gather list, entry = coef(double, low 16 mantissa bits = slot) */
  int words;
};

}  // namespace ckb
