/*
 * ckb_host.h -- host-side types shared by ckb_api.cu (C ABI, packing, dispatch) and ckb_inst.cu (one
 * object per (lanes-per-system, slots-per-lane) instantiation of the kernels).
 */
#pragma once
#include <cuda_runtime.h>

#include <atomic>
#include <cstdint>
#include <memory>
#include <string>
#include <utility>
#include <vector>

#include "../../include/ckb.h"
#include "ckb_tables.h"

namespace ckb_host {
int cuda_fail(cudaError_t e, const char *what);
}
#define CK(call)                                                  \
  do {                                                            \
    cudaError_t e_ = (call);                                      \
    if (e_ != cudaSuccess) return ckb_host::cuda_fail(e_, #call); \
  } while (0)

struct ckb_mech;
namespace ckb_host {
/* one packing of the mechanism per lanes-per-system value L (ckb_tables.h) */
struct Packed {
  ckb::DevMech dm{};
  std::vector<unsigned long long> blob; /* host copy of the packed tables */
  unsigned long long *d_blob = nullptr;
  int rc = CKB_EUNSUPPORTED;            /* CKB_OK when this packing exists */
  /* schedule report (L = 32): gather steps per f(y), bank-conflict replays left in the gather and in the
   * concentration reads */
  int gather_steps = 0, gather_excess_wavefronts = 0, slot_excess_wavefronts = 0;
};
/* the mechanism as parsed from ckb_mech_desc: what the packer and the code generator work from */
struct Rx {
  std::vector<int> reac, prod; /* molecule lists (species repeated nu times), sorted */
  int tbset = -1;
};
struct Parsed {
  int K = 0, R = 0;
  std::vector<double> W, nasa;                                  /* [K], [K][7] */
  std::vector<double> nasa_hi, Tmid;                            /* [K][7], [K]: second temperature range, or empty */
  std::vector<double> A, beta, E;                               /* [R] */
  std::vector<Rx> rx;                                           /* [R] */
  std::vector<std::vector<std::pair<int, double>>> sets;        /* third-body sets: (species, alpha) */
  /* fall-off reactions (R31): each owns one efficiency set; fo[t] describes set t (kind 0: an ordinary set).
   * kind 1 Lindemann, 2 Troe with the T** term, 3 Troe without it */
  struct Fo { int kind = 0; double dlnA = 0, dbeta = 0, dtheta = 0, a = 0, invT3 = 0, invT1 = 0, T2 = 0; };
  std::vector<Fo> fo;                                           /* [sets.size()] or empty */
  struct Slot { int f, r; };
  std::vector<Slot> slots;                                      /* fused forward/reverse pairs */
  std::vector<std::vector<std::pair<int, int>>> rows;           /* [K] gather rows: (slot, net coefficient) */
  double flops_per_rhs = 0.0;
};
/* components: 0 = T, then species by decreasing gather-row length (ckb_tables.h) */
/* cap > 0: rows count as min(length, cap) (their tails live elsewhere, pack_for) */
void component_order(const Parsed &P, std::vector<int> &sp_of_comp, std::vector<int> &comp_of_sp, int cap = 0);
struct FoDesc { int n; const int32_t *reaction; const double *low3, *troe4; };
int parse_mechanism(const ckb_mech_desc *d, Parsed &P, const FoDesc *fo = nullptr);
int pack_for(const Parsed &P, int L, Packed &out);
/* RKC coefficients of an s-stage step (Eq. 22-26): mu~_1, then (mu_j, nu_j, mu~_j, gamma~_j) for j = 2..s */
void rkc_stage_coefficients(int s, double *mut1, double *stages);

/* thread-per-ODE packing for mechanisms with more than 16 unknowns (ckb_thread.cu) */
struct ThreadPack {
  ckbt::DevThread dm{};
  std::vector<unsigned long long> slots, aux; /* class directory + slot streams; species / sets / RKC tables */
  unsigned long long *d_slots = nullptr, *d_aux = nullptr;
  double *d_ws = nullptr;                     /* stage vectors of the resident grid: [CKBT_VECS][n][ws_threads] */
  size_t ws_threads = 0, smem = 0;
  int warps = 0, sms = 0;
  bool param = false;                         /* the slot table travels as a kernel parameter (constant bank) */
  int rc = CKB_EUNSUPPORTED;
};
int pack_thread(const Parsed &P, ThreadPack &out);
int thread_upload(ThreadPack &tp);
void thread_free(ThreadPack &tp);
int load_packings(const ckb_mech_desc *d, const double *nasa_high, const double *T_mid, const FoDesc *fo, ckb_mech *m);
#define CKB_NPACK 6
inline int pack_index(int L) { return L == 1 ? 0 : L == 8 ? 1 : L == 16 ? 2 : L == 32 ? 3 : L == 2 ? 4 : 5; }
}  // namespace ckb_host

#define CKB_SCRATCH_SLOTS 4

namespace ckb_host {
/* mechanism-specialised thread-per-ODE kernels (ckb_gen.cu): integrate RKCK, integrate RKC, rhs, cost proxy */
struct GenKernels {
  cudaLibrary_t lib = nullptr;
  cudaKernel_t k[8] = {}; /* [4..7]: the constant-volume instantiations */
  int NV = 0, resident[2] = {0, 0};
  size_t smem[2] = {0, 0};
  bool ok = false;
};
}  // namespace ckb_host

struct ckb_mech {
  std::shared_ptr<ckb_host::Parsed> parsed; /* kept for ckb_mech_specialize */
  std::unique_ptr<ckb_host::ThreadPack> tp; /* K+1 > 16: thread-per-ODE with memory-resident stage vectors */
  ckb_host::GenKernels gen;
  ckb_host::Packed pk[CKB_NPACK]; /* L = 1, 8, 16, 32, 2, 4 (pack_index) */
  int K = 0, R = 0, NS = 0;
  double flops_per_rhs = 0.0;
  /* grow-only device workspace of ckb_integrate_host */
  double *ws_states = nullptr, *ws_pressure = nullptr;
  int32_t *ws_status = nullptr, *ws_stats = nullptr;
  size_t ws_states_cap = 0, ws_n_cap = 0;
  /* work-queue counters of the persistent kernels: a ring, one slot per launch in flight */
  unsigned long long *d_counters = nullptr;
  mutable std::atomic<unsigned> next_counter{0};
  /* queue order scratch (ckb_order.cu): slot 0 is sized at load / by ckb_mech_reserve and never grows inside
   * ckb_integrate; calls on one handle must be stream-ordered (they share it) */
  struct OrderScratch { int *d_order = nullptr; unsigned *d_bins = nullptr; double *d_keys = nullptr; size_t cap = 0; };
  mutable OrderScratch osc[CKB_SCRATCH_SLOTS]; /* slot 0: ckb_integrate; slots 0..: the chunks of ckb_integrate_host */
  cudaStream_t hstream[CKB_SCRATCH_SLOTS] = {};  /* internal streams of the pipelined host entry */
  cudaEvent_t hevent[CKB_SCRATCH_SLOTS + 1] = {};
};


#define CKB_COUNTER_RING 256

namespace ckb_host {

struct IntegrateArgs {
  double *states; const double *pressure; double p_uniform; long long N, ld;
  double t, dt, rtol, atol; int *status, *stats; cudaStream_t stream;
  const int *order; /* queue order (device) or NULL */
  int cv = 0;       /* 1: constant volume (pressure / p_uniform carry the density) */
};

/* mode 0: keys are temperatures (hottest first); mode 1: keys are cost proxies (largest first, log-spaced bins) */
int make_queue_order(const ckb_mech *m, int slot, int mode, const double *keys, long long N, cudaStream_t s,
                     const int **order, bool grow);
int queue_scratch(const ckb_mech *m, int slot, long long N, bool grow);
/* the same with the scratch in a file-scope device array (ckb_order.cu; ckb_integrate_static): no allocation ever */
int static_scratch(double **keys, int **order, unsigned **bins);
int static_queue_order(int mode, const double *keys, long long N, cudaStream_t s, const int **order);

struct ProxyArgs {
  const double *states; const double *pressure; double p_uniform; long long N, ld; double h, rtol, atol;
  double *key; cudaStream_t stream;
  int cv = 0;
};
struct RhsArgs {
  const double *states; const double *pressure; double p_uniform; long long N, ld; double *dydt; int repeat;
  cudaStream_t stream;
  int cv = 0;
};

/* the instantiation list: (lanes per system L, register slots per lane NV); a system needs K+1 <= L*NV */
#define CKB_FOR_THREAD(X) X(1, 4) X(1, 10) X(1, 14) X(1, 16)
#define CKB_FOR_WARP(X) X(32, 1) X(32, 2) X(32, 4) /* the warp-per-ODE subset of CKB_FOR_GROUP (cost-proxy kernels) */
#define CKB_FOR_GROUP(X) X(2, 5) X(2, 8) X(4, 3) X(4, 4) X(8, 7) X(8, 14) X(16, 4) X(16, 7) X(32, 1) X(32, 2) X(32, 4)

/* smallest instantiated NV that holds n unknowns on L lanes, or -1 */
inline int pick_nv(int L, int n) {
  int best = -1;
#define X(L_, NV_) \
  if (L == L_ && n <= L_ * NV_ && (best < 0 || NV_ < best)) best = NV_;
  CKB_FOR_THREAD(X)
  CKB_FOR_GROUP(X)
#undef X
  return best;
}

/* ckb_thread.cu */
int thread_integrate(const ckb_mech *m, int method, const IntegrateArgs &a);
int thread_rhs(const ckb_mech *m, const RhsArgs &a);

/* ckb_gen.cu */
std::string generate_rhs(const Parsed &P);
int gen_load(ckb_mech *m, const std::string &arch);
void gen_unload(ckb_mech *m);
int gen_integrate(const ckb_mech *m, int method, const IntegrateArgs &a);
int gen_rhs(const ckb_mech *m, const RhsArgs &a);
int gen_proxy(const ckb_mech *m, const ProxyArgs &a);
const char *gen_log();

#define CKB_DECL(L_, NV_)                                                                         \
  int integrate_L##L_##_NV##NV_(const ckb_mech *m, int method, const IntegrateArgs &a);           \
  int rhs_L##L_##_NV##NV_(const ckb_mech *m, const RhsArgs &a);                                    \
  int proxy_L##L_##_NV##NV_(const ckb_mech *m, const ProxyArgs &a);
CKB_FOR_THREAD(CKB_DECL)
CKB_FOR_GROUP(CKB_DECL)
#undef CKB_DECL

}  // namespace ckb_host
