/*
 * ckb_inst.cu -- one object per kernel instantiation: compile with -DCKB_L=<lanes per system>
 * -DCKB_NV=<register slots per lane>.  L = 1 takes the packed mechanism as a kernel parameter
 * (ParamTab), L > 1 reads it from the device blob (GlobalTab).
 */
#include <cstdlib>
#include <cstring>

#include "ckb_device.cuh"
#include "ckb_host.h"

#ifndef CKB_TMEM_MIN_N
#define CKB_TMEM_MIN_N 2368 /* 148 SMs x 16 warps */
#endif
#ifndef CKB_M
#define CKB_M 1 /* systems evaluated together per group */
#endif
#ifndef CKB_L
#error "compile with -DCKB_L=.. -DCKB_NV=.."
#endif

#define CKB_CAT_(a, b, c, d) a##b##c##d
#define CKB_CAT(a, b, c, d) CKB_CAT_(a, b, c, d)

namespace ckb_host {

namespace {

constexpr int L = CKB_L, NV = CKB_NV;
#if CKB_L == 1
typedef ckb::ParamTab Tab;
#else
typedef ckb::GlobalTab Tab;
#endif

static const Packed &pack_of(const ckb_mech *m) { return m->pk[pack_index(L)]; }


static size_t smem_bytes(const ckb_mech *m, int M, int xdoubles, int block = CKB_BLOCK) {
  const ckb::DevMech &dm = pack_of(m).dm;
  return (size_t)(ckb::region_doubles(dm) + xdoubles) * (32 / L) * M * (block / 32) * sizeof(double);
}

template <class KERN>
static int prep(KERN kern, size_t smem) {
  if (smem > 227 * 1024) return CKB_EUNSUPPORTED;
  if (smem > 48 * 1024) CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  return CKB_OK;
}

static void make_tab(const ckb_mech *m, ckb::ParamTab &t) { std::memcpy(t.w, pack_of(m).blob.data(), pack_of(m).blob.size() * 8); }
static void make_tab(const ckb_mech *m, ckb::GlobalTab &t) { t.p = pack_of(m).d_blob; }

static long long n_blocks(long long N, int M, int block = CKB_BLOCK) {
  const long long per_block = (long long)(block / 32) * (32 / L) * M;
  return (N + per_block - 1) / per_block;
}

template <int METHOD, int CV, int TM = 0>
static int launch(const ckb_mech *m, const IntegrateArgs &a) {
  constexpr int BLOCK = TM ? CKB_TMEM_BLOCK : CKB_BLOCK;
  auto kern = ckb::integrate_kernel<L, NV, Tab, METHOD, CKB_M, CV, TM>;
  const size_t smem = smem_bytes(m, CKB_M, ckb::IntegratorOf<ckb::Sys<L, NV, Tab, CKB_M>, METHOD>::type::XDOUBLES + ckb::Sys<L, NV, Tab, CKB_M>::HDOUBLES, BLOCK);
  int rc = prep(kern, smem);
  if (rc) return rc;
  /* persistent grid: resident capacity of the device (a multiple of the SM count), capped by the batch */
  static int resident = 0, resident_smem = -1; /* per instantiation */
  if (resident == 0 || resident_smem != (int)smem) {
    int dev = 0, sms = 0, per_sm = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, BLOCK, smem));
    if (per_sm < 1) return CKB_EUNSUPPORTED;
    if (TM && per_sm > 1) per_sm = 1; /* the block owns all of the SM's tensor memory */
    resident = sms * per_sm;
    resident_smem = (int)smem;
  }
  long long blocks = n_blocks(a.N, CKB_M, BLOCK);
  if (blocks > resident) blocks = resident;
  unsigned long long *counter = m->d_counters + (m->next_counter.fetch_add(1) % CKB_COUNTER_RING);
  CK(cudaMemsetAsync(counter, 0, 8, a.stream));
  Tab tab;
  make_tab(m, tab);
  kern<<<(unsigned)blocks, BLOCK, smem, a.stream>>>(pack_of(m).dm, tab, a.states, a.pressure, a.p_uniform, a.N, a.ld,
                                                   a.t, a.dt, a.rtol, a.atol, a.status, a.stats, counter, a.order);
  CK(cudaGetLastError());
  return CKB_OK;
}

}  // namespace

int CKB_CAT(integrate_L, CKB_L, _NV, CKB_NV)(const ckb_mech *m, int method, const IntegrateArgs &a) {
#if CKB_TMEM
  /* Slot table in tensor memory: one 512-thread block per SM, so only once the batch fills the 16
   * warps of every SM; the table must fit the 512 columns (16 per slot round). */
  static const bool tm_allowed = [] { const char *e = std::getenv("CKB_NO_TMEM"); return !(e && *e == '1'); }();
  if (tm_allowed && a.N >= CKB_TMEM_MIN_N && pack_of(m).dm.NSR * 16 <= 512) {
    if (a.cv) return method == 0 ? launch<0, 1, 1>(m, a) : launch<1, 1, 1>(m, a);
    return method == 0 ? launch<0, 0, 1>(m, a) : launch<1, 0, 1>(m, a);
  }
#endif
  if (a.cv) return method == 0 ? launch<0, 1>(m, a) : launch<1, 1>(m, a);
  return method == 0 ? launch<0, 0>(m, a) : launch<1, 0>(m, a);
}

int CKB_CAT(rhs_L, CKB_L, _NV, CKB_NV)(const ckb_mech *m, const RhsArgs &a) {
  auto kern = a.cv ? ckb::rhs_kernel<L, NV, Tab, 1> : ckb::rhs_kernel<L, NV, Tab, 0>;
  const size_t smem = smem_bytes(m, 1, ckb::Sys<L, NV, Tab, 1>::HDOUBLES);
  int rc = prep(kern, smem);
  if (rc) return rc;
  const long long blocks = n_blocks(a.N, 1);
  if (blocks > 2147483647LL) return CKB_EINVAL;
  Tab tab;
  make_tab(m, tab);
  kern<<<(unsigned)blocks, CKB_BLOCK, smem, a.stream>>>(pack_of(m).dm, tab, a.states, a.pressure, a.p_uniform, a.N, a.ld,
                                                       a.dydt, a.repeat);
  CK(cudaGetLastError());
  return CKB_OK;
}

int CKB_CAT(proxy_L, CKB_L, _NV, CKB_NV)(const ckb_mech *m, const ProxyArgs &a) {
#if CKB_L == 1 || CKB_L == 32
  auto kern = a.cv ? ckb::cost_proxy_kernel<L, NV, Tab, 1> : ckb::cost_proxy_kernel<L, NV, Tab, 0>;
  const size_t smem = smem_bytes(m, 1, ckb::Sys<L, NV, Tab, 1>::HDOUBLES);
  int rc = prep(kern, smem);
  if (rc) return rc;
  const long long blocks = n_blocks(a.N, 1);
  if (blocks > 2147483647LL) return CKB_EINVAL;
  Tab tab;
  make_tab(m, tab);
  kern<<<(unsigned)blocks, CKB_BLOCK, smem, a.stream>>>(pack_of(m).dm, tab, a.states, a.pressure, a.p_uniform, a.N,
                                                       a.ld, a.h, a.rtol, a.atol, a.key);
  CK(cudaGetLastError());
  return CKB_OK;
#else
  (void)m; (void)a;
  return CKB_EUNSUPPORTED; /* the proxy is computed thread-per-ODE (K+1 <= 16) or warp-per-ODE */
#endif
}

}  // namespace ckb_host
