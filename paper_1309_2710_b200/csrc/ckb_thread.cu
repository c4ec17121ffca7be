/*
 * ckb_thread.cu -- host side of the thread-per-ODE kernels for mechanisms with more than 16 unknowns
 * (ckb_thread.cuh): packing of the class-sorted reaction-slot stream, the stage-vector
 * workspace, launches.
 */
#include <algorithm>
#include <cmath>
#include <cstring>
#include <map>
#include <vector>

#include "ckb_thread.cuh"
#include "ckb_host.h"

namespace ckb_host {

namespace {

constexpr double RC_CAL = 1.98720425864; /* R20 */
constexpr double LN_ZERO = -1.0e4;       /* stands for ln 0 (ckb_exp gives ~1e-308) */

inline unsigned long long dbits(double x) {
  unsigned long long u;
  std::memcpy(&u, &x, 8);
  return u;
}

void put_arrhenius(const Parsed &P, int f, int rv, unsigned long long *w) {
  w[CKB_SL_LNAF] = dbits(P.A[f] > 0.0 ? std::log(P.A[f]) : LN_ZERO);
  w[CKB_SL_BF] = dbits(P.beta[f]);
  w[CKB_SL_THF] = dbits(P.E[f] / RC_CAL);
  w[CKB_SL_LNAR] = dbits((rv >= 0 && P.A[rv] > 0.0) ? std::log(P.A[rv]) : LN_ZERO);
  w[CKB_SL_BR] = dbits(rv >= 0 ? P.beta[rv] : 0.0);
  w[CKB_SL_THR] = dbits(rv >= 0 ? P.E[rv] / RC_CAL : 0.0);
}

}  // namespace

int pack_thread(const Parsed &P, ThreadPack &out) {
  const int K = P.K, n = K + 1;
  if (n * 256 > 65535) return CKB_EUNSUPPORTED; /* 16-bit byte offsets of the interleaved regions */
  const int NS = (int)P.slots.size(), NTB = (int)P.sets.size();
  auto off_of = [](int species) { return (unsigned long long)((1 + species) * 256); };

  /* classes */
  std::vector<std::vector<int>> by_kind(CKBT_KIND_IRREGULAR + 1);
  for (int s = 0; s < NS; s++) {
    const Rx &x = P.rx[P.slots[s].f];
    std::vector<int> all(x.reac);
    all.insert(all.end(), x.prod.begin(), x.prod.end());
    std::sort(all.begin(), all.end());
    const bool distinct = std::adjacent_find(all.begin(), all.end()) == all.end();
    const int na = (int)x.reac.size(), nb = (int)x.prod.size();
    const bool regular = distinct && na >= 1 && na <= 3 && nb >= 1 && nb <= 3;
    by_kind[regular ? (na - 1) * 6 + (nb - 1) * 2 + (x.tbset >= 0 ? 1 : 0) : CKBT_KIND_IRREGULAR].push_back(s);
  }
  int ncls = 0;
  for (auto &v : by_kind) ncls += !v.empty();
  std::vector<unsigned long long> &st = out.slots;
  st.assign((size_t)2 * ncls, 0ull);
  int c = 0;
  for (int kind = 0; kind <= CKBT_KIND_IRREGULAR; kind++) {
    const std::vector<int> &v = by_kind[kind];
    if (v.empty()) continue;
    st[(size_t)2 * c] = (unsigned long long)kind | ((unsigned long long)v.size() << 32);
    st[(size_t)2 * c + 1] = (unsigned long long)st.size();
    c++;
    for (int s : v) {
      const int f = P.slots[s].f, rv = P.slots[s].r;
      const Rx &x = P.rx[f];
      unsigned long long w[CKBT_IRR_WORDS] = {0};
      put_arrhenius(P, f, rv, w);
      unsigned long long wa = 0, wb = 0;
      for (size_t q = 0; q < x.reac.size(); q++) wa |= off_of(x.reac[q]) << (16 * q);
      for (size_t q = 0; q < x.prod.size(); q++) wb |= off_of(x.prod[q]) << (16 * q);
      if (x.tbset >= 0) wa |= (unsigned long long)x.tbset << 48;
      if (kind == CKBT_KIND_IRREGULAR) {
        wb |= (unsigned long long)(x.reac.size() | (x.prod.size() << 2) | (x.tbset >= 0 ? 16u : 0u)) << 48;
        std::map<int, int> net;
        for (int k : x.prod) net[k] += 1;
        for (int k : x.reac) net[k] -= 1;
        int e = 0;
        for (auto &kv : net) {
          if (kv.second == 0) continue;
          const unsigned long long ent = ((unsigned long long)(unsigned)(kv.second & 0xFFFF) << 16) | off_of(kv.first);
          w[8 + e / 2] |= ent << (32 * (e & 1));
          e++;
        }
      }
      w[CKB_SL_IDXA] = wa;
      w[CKB_SL_IDXB] = wb;
      st.insert(st.end(), w, w + (kind == CKBT_KIND_IRREGULAR ? CKBT_IRR_WORDS : CKBT_SLOT_WORDS));
    }
  }

  ckbt::DevThread &m = out.dm;
  m.K = K; m.n = n; m.ncls = ncls; m.o_cls = 0; m.NS = NS; m.NTB = NTB; m.has_fo = 0;
  std::vector<unsigned long long> &a = out.aux;
  a.clear();
  auto take = [&a](size_t words) {
    const int o = (int)a.size();
    a.resize(a.size() + words, 0ull);
    return o;
  };
  take(4); /* word 0 is never a valid table offset (0 = "absent") */
  auto species_rows = [&](const std::vector<double> &nasa, int o, bool second) {
    for (int k = 0; k < K; k++) {
      const double *c7 = &nasa[7 * (size_t)k];
      const int b = o + k * CKB_SP_WORDS;
      a[b + CKB_SP_INVW] = dbits(second ? P.Tmid[k] : 1.0 / P.W[k]);
      a[b + CKB_SP_W] = dbits(P.W[k]);
      for (int q = 0; q < 5; q++) {
        a[b + CKB_SP_CP + q] = dbits(c7[q]);
        a[b + CKB_SP_H + q] = dbits(c7[q] / (double)(q + 1));
      }
      a[b + CKB_SP_H + 5] = dbits(c7[5]);
    }
  };
  m.o_sp = take((size_t)K * CKB_SP_WORDS);
  species_rows(P.nasa, m.o_sp, false);
  m.o_sp2 = 0;
  if (!P.nasa_hi.empty()) {
    m.o_sp2 = take((size_t)K * CKB_SP_WORDS);
    species_rows(P.nasa_hi, m.o_sp2, true);
  }
  m.o_set = take((size_t)2 * NTB);
  for (int t = 0; t < NTB; t++) {
    const int o = take(2 * P.sets[t].size());
    for (size_t e = 0; e < P.sets[t].size(); e++) {
      a[o + 2 * e] = dbits(P.sets[t][e].second - 1.0);
      a[o + 2 * e + 1] = off_of(P.sets[t][e].first);
    }
    unsigned long long fo_word = 0;
    if (!P.fo.empty() && P.fo[t].kind > 0) {
      const Parsed::Fo &f = P.fo[t];
      const int fb = take(8);
      const double w8[8] = {(double)f.kind, f.dlnA, f.dbeta, f.dtheta, f.a, f.invT3, f.invT1, f.T2};
      for (int q = 0; q < 8; q++) a[fb + q] = dbits(w8[q]);
      fo_word = (unsigned long long)fb;
      m.has_fo = 1;
    }
    a[m.o_set + 2 * t] = (unsigned long long)o;
    a[m.o_set + 2 * t + 1] = (unsigned long long)P.sets[t].size() | (fo_word << 32);
  }
  m.s_tab = 48;
  m.o_rkc = take(m.s_tab - 1);
  m.o_rkcs = take((size_t)4 * (m.s_tab - 1) * m.s_tab / 2);
  for (int s = 2; s <= m.s_tab; s++) {
    double mut1;
    std::vector<double> stg(4 * (size_t)(s - 1));
    rkc_stage_coefficients(s, &mut1, stg.data());
    a[m.o_rkc + (s - 2)] = dbits(mut1);
    const int base = m.o_rkcs + 4 * ((s - 2) * (s - 1) / 2);
    for (size_t q = 0; q < stg.size(); q++) a[base + q] = dbits(stg[q]);
  }
  out.param = st.size() <= CKBT_PARAM_WORDS;
  out.rc = CKB_OK;
  return CKB_OK;
}

/* device side of a packing: tables and the stage-vector workspace of the resident grid (sized here, at load) */
int thread_upload(ThreadPack &tp) {
  int dev = 0, sms = 0, smem_max = 0;
  CK(cudaGetDevice(&dev));
  CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  CK(cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
  const size_t per_warp = (size_t)2 * tp.dm.n * 32 * sizeof(double);
  int warps = (int)(((size_t)smem_max - 256) / per_warp); /* 256 B: the static words of the block-wide stage vote */
  if (warps > CKBT_MAX_BLOCK / 32) warps = CKBT_MAX_BLOCK / 32;
  if (warps < 1) return CKB_EUNSUPPORTED;
  tp.warps = warps;
  tp.sms = sms;
  tp.smem = per_warp * warps;
  tp.ws_threads = (size_t)sms * warps * 32;
  CK(cudaMalloc((void **)&tp.d_slots, tp.slots.size() * 8 + 8));
  CK(cudaMemcpy(tp.d_slots, tp.slots.data(), tp.slots.size() * 8, cudaMemcpyHostToDevice));
  CK(cudaMalloc((void **)&tp.d_aux, tp.aux.size() * 8 + 8));
  CK(cudaMemcpy(tp.d_aux, tp.aux.data(), tp.aux.size() * 8, cudaMemcpyHostToDevice));
  CK(cudaMalloc((void **)&tp.d_ws, (size_t)CKBT_VECS * tp.dm.n * tp.ws_threads * sizeof(double)));
  return CKB_OK;
}

void thread_free(ThreadPack &tp) {
  if (tp.d_slots) cudaFree(tp.d_slots);
  if (tp.d_aux) cudaFree(tp.d_aux);
  if (tp.d_ws) cudaFree(tp.d_ws);
  tp.d_slots = tp.d_aux = nullptr;
  tp.d_ws = nullptr;
}

namespace {

void make_tab(const ThreadPack &tp, ckbt::SlotParamTab &t) { std::memcpy(t.w, tp.slots.data(), tp.slots.size() * 8); }
void make_tab(const ThreadPack &tp, ckbt::SlotGlobalTab &t) { t.p = tp.d_slots; }

template <class KERN>
int prep(KERN kern, size_t smem) {
  if (smem > 48 * 1024) CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  return CKB_OK;
}

template <class STAB, int METHOD, int CV>
int launch_integrate(const ckb_mech *m, const IntegrateArgs &a) {
  const ThreadPack &tp = *m->tp;
  auto kern = ckbt::integrate_thread_kernel<STAB, METHOD, CV>;
  int rc = prep(kern, tp.smem);
  if (rc) return rc;
  const int block = tp.warps * 32;
  long long blocks = (a.N + block - 1) / block;
  if (blocks > tp.sms) blocks = tp.sms; /* persistent: one block per SM, the workspace is sized for exactly that */
  unsigned long long *counter = m->d_counters + (m->next_counter.fetch_add(1) % CKB_COUNTER_RING);
  CK(cudaMemsetAsync(counter, 0, 8, a.stream));
  STAB tab;
  make_tab(tp, tab);
  kern<<<(unsigned)blocks, block, tp.smem, a.stream>>>(tp.dm, tab, tp.d_aux, tp.d_ws, a.states, a.pressure, a.p_uniform,
                                                       a.N, a.ld, a.t, a.dt, a.rtol, a.atol, a.status, a.stats, counter,
                                                       a.order);
  CK(cudaGetLastError());
  return CKB_OK;
}

template <class STAB, int CV>
int launch_rhs(const ckb_mech *m, const RhsArgs &a) {
  const ThreadPack &tp = *m->tp;
  auto kern = ckbt::rhs_thread_kernel<STAB, CV>;
  int rc = prep(kern, tp.smem);
  if (rc) return rc;
  const int block = tp.warps * 32;
  long long blocks = (a.N + block - 1) / block;
  if (blocks > tp.sms) blocks = tp.sms;
  STAB tab;
  make_tab(tp, tab);
  kern<<<(unsigned)blocks, block, tp.smem, a.stream>>>(tp.dm, tab, tp.d_aux, tp.d_ws, a.states, a.pressure, a.p_uniform,
                                                       a.N, a.ld, a.dydt, a.repeat);
  CK(cudaGetLastError());
  return CKB_OK;
}

}  // namespace

int thread_integrate(const ckb_mech *m, int method, const IntegrateArgs &a) {
  if (!m->tp || m->tp->rc != CKB_OK) return CKB_EUNSUPPORTED;
#define CKBT_GO(STAB)                                                                         \
  if (a.cv) return method == 0 ? launch_integrate<STAB, 0, 1>(m, a) : launch_integrate<STAB, 1, 1>(m, a); \
  return method == 0 ? launch_integrate<STAB, 0, 0>(m, a) : launch_integrate<STAB, 1, 0>(m, a);
  if (m->tp->param) { CKBT_GO(ckbt::SlotParamTab) }
  CKBT_GO(ckbt::SlotGlobalTab)
#undef CKBT_GO
}

int thread_rhs(const ckb_mech *m, const RhsArgs &a) {
  if (!m->tp || m->tp->rc != CKB_OK) return CKB_EUNSUPPORTED;
  if (m->tp->param) return a.cv ? launch_rhs<ckbt::SlotParamTab, 1>(m, a) : launch_rhs<ckbt::SlotParamTab, 0>(m, a);
  return a.cv ? launch_rhs<ckbt::SlotGlobalTab, 1>(m, a) : launch_rhs<ckbt::SlotGlobalTab, 0>(m, a);
}

}  // namespace ckb_host
