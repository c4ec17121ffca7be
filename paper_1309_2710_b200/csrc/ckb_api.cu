/*
 * ckb_api.cu -- C ABI (include/ckb.h): mechanism validation and packing, kernel dispatch.
 * Host logic only; every step of the integration path runs in the kernels of ckb_device.cuh.
 */
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <limits>
#include <map>
#include <new>
#include <string>
#include <vector>

#include "ckb_host.h"

using ckb::DevMech;

namespace {

thread_local std::string g_cuda_err;

constexpr double RC_CAL = 1.98720425864; /* R20: cal/(mol K) */

inline unsigned long long dbits(double x) {
  unsigned long long u;
  std::memcpy(&u, &x, 8);
  return u;
}

}  // namespace

namespace ckb_host {
int cuda_fail(cudaError_t e, const char *what) {
  g_cuda_err = std::string(what) + ": " + cudaGetErrorString(e);
  return CKB_ECUDA;
}
}  // namespace ckb_host

/* ------------------------------------------------------------------------------------------------
 * Packing
 * ---------------------------------------------------------------------------------------------- */
namespace {

struct Rx {
  std::vector<int> reac, prod; /* molecule lists (species repeated nu times), sorted */
  int tbset = -1;
};

int pack_mechanism(const ckb_mech_desc *d, ckb_mech *out) {
  const int K = d->n_species, R = d->n_reactions, R3 = d->n_third_body;
  if (K < 1 || R < 0 || R3 < 0) return CKB_EINVAL;
  if (!d->mol_weight || !d->nasa) return CKB_EINVAL;
  if (R > 0 && (!d->arr_A || !d->arr_beta || !d->arr_E || !d->reac_ptr || !d->prod_ptr)) return CKB_EINVAL;
  if (R3 > 0 && (!d->tb_reaction || !d->tb_ptr)) return CKB_EINVAL;
  if (K > 254) return CKB_EUNSUPPORTED;
  for (int k = 0; k < K; k++)
    if (!(d->mol_weight[k] > 0.0) || !std::isfinite(d->mol_weight[k])) return CKB_EINVAL;
  if (R > 0 && (d->reac_ptr[0] != 0 || d->prod_ptr[0] != 0)) return CKB_EINVAL;
  if (R3 > 0 && d->tb_ptr[0] != 0) return CKB_EINVAL;

  std::vector<Rx> rx(R);
  for (int j = 0; j < R; j++) {
    if (d->reac_ptr[j + 1] < d->reac_ptr[j] || d->prod_ptr[j + 1] < d->prod_ptr[j]) return CKB_EINVAL;
    if (!(d->arr_A[j] >= 0.0) || !std::isfinite(d->arr_A[j]) || !std::isfinite(d->arr_beta[j]) ||
        !std::isfinite(d->arr_E[j]))
      return CKB_EINVAL;
    for (int side = 0; side < 2; side++) {
      const int32_t *ptr = side ? d->prod_ptr : d->reac_ptr;
      const int32_t *sp = side ? d->prod_species : d->reac_species;
      const int32_t *nu = side ? d->prod_nu : d->reac_nu;
      std::vector<int> &mol = side ? rx[j].prod : rx[j].reac;
      if (ptr[j + 1] > ptr[j] && (!sp || !nu)) return CKB_EINVAL;
      for (int e = ptr[j]; e < ptr[j + 1]; e++) {
        if (sp[e] < 0 || sp[e] >= K || nu[e] < 1) return CKB_EINVAL;
        if (nu[e] > 3) return CKB_EUNSUPPORTED;
        for (int q = 0; q < nu[e]; q++) mol.push_back(sp[e]);
      }
      if (mol.size() > 3) return CKB_EUNSUPPORTED;
      std::sort(mol.begin(), mol.end());
    }
  }
  /* third-body efficiency sets, deduplicated */
  std::map<std::vector<std::pair<int, double>>, int> set_id;
  std::vector<std::vector<std::pair<int, double>>> sets;
  for (int r = 0; r < R3; r++) {
    const int j = d->tb_reaction[r];
    if (j < 0 || j >= R || rx[j].tbset >= 0) return CKB_EINVAL;
    if (d->tb_ptr[r + 1] < d->tb_ptr[r]) return CKB_EINVAL;
    std::map<int, double> eff; /* a species listed twice: the last entry wins */
    for (int e = d->tb_ptr[r]; e < d->tb_ptr[r + 1]; e++) {
      if (!d->tb_species || !d->tb_eff) return CKB_EINVAL;
      if (d->tb_species[e] < 0 || d->tb_species[e] >= K || !std::isfinite(d->tb_eff[e])) return CKB_EINVAL;
      eff[d->tb_species[e]] = d->tb_eff[e];
    }
    std::vector<std::pair<int, double>> key(eff.begin(), eff.end());
    auto it = set_id.find(key);
    if (it == set_id.end()) {
      it = set_id.emplace(key, (int)sets.size()).first;
      sets.push_back(key);
    }
    rx[j].tbset = it->second;
  }
  const int NTB = (int)sets.size();
  if (NTB > 65534) return CKB_EUNSUPPORTED;

  /* fuse forward / reverse reactions over the same species into one slot */
  struct Slot { int f, r; };
  std::vector<Slot> slots;
  typedef std::pair<std::pair<std::vector<int>, std::vector<int>>, int> Key;
  std::map<Key, std::vector<int>> waiting; /* key of an unpaired reaction -> its slot index */
  for (int j = 0; j < R; j++) {
    Key rev{{rx[j].prod, rx[j].reac}, rx[j].tbset};
    auto it = waiting.find(rev);
    if (it != waiting.end() && !it->second.empty()) {
      slots[it->second.back()].r = j;
      it->second.pop_back();
    } else {
      Key self{{rx[j].reac, rx[j].prod}, rx[j].tbset};
      waiting[self].push_back((int)slots.size());
      slots.push_back({j, -1});
    }
  }
  const int NS = (int)slots.size();
  if (NS > 65534) return CKB_EUNSUPPORTED;

  /* species-major gather lists: net coefficient of the slot's forward direction */
  std::vector<std::vector<std::pair<int, int>>> rows(K);
  for (int s = 0; s < NS; s++) {
    const Rx &f = rx[slots[s].f];
    std::map<int, int> net;
    for (int k : f.prod) net[k] += 1;
    for (int k : f.reac) net[k] -= 1;
    for (auto &kv : net)
      if (kv.second != 0) rows[kv.first].push_back({s, kv.second});
  }
  size_t nnz_g = 0, nnz_tb = 0;
  for (auto &r : rows) nnz_g += r.size();
  for (auto &s : sets) nnz_tb += s.size();

  DevMech &m = out->dm;
  m.K = K; m.n = K + 1; m.NS = NS; m.NTB = NTB;
  int off = 0;
  auto take = [&off](size_t words) { int o = off; off += (int)words; return o; };
  m.o_invW = take(K); m.o_W = take(K);
  m.o_cp = take(5 * (size_t)K); m.o_h = take(6 * (size_t)K);
  m.o_lnAf = take(NS); m.o_bf = take(NS); m.o_thf = take(NS);
  m.o_lnAr = take(NS); m.o_br = take(NS); m.o_thr = take(NS);
  m.o_idx = take(NS);
  m.o_tbptr = take(NTB + 1); m.o_tbsp = take(nnz_tb); m.o_tbam1 = take(nnz_tb);
  m.o_gptr = take(K + 1); m.o_gat = take(nnz_g);
  m.words = off;
  std::vector<unsigned long long> &b = out->blob;
  b.assign((size_t)off, 0ull);
  auto putd = [&b](int o, double x) { b[(size_t)o] = dbits(x); };
  for (int k = 0; k < K; k++) {
    putd(m.o_invW + k, 1.0 / d->mol_weight[k]);
    putd(m.o_W + k, d->mol_weight[k]);
    const double *a = d->nasa + 7 * (size_t)k;
    for (int q = 0; q < 5; q++) {
      if (!std::isfinite(a[q])) return CKB_EINVAL;
      putd(m.o_cp + q * K + k, a[q]);
      putd(m.o_h + q * K + k, a[q] / (double)(q + 1));
    }
    if (!std::isfinite(a[5])) return CKB_EINVAL;
    putd(m.o_h + 5 * K + k, a[5]);
  }
  const double NEG_INF = -std::numeric_limits<double>::infinity();
  for (int s = 0; s < NS; s++) {
    const int f = slots[s].f, r = slots[s].r;
    putd(m.o_lnAf + s, d->arr_A[f] > 0.0 ? std::log(d->arr_A[f]) : NEG_INF);
    putd(m.o_bf + s, d->arr_beta[f]);
    putd(m.o_thf + s, d->arr_E[f] / RC_CAL);
    if (r >= 0) {
      putd(m.o_lnAr + s, d->arr_A[r] > 0.0 ? std::log(d->arr_A[r]) : NEG_INF);
      putd(m.o_br + s, d->arr_beta[r]);
      putd(m.o_thr + s, d->arr_E[r] / RC_CAL);
    } else {
      putd(m.o_lnAr + s, NEG_INF);
      putd(m.o_br + s, 0.0);
      putd(m.o_thr + s, 0.0);
    }
    unsigned long long w = 0;
    for (int q = 0; q < 3; q++) {
      const unsigned long long a = q < (int)rx[f].reac.size() ? (unsigned)rx[f].reac[q] : (unsigned)K;
      /* a slot without reverse reaction multiplies k_r = 0 by C = 1, never by a product concentration */
      const unsigned long long c = (r >= 0 && q < (int)rx[f].prod.size()) ? (unsigned)rx[f].prod[q] : (unsigned)K;
      w |= a << (8 * q);
      w |= c << (8 * (3 + q));
    }
    w |= (unsigned long long)(rx[f].tbset >= 0 ? rx[f].tbset : NTB) << 48;
    b[(size_t)m.o_idx + s] = w;
  }
  {
    int e = 0;
    for (int t = 0; t < NTB; t++) {
      b[(size_t)m.o_tbptr + t] = (unsigned long long)e;
      for (auto &kv : sets[t]) {
        b[(size_t)m.o_tbsp + e] = (unsigned long long)kv.first;
        putd(m.o_tbam1 + e, kv.second - 1.0);
        e++;
      }
    }
    b[(size_t)m.o_tbptr + NTB] = (unsigned long long)e;
  }
  {
    int e = 0;
    for (int k = 0; k < K; k++) {
      b[(size_t)m.o_gptr + k] = (unsigned long long)e;
      for (auto &sc : rows[k]) {
        b[(size_t)m.o_gat + e] = (dbits((double)sc.second) & ~0xFFFFull) | (unsigned long long)sc.first;
        e++;
      }
    }
    b[(size_t)m.o_gptr + K] = (unsigned long long)e;
  }
  /* algorithmic flops per f(y), DESIGN.md 7.2 (FMA = 2, exp = 30, log = 46, division = 36) */
  double F = 0.0;
  for (int j = 0; j < R; j++) {
    F += 4.0 + 30.0;                                                    /* Eq. 5 */
    F += (double)rx[j].reac.size() + (rx[j].tbset >= 0 ? 1.0 : 0.0);    /* Eq. 4 */
    for (int side = 0; side < 2; side++) {                              /* Eq. 3 */
      const int32_t *ptr = side ? d->prod_ptr : d->reac_ptr;
      const int32_t *nu = side ? d->prod_nu : d->reac_nu;
      for (int e = ptr[j]; e < ptr[j + 1]; e++) F += nu[e] == 1 ? 1.0 : 2.0;
    }
  }
  for (int r = 0; r < R3; r++) F += 2.0 * (d->tb_ptr[r + 1] - d->tb_ptr[r]) + 1.0;
  F += 27.0 * K + 46.0 + 3.0 * 36.0; /* thermo, Eq. 2, Eq. 6, rho, ln T, 1/T */
  out->flops_per_rhs = F;
  out->R = R;
  return CKB_OK;
}

/* ------------------------------------------------------------------------------------------------
 * Dispatch
 * ---------------------------------------------------------------------------------------------- */
struct Launch {
  int L, NV;
  bool param_tab;
};

int choose(const ckb_mech *m, int variant, Launch *out) {
  const int n = m->dm.n;
  static const int nv1[] = {4, 10, 14, 16}; /* must match CKB_FOR_THREAD / CKB_FOR_GROUP */
  static const int nv8[] = {7, 14};
  static const int nv16[] = {4, 7};
  static const int nv32[] = {1, 2, 4};
  if (variant == CKB_VARIANT_AUTO) variant = (n <= 16 && m->dm.words <= CKB_PARAM_WORDS) ? CKB_VARIANT_THREAD : CKB_VARIANT_WARP;
  const int *tab; int cnt, L;
  switch (variant) {
    case CKB_VARIANT_THREAD: tab = nv1; cnt = 4; L = 1; break;
    case CKB_VARIANT_SUB8: tab = nv8; cnt = 2; L = 8; break;
    case CKB_VARIANT_SUB16: tab = nv16; cnt = 2; L = 16; break;
    case CKB_VARIANT_WARP: tab = nv32; cnt = 3; L = 32; break;
    default: return CKB_EINVAL;
  }
  if (L == 1 && m->dm.words > CKB_PARAM_WORDS) return CKB_EUNSUPPORTED;
  for (int i = 0; i < cnt; i++)
    if (n <= L * tab[i]) {
      out->L = L; out->NV = tab[i]; out->param_tab = (L == 1);
      return CKB_OK;
    }
  return CKB_EUNSUPPORTED;
}

int dispatch_integrate(const ckb_mech *m, const Launch &l, int method, const ckb_host::IntegrateArgs &a) {
#define X(L_, NV_) \
  if (l.L == L_ && l.NV == NV_) return ckb_host::integrate_L##L_##_NV##NV_(m, method, a);
  CKB_FOR_THREAD(X)
  CKB_FOR_GROUP(X)
#undef X
  return CKB_EUNSUPPORTED;
}

int dispatch_rhs(const ckb_mech *m, const Launch &l, const ckb_host::RhsArgs &a) {
#define X(L_, NV_) \
  if (l.L == L_ && l.NV == NV_) return ckb_host::rhs_L##L_##_NV##NV_(m, a);
  CKB_FOR_THREAD(X)
  CKB_FOR_GROUP(X)
#undef X
  return CKB_EUNSUPPORTED;
}

}  // namespace

/* ------------------------------------------------------------------------------------------------
 * C ABI
 * ---------------------------------------------------------------------------------------------- */
extern "C" {

int ckb_mech_load(const ckb_mech_desc *d, ckb_mech **out) {
  if (!d || !out) return CKB_EINVAL;
  *out = nullptr;
  ckb_mech *m = new (std::nothrow) ckb_mech();
  if (!m) return CKB_ENOMEM;
  int rc;
  try {
    rc = pack_mechanism(d, m);
  } catch (const std::bad_alloc &) {
    rc = CKB_ENOMEM;
  }
  if (rc != CKB_OK) {
    delete m;
    return rc;
  }
  cudaError_t e = cudaMalloc((void **)&m->d_blob, m->blob.size() * 8 + 8);
  if (e == cudaSuccess) e = cudaMemcpy(m->d_blob, m->blob.data(), m->blob.size() * 8, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMalloc((void **)&m->d_counters, CKB_COUNTER_RING * 8);
  if (e != cudaSuccess) {
    if (m->d_blob) cudaFree(m->d_blob);
    if (m->d_counters) cudaFree(m->d_counters);
    delete m;
    return ckb_host::cuda_fail(e, "ckb_mech_load upload");
  }
  *out = m;
  return CKB_OK;
}

void ckb_mech_free(ckb_mech *m) {
  if (!m) return;
  if (m->d_blob) cudaFree(m->d_blob);
  if (m->d_counters) cudaFree(m->d_counters);
  if (m->ws_states) cudaFree(m->ws_states);
  if (m->ws_pressure) cudaFree(m->ws_pressure);
  if (m->ws_status) cudaFree(m->ws_status);
  if (m->ws_stats) cudaFree(m->ws_stats);
  delete m;
}

int ckb_mech_info(const ckb_mech *m, int32_t *n_species, int32_t *n_reactions, int32_t *n_slots,
                  double *flops_per_rhs) {
  if (!m) return CKB_EINVAL;
  if (n_species) *n_species = m->dm.K;
  if (n_reactions) *n_reactions = m->R;
  if (n_slots) *n_slots = m->dm.NS;
  if (flops_per_rhs) *flops_per_rhs = m->flops_per_rhs;
  return CKB_OK;
}

int ckb_integrate(const ckb_mech *m, double *states, const double *pressure, double p_uniform, int64_t N,
                  int64_t ld, double t, double dt, double rtol, double atol, int32_t method, int32_t variant,
                  int32_t *status, int32_t *stats, void *stream) {
  if (!m || N < 0 || (method != CKB_METHOD_RKCK && method != CKB_METHOD_RKC)) return CKB_EINVAL;
  if (!(dt > 0.0) || !std::isfinite(dt) || !std::isfinite(t) || !(rtol > 0.0) || !(atol >= 0.0)) return CKB_EINVAL;
  if (!pressure && !(p_uniform > 0.0)) return CKB_EINVAL;
  Launch l;
  int rc = choose(m, variant, &l);
  if (rc) return rc;
  if (N == 0) return CKB_OK;
  if (!states || ld < N) return CKB_EINVAL;
  ckb_host::IntegrateArgs a{states, pressure, p_uniform, (long long)N, (long long)ld, t, dt, rtol, atol,
                  status, stats, (cudaStream_t)stream};
  return dispatch_integrate(m, l, method, a);
}

int ckb_rhs(const ckb_mech *m, const double *states, const double *pressure, double p_uniform, int64_t N,
            int64_t ld, double *dydt, int32_t variant, int32_t repeat, void *stream) {
  if (!m || N < 0 || repeat < 1) return CKB_EINVAL;
  if (!pressure && !(p_uniform > 0.0)) return CKB_EINVAL;
  Launch l;
  int rc = choose(m, variant, &l);
  if (rc) return rc;
  if (N == 0) return CKB_OK;
  if (!states || !dydt || ld < N) return CKB_EINVAL;
  ckb_host::RhsArgs a{states, pressure, p_uniform, (long long)N, (long long)ld, dydt, repeat, (cudaStream_t)stream};
  return dispatch_rhs(m, l, a);
}

int ckb_integrate_host(ckb_mech *m, double *states, const double *pressure, double p_uniform, int64_t N,
                       int64_t ld, double t, double dt, double rtol, double atol, int32_t method,
                       int32_t variant, int32_t *status, int32_t *stats, void *stream) {
  if (!m || N < 0) return CKB_EINVAL;
  if (N == 0) return ckb_integrate(m, nullptr, nullptr, p_uniform, 0, 0, t, dt, rtol, atol, method, variant,
                                   nullptr, nullptr, stream);
  if (!states || ld < N) return CKB_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  const int n = m->dm.n;
  const size_t need = (size_t)n * (size_t)N;
  if (need > m->ws_states_cap) {
    if (m->ws_states) cudaFree(m->ws_states);
    m->ws_states = nullptr; m->ws_states_cap = 0;
    CK(cudaMalloc((void **)&m->ws_states, need * sizeof(double)));
    m->ws_states_cap = need;
  }
  if ((size_t)N > m->ws_n_cap) {
    if (m->ws_pressure) cudaFree(m->ws_pressure);
    if (m->ws_status) cudaFree(m->ws_status);
    if (m->ws_stats) cudaFree(m->ws_stats);
    m->ws_pressure = nullptr; m->ws_status = nullptr; m->ws_stats = nullptr; m->ws_n_cap = 0;
    CK(cudaMalloc((void **)&m->ws_pressure, (size_t)N * sizeof(double)));
    CK(cudaMalloc((void **)&m->ws_status, (size_t)N * sizeof(int32_t)));
    CK(cudaMalloc((void **)&m->ws_stats, (size_t)N * 4 * sizeof(int32_t)));
    m->ws_n_cap = (size_t)N;
  }
  /* host rows have stride ld, the device copy is dense (stride N) */
  CK(cudaMemcpy2DAsync(m->ws_states, (size_t)N * 8, states, (size_t)ld * 8, (size_t)N * 8, (size_t)n,
                       cudaMemcpyHostToDevice, s));
  if (pressure) CK(cudaMemcpyAsync(m->ws_pressure, pressure, (size_t)N * 8, cudaMemcpyHostToDevice, s));
  int rc = ckb_integrate(m, m->ws_states, pressure ? m->ws_pressure : nullptr, p_uniform, N, N, t, dt, rtol, atol,
                         method, variant, status ? m->ws_status : nullptr, stats ? m->ws_stats : nullptr, stream);
  if (rc) return rc;
  CK(cudaMemcpy2DAsync(states, (size_t)ld * 8, m->ws_states, (size_t)N * 8, (size_t)N * 8, (size_t)n,
                       cudaMemcpyDeviceToHost, s));
  if (status) CK(cudaMemcpyAsync(status, m->ws_status, (size_t)N * 4, cudaMemcpyDeviceToHost, s));
  if (stats) CK(cudaMemcpyAsync(stats, m->ws_stats, (size_t)N * 16, cudaMemcpyDeviceToHost, s));
  CK(cudaStreamSynchronize(s));
  return CKB_OK;
}

const char *ckb_strerror(int code) {
  switch (code) {
    case CKB_OK: return "ok";
    case CKB_EINVAL: return "invalid argument";
    case CKB_ENOMEM: return "out of memory";
    case CKB_ECUDA: return "CUDA runtime error (see ckb_last_cuda_error)";
    case CKB_EUNSUPPORTED: return "mechanism or variant outside the supported limits";
    default: return "unknown error code";
  }
}

const char *ckb_last_cuda_error(void) { return g_cuda_err.c_str(); }

} /* extern "C" */
