/*
 * ckb_api.cu -- C ABI (include/ckb.h): mechanism validation and packing, kernel dispatch.
 * Host logic only; every step of the integration path runs in the kernels of ckb_device.cuh.
 */
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdlib>
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

}  // namespace

namespace ckb_host {
int cuda_fail(cudaError_t e, const char *what) {
  g_cuda_err = std::string(what) + ": " + cudaGetErrorString(e);
  return CKB_ECUDA;
}
}  // namespace ckb_host

/* ------------------------------------------------------------------------------------------------
 * Dispatch
 * ---------------------------------------------------------------------------------------------- */
namespace {

struct Launch {
  int L, NV;
  bool param_tab;
  bool big = false; /* thread-per-ODE with memory-resident stage vectors (K+1 > 16, ckb_thread.cu) */
};

/* AUTO, from the variant map measured on B200: mechanisms with K+1 <= 16 go thread-per-ODE once the batch fills
 * the lanes that mapping keeps resident several times over (148 SMs x 3 x 128; a lone thread takes ~6 us per f(y)),
 * 4 lanes per system at mid sizes (4x the systems in flight per f(y) latency), and warp-per-ODE (~1 us per f(y)) for small
 * batches; larger mechanisms always go warp-per-ODE. */
#define CKB_AUTO_SUB4_MIN_N_RKCK 12288
#define CKB_AUTO_SUB4_MIN_N_RKC 24576
#define CKB_AUTO_THREAD_MIN_N_RKCK 131072
#define CKB_AUTO_THREAD_MIN_N 196608
#define CKB_AUTO_THREAD_MIN_N_SPECIALISED 98304 /* after ckb_mech_specialize(): thread-per-ODE is ~2x faster at full size */
#define CKB_AUTO_THREAD_MIN_N_SPECIALISED_RKCK 49152

int choose(const ckb_mech *m, int variant, long long N, int method, Launch *out) {
  const int n = m->K + 1;
  if (variant == CKB_VARIANT_AUTO) {
    const bool thread_ok = n <= 16 && m->pk[ckb_host::pack_index(1)].rc == CKB_OK;
    const bool sub4_ok = n <= 16 && m->pk[ckb_host::pack_index(4)].rc == CKB_OK;
    const bool warp_ok = m->pk[ckb_host::pack_index(32)].rc == CKB_OK;
    const long long sub4_min = method == CKB_METHOD_RKC ? CKB_AUTO_SUB4_MIN_N_RKC : CKB_AUTO_SUB4_MIN_N_RKCK;
    const long long thread_min = m->gen.ok ? (method == CKB_METHOD_RKC ? CKB_AUTO_THREAD_MIN_N_SPECIALISED
                                                                       : CKB_AUTO_THREAD_MIN_N_SPECIALISED_RKCK)
                                           : (method == CKB_METHOD_RKC ? CKB_AUTO_THREAD_MIN_N : CKB_AUTO_THREAD_MIN_N_RKCK);
    if (thread_ok && (N >= thread_min || (!warp_ok && !sub4_ok)))
      variant = CKB_VARIANT_THREAD;
    else if (sub4_ok && (N >= sub4_min || !warp_ok))
      variant = CKB_VARIANT_SUB4;
    else
      variant = CKB_VARIANT_WARP;
  }
  int L;
  if (variant == CKB_VARIANT_THREAD && n > 16) {
    if (!m->tp) return CKB_EUNSUPPORTED;
    out->L = 1; out->NV = 0; out->param_tab = false; out->big = true;
    return m->tp->rc;
  }
  switch (variant) {
    case CKB_VARIANT_THREAD: L = 1; break;
    case CKB_VARIANT_SUB8: L = 8; break;
    case CKB_VARIANT_SUB16: L = 16; break;
    case CKB_VARIANT_WARP: L = 32; break;
    case CKB_VARIANT_SUB2: L = 2; break;
    case CKB_VARIANT_SUB4: L = 4; break;
    default: return CKB_EINVAL;
  }
  const ckb_host::Packed &pk = m->pk[ckb_host::pack_index(L)];
  if (pk.rc != CKB_OK) return pk.rc;
  out->L = L;
  out->NV = pk.dm.NV;
  out->param_tab = (L == 1);
  return CKB_OK;
}

/* thread-per-ODE launches go to the mechanism-specialised kernels once ckb_mech_specialize() has built them */
int dispatch_integrate(const ckb_mech *m, const Launch &l, int method, const ckb_host::IntegrateArgs &a) {
  if (l.big) return ckb_host::thread_integrate(m, method, a);
  if (l.L == 1 && m->gen.ok) return ckb_host::gen_integrate(m, method, a);
#define X(L_, NV_) \
  if (l.L == L_ && l.NV == NV_) return ckb_host::integrate_L##L_##_NV##NV_(m, method, a);
  CKB_FOR_THREAD(X)
  CKB_FOR_GROUP(X)
#undef X
  return CKB_EUNSUPPORTED;
}

int dispatch_proxy(const ckb_mech *m, const Launch &l, const ckb_host::ProxyArgs &a) {
  if (l.L == 1 && m->gen.ok) return ckb_host::gen_proxy(m, a);
#define X(L_, NV_) \
  if (l.L == L_ && l.NV == NV_) return ckb_host::proxy_L##L_##_NV##NV_(m, a);
  CKB_FOR_THREAD(X)
  CKB_FOR_WARP(X)
#undef X
  return CKB_EUNSUPPORTED;
}

int dispatch_rhs(const ckb_mech *m, const Launch &l, const ckb_host::RhsArgs &a) {
  if (l.big) return ckb_host::thread_rhs(m, a);
  if (l.L == 1 && m->gen.ok) return ckb_host::gen_rhs(m, a);
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

int ckb_mech_load(const ckb_mech_desc *d, ckb_mech **out) { return ckb_mech_load2(d, nullptr, nullptr, out); }

int ckb_mech_load2(const ckb_mech_desc *d, const double *nasa_high, const double *T_mid, ckb_mech **out) {
  return ckb_mech_load3(d, nasa_high, T_mid, 0, nullptr, nullptr, nullptr, out);
}

int ckb_mech_load3(const ckb_mech_desc *d, const double *nasa_high, const double *T_mid, int32_t n_falloff,
                   const int32_t *fo_reaction, const double *fo_low, const double *fo_troe, ckb_mech **out) {
  if (!d || !out || n_falloff < 0) return CKB_EINVAL;
  const ckb_host::FoDesc fo{n_falloff, fo_reaction, fo_low, fo_troe};
  *out = nullptr;
  ckb_mech *m = new (std::nothrow) ckb_mech();
  if (!m) return CKB_ENOMEM;
  int rc;
  try {
    rc = ckb_host::load_packings(d, nasa_high, T_mid, n_falloff > 0 ? &fo : nullptr, m);
  } catch (const std::bad_alloc &) {
    rc = CKB_ENOMEM;
  }
  if (rc != CKB_OK) {
    delete m;
    return rc;
  }
  if (m->tp) {
    rc = ckb_host::thread_upload(*m->tp);
    if (rc != CKB_OK) {
      ckb_mech_free(m);
      return rc;
    }
  }
  rc = ckb_mech_reserve(m, CKB_DEFAULT_MAX_BATCH);
  if (rc != CKB_OK) {
    ckb_mech_free(m);
    return rc;
  }
  cudaError_t e = cudaMalloc((void **)&m->d_counters, CKB_COUNTER_RING * 8);
  for (int i = 0; i < CKB_NPACK && e == cudaSuccess; i++) {
    ckb_host::Packed &p = m->pk[i];
    if (p.rc != CKB_OK) continue;
    e = cudaMalloc((void **)&p.d_blob, p.blob.size() * 8 + 8);
    if (e == cudaSuccess) e = cudaMemcpy(p.d_blob, p.blob.data(), p.blob.size() * 8, cudaMemcpyHostToDevice);
  }
  if (e != cudaSuccess) {
    ckb_mech_free(m);
    return ckb_host::cuda_fail(e, "ckb_mech_load upload");
  }
  *out = m;
  return CKB_OK;
}

int ckb_mech_reserve(ckb_mech *m, int64_t max_batch) {
  if (!m || max_batch < 0) return CKB_EINVAL;
  CK(cudaDeviceSynchronize()); /* nothing of this handle may be in flight while its scratch is replaced */
  return ckb_host::queue_scratch(m, 0, (long long)max_batch, true);
}

void ckb_mech_free(ckb_mech *m) {
  if (!m) return;
  for (int i = 0; i < CKB_NPACK; i++)
    if (m->pk[i].d_blob) cudaFree(m->pk[i].d_blob);
  if (m->tp) ckb_host::thread_free(*m->tp);
  ckb_host::gen_unload(m);
  if (m->d_counters) cudaFree(m->d_counters);
  for (int i = 0; i < CKB_SCRATCH_SLOTS; i++) {
    if (m->osc[i].d_order) cudaFree(m->osc[i].d_order);
    if (m->osc[i].d_bins) cudaFree(m->osc[i].d_bins);
    if (m->osc[i].d_keys) cudaFree(m->osc[i].d_keys);
    if (m->hstream[i]) cudaStreamDestroy(m->hstream[i]);
  }
  for (int i = 0; i <= CKB_SCRATCH_SLOTS; i++)
    if (m->hevent[i]) cudaEventDestroy(m->hevent[i]);
  if (m->ws_states) cudaFree(m->ws_states);
  if (m->ws_pressure) cudaFree(m->ws_pressure);
  if (m->ws_status) cudaFree(m->ws_status);
  if (m->ws_stats) cudaFree(m->ws_stats);
  delete m;
}

int ckb_mech_info(const ckb_mech *m, int32_t *n_species, int32_t *n_reactions, int32_t *n_slots,
                  double *flops_per_rhs) {
  if (!m) return CKB_EINVAL;
  if (n_species) *n_species = m->K;
  if (n_reactions) *n_reactions = m->R;
  if (n_slots) *n_slots = m->NS;
  if (flops_per_rhs) *flops_per_rhs = m->flops_per_rhs;
  return CKB_OK;
}

/* slot: which queue-order scratch to use; n_choice: batch size the AUTO mapping is chosen for (the whole batch
 * when ckb_integrate_host feeds it in chunks) */
static int integrate_impl(const ckb_mech *m, double *states, const double *pressure, double p_uniform, int64_t N,
                          int64_t ld, double t, double dt, double rtol, double atol, int32_t method,
                          int32_t variant, int32_t *status, int32_t *stats, cudaStream_t stream, int slot,
                          int64_t n_choice, int cv, bool grow) {
  if (!m || N < 0 || (method != CKB_METHOD_RKCK && method != CKB_METHOD_RKC)) return CKB_EINVAL;
  if (!(dt > 0.0) || !std::isfinite(dt) || !std::isfinite(t) || !(rtol > 0.0) || !(atol >= 0.0)) return CKB_EINVAL;
  if (!pressure && !(p_uniform > 0.0)) return CKB_EINVAL;
  Launch l;
  int rc = choose(m, variant, (long long)n_choice, method, &l);
  if (rc) return rc;
  if (N == 0) return CKB_OK;
  if (!states || ld < N) return CKB_EINVAL;
  ckb_host::IntegrateArgs a{states, pressure, p_uniform, (long long)N, (long long)ld, t, dt, rtol, atol,
                            status, stats, stream, nullptr, cv};
  /* queue order: hottest systems first (row 0 of states = T); pointless when every system starts at once */
  if (N >= 4096) {
    const ckb_host::Packed &pk32 = m->pk[ckb_host::pack_index(32)];
    if (l.L <= 4 && method == CKB_METHOD_RKC && (m->pk[0].rc == CKB_OK || pk32.rc == CKB_OK)) {
      /* RKC with 8 or more systems per warp: order by the cost proxy || J f / wt || (two evaluations of f per
       * system, computed by the register-resident thread-per-ODE kernel whatever mapping integrates; mechanisms
       * beyond 16 unknowns: by the warp-per-ODE one) */
      const Launch l1 = m->pk[0].rc == CKB_OK ? Launch{1, m->pk[0].dm.NV, true} : Launch{32, pk32.dm.NV, false};
      rc = ckb_host::queue_scratch(m, slot, N, grow);
      if (rc) return rc;
      ckb_host::ProxyArgs pa{states, pressure, p_uniform, (long long)N, (long long)ld, 1e-3 * dt, rtol, atol,
                             m->osc[slot].d_keys, stream, cv};
      rc = dispatch_proxy(m, l1, pa);
      if (rc) return rc;
      rc = ckb_host::make_queue_order(m, slot, 1, m->osc[slot].d_keys, N, a.stream, &a.order, grow);
    } else {
      rc = ckb_host::make_queue_order(m, slot, 0, states, N, a.stream, &a.order, grow);
    }
    if (rc) return rc;
  }
  return dispatch_integrate(m, l, method, a);
}

int ckb_integrate(const ckb_mech *m, double *states, const double *pressure, double p_uniform, int64_t N,
                  int64_t ld, double t, double dt, double rtol, double atol, int32_t method, int32_t variant,
                  int32_t *status, int32_t *stats, void *stream) {
  return integrate_impl(m, states, pressure, p_uniform, N, ld, t, dt, rtol, atol, method, variant, status, stats,
                        (cudaStream_t)stream, 0, N, 0, false);
}

int ckb_integrate_cv(const ckb_mech *m, double *states, const double *density, double rho_uniform, int64_t N,
                     int64_t ld, double t, double dt, double rtol, double atol, int32_t method, int32_t variant,
                     int32_t *status, int32_t *stats, void *stream) {
  return integrate_impl(m, states, density, rho_uniform, N, ld, t, dt, rtol, atol, method, variant, status, stats,
                        (cudaStream_t)stream, 0, N, 1, false);
}

/* ckb_integrate with the queue-order scratch in the library's static device array (ckb_order.cu): a separate path, so
 * that ckb_integrate is untouched.  Calls no cudaMalloc / cudaFree and no routine that allocates. */
int ckb_integrate_static(const ckb_mech *m, double *states, const double *pressure, double p_uniform, int64_t N,
                         int64_t ld, double t, double dt, double rtol, double atol, int32_t method, int32_t variant,
                         int32_t *status, int32_t *stats, void *stream) {
  if (!m || N < 0 || (method != CKB_METHOD_RKCK && method != CKB_METHOD_RKC)) return CKB_EINVAL;
  if (!(dt > 0.0) || !std::isfinite(dt) || !std::isfinite(t) || !(rtol > 0.0) || !(atol >= 0.0)) return CKB_EINVAL;
  if (!pressure && !(p_uniform > 0.0)) return CKB_EINVAL;
  if (N > CKB_STATIC_MAX_BATCH) return CKB_ECAPACITY; /* the static scratch holds CKB_STATIC_MAX_BATCH systems */
  Launch l;
  int rc = choose(m, variant, (long long)N, method, &l);
  if (rc) return rc;
  if (N == 0) return CKB_OK;
  if (!states || ld < N) return CKB_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  ckb_host::IntegrateArgs a{states, pressure, p_uniform, (long long)N, (long long)ld, t, dt, rtol, atol,
                            status, stats, s, nullptr, 0};
  if (N >= 4096) { /* the same queue order as ckb_integrate: cost proxy for RKC with 8 or more systems per warp, else T */
    const ckb_host::Packed &pk32 = m->pk[ckb_host::pack_index(32)];
    if (l.L <= 4 && method == CKB_METHOD_RKC && (m->pk[0].rc == CKB_OK || pk32.rc == CKB_OK)) {
      const Launch l1 = m->pk[0].rc == CKB_OK ? Launch{1, m->pk[0].dm.NV, true} : Launch{32, pk32.dm.NV, false};
      double *d_keys;
      int *d_order;
      unsigned *d_bins;
      rc = ckb_host::static_scratch(&d_keys, &d_order, &d_bins);
      if (rc) return rc;
      ckb_host::ProxyArgs pa{states, pressure, p_uniform, (long long)N, (long long)ld, 1e-3 * dt, rtol, atol, d_keys, s, 0};
      rc = dispatch_proxy(m, l1, pa);
      if (rc) return rc;
      rc = ckb_host::static_queue_order(1, d_keys, N, s, &a.order);
    } else {
      rc = ckb_host::static_queue_order(0, states, N, s, &a.order);
    }
    if (rc) return rc;
  }
  return dispatch_integrate(m, l, method, a);
}

static int rhs_impl(const ckb_mech *m, const double *states, const double *pressure, double p_uniform, int64_t N,
                    int64_t ld, double *dydt, int32_t variant, int32_t repeat, void *stream, int cv) {
  if (!m || N < 0 || repeat < 1) return CKB_EINVAL;
  if (!pressure && !(p_uniform > 0.0)) return CKB_EINVAL;
  Launch l;
  int rc = choose(m, variant, (long long)N, CKB_METHOD_RKCK, &l);
  if (rc) return rc;
  if (N == 0) return CKB_OK;
  if (!states || !dydt || ld < N) return CKB_EINVAL;
  ckb_host::RhsArgs a{states, pressure, p_uniform, (long long)N, (long long)ld, dydt, repeat, (cudaStream_t)stream, cv};
  return dispatch_rhs(m, l, a);
}

int ckb_rhs(const ckb_mech *m, const double *states, const double *pressure, double p_uniform, int64_t N,
            int64_t ld, double *dydt, int32_t variant, int32_t repeat, void *stream) {
  return rhs_impl(m, states, pressure, p_uniform, N, ld, dydt, variant, repeat, stream, 0);
}

int ckb_rhs_cv(const ckb_mech *m, const double *states, const double *density, double rho_uniform, int64_t N,
               int64_t ld, double *dydt, int32_t variant, int32_t repeat, void *stream) {
  return rhs_impl(m, states, density, rho_uniform, N, ld, dydt, variant, repeat, stream, 1);
}

static int integrate_host_impl(ckb_mech *m, double *states, const double *pressure, double p_uniform, int64_t N,
                               int64_t ld, double t, double dt, double rtol, double atol, int32_t method,
                               int32_t variant, int32_t *status, int32_t *stats, void *stream, int cv) {
  if (!m || N < 0) return CKB_EINVAL;
  if (N == 0) return integrate_impl(m, nullptr, nullptr, p_uniform, 0, 0, t, dt, rtol, atol, method, variant,
                                    nullptr, nullptr, (cudaStream_t)stream, 0, 0, cv, true);
  if (!states || ld < N) return CKB_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  const int n = m->K + 1;
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
  /* Large RKCK batches go through in chunks on internal streams, so that the upload of chunk c+1 and the download of
   * chunk c-1 overlap the kernel of chunk c (PCIe is full duplex): there the kernel takes about as long as either
   * copy (configs[1]: 0.64 ms against 0.8 ms each way).  One stream per chunk: measured faster than one upload, one
   * compute and one download stream (1.57 against 1.80 ms; concurrent row-wise copies use more copy engines).
   * RKC batches are stiff problems whose kernel outlasts the copies by one to two orders of magnitude; splitting them
   * only adds a queue tail per chunk (configs[2]: 80 ms in 3 chunks against 46 ms in one), so they go through whole.
   * The device copy is dense (row stride N). */
  const int chunks = (N >= 65536 && method == CKB_METHOD_RKCK) ? CKB_SCRATCH_SLOTS : 1;
  if (chunks > 1 && !m->hstream[0]) {
    for (int i = 0; i < CKB_SCRATCH_SLOTS; i++) CK(cudaStreamCreateWithFlags(&m->hstream[i], cudaStreamNonBlocking));
    for (int i = 0; i <= CKB_SCRATCH_SLOTS; i++) CK(cudaEventCreateWithFlags(&m->hevent[i], cudaEventDisableTiming));
  }
  if (chunks > 1) CK(cudaEventRecord(m->hevent[CKB_SCRATCH_SLOTS], s)); /* order after the caller's stream */
  for (int c = 0; c < chunks; c++) {
    const int64_t c0 = N * c / chunks, c1 = N * (c + 1) / chunks, nc = c1 - c0;
    cudaStream_t cs = chunks > 1 ? m->hstream[c] : s;
    if (chunks > 1) CK(cudaStreamWaitEvent(cs, m->hevent[CKB_SCRATCH_SLOTS], 0));
    CK(cudaMemcpy2DAsync(m->ws_states + c0, (size_t)N * 8, states + c0, (size_t)ld * 8, (size_t)nc * 8, (size_t)n,
                         cudaMemcpyHostToDevice, cs));
    if (pressure) CK(cudaMemcpyAsync(m->ws_pressure + c0, pressure + c0, (size_t)nc * 8, cudaMemcpyHostToDevice, cs));
    int rc = integrate_impl(m, m->ws_states + c0, pressure ? m->ws_pressure + c0 : nullptr, p_uniform, nc, N, t, dt,
                            rtol, atol, method, variant, status ? m->ws_status + c0 : nullptr,
                            stats ? m->ws_stats + 4 * c0 : nullptr, cs, c, N, cv, true);
    if (rc) return rc;
    CK(cudaMemcpy2DAsync(states + c0, (size_t)ld * 8, m->ws_states + c0, (size_t)N * 8, (size_t)nc * 8, (size_t)n,
                         cudaMemcpyDeviceToHost, cs));
    if (status) CK(cudaMemcpyAsync(status + c0, m->ws_status + c0, (size_t)nc * 4, cudaMemcpyDeviceToHost, cs));
    if (stats) /* device block [4][nc] -> host rows of stride N */
      CK(cudaMemcpy2DAsync(stats + c0, (size_t)N * 4, m->ws_stats + 4 * c0, (size_t)nc * 4, (size_t)nc * 4, 4,
                           cudaMemcpyDeviceToHost, cs));
    if (chunks > 1) {
      CK(cudaEventRecord(m->hevent[c], cs));
      CK(cudaStreamWaitEvent(s, m->hevent[c], 0));
    }
  }
  CK(cudaStreamSynchronize(s));
  return CKB_OK;
}

int ckb_integrate_host(ckb_mech *m, double *states, const double *pressure, double p_uniform, int64_t N,
                       int64_t ld, double t, double dt, double rtol, double atol, int32_t method,
                       int32_t variant, int32_t *status, int32_t *stats, void *stream) {
  return integrate_host_impl(m, states, pressure, p_uniform, N, ld, t, dt, rtol, atol, method, variant, status, stats,
                             stream, 0);
}

int ckb_integrate_host_cv(ckb_mech *m, double *states, const double *density, double rho_uniform, int64_t N,
                          int64_t ld, double t, double dt, double rtol, double atol, int32_t method,
                          int32_t variant, int32_t *status, int32_t *stats, void *stream) {
  return integrate_host_impl(m, states, density, rho_uniform, N, ld, t, dt, rtol, atol, method, variant, status, stats,
                             stream, 1);
}

const char *ckb_strerror(int code) {
  switch (code) {
    case CKB_OK: return "ok";
    case CKB_EINVAL: return "invalid argument";
    case CKB_ENOMEM: return "out of memory";
    case CKB_ECUDA: return "CUDA runtime error (see ckb_last_cuda_error)";
    case CKB_EUNSUPPORTED: return "mechanism or variant outside the supported limits";
    case CKB_ECAPACITY:
      return "batch larger than the size reserved for this handle (ckb_mech_reserve) or than CKB_STATIC_MAX_BATCH "
             "(ckb_integrate_static)";
    default: return "unknown error code";
  }
}

const char *ckb_last_cuda_error(void) { return g_cuda_err.c_str(); }

} /* extern "C" */
