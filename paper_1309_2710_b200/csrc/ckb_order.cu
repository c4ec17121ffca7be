/*
 * ckb_order.cu -- work-queue order for the persistent integrate kernels.
 *
 * The kernels pull systems from a queue; the batch finishes when the last system does, so a system that needs
 * many sub-steps should start early (longest-processing-time-first).  How many sub-steps a system needs is
 * not known in advance, but it grows with temperature (Arrhenius, Eq. 5): the queue is therefore ordered by
 * decreasing initial T with a counting sort on the device -- histogram, scan, scatter; three tiny launches on
 * the caller's stream.  The order inside a bin is whatever the atomics give: every system is integrated
 * independently, so results do not depend on it.
 */
#include "ckb_host.h"

namespace ckb {

#define CKB_ORDER_BINS 2048
#define CKB_ORDER_TMIN 200.0
#define CKB_ORDER_TMAX 4296.0 /* 2 K per bin */

/* mode 1: cost-proxy keys, 16 bins per binade over [1, 2^128), largest first */
__device__ __forceinline__ int order_bin_log(double key) {
  double x = (double)(CKB_ORDER_BINS - 1) - 16.0 * log2(fmax(key, 1.0));
  if (!(x >= 0.0)) x = 0.0; /* huge, inf and NaN keys go first */
  if (x > (double)(CKB_ORDER_BINS - 1)) x = (double)(CKB_ORDER_BINS - 1);
  return (int)x;
}

__device__ __forceinline__ int order_bin_T(double T) {
  double x = (CKB_ORDER_TMAX - T) * ((double)CKB_ORDER_BINS / (CKB_ORDER_TMAX - CKB_ORDER_TMIN)); /* hot first */
  if (!(x >= 0.0)) x = 0.0; /* also NaN */
  if (x > (double)(CKB_ORDER_BINS - 1)) x = (double)(CKB_ORDER_BINS - 1);
  return (int)x;
}

__device__ __forceinline__ int order_bin(double key, int mode) { return mode ? order_bin_log(key) : order_bin_T(key); }

#define CKB_ORDER_THREADS 512
#define CKB_ORDER_ITEMS 8 /* systems per thread */

/* block-private histogram in shared memory, then one global atomic per non-empty bin and block */
__global__ void __launch_bounds__(CKB_ORDER_THREADS)
order_hist_kernel(const double *__restrict__ T, long long N, unsigned *__restrict__ bins, int mode) {
  __shared__ unsigned s[CKB_ORDER_BINS];
  for (int b = threadIdx.x; b < CKB_ORDER_BINS; b += CKB_ORDER_THREADS) s[b] = 0u;
  __syncthreads();
  const long long base = (long long)blockIdx.x * (CKB_ORDER_THREADS * CKB_ORDER_ITEMS);
#pragma unroll
  for (int k = 0; k < CKB_ORDER_ITEMS; k++) {
    const long long i = base + k * CKB_ORDER_THREADS + threadIdx.x;
    if (i < N) atomicAdd(&s[order_bin(T[i], mode)], 1u);
  }
  __syncthreads();
  for (int b = threadIdx.x; b < CKB_ORDER_BINS; b += CKB_ORDER_THREADS)
    if (s[b]) atomicAdd(&bins[b], s[b]);
}

/* exclusive scan of the bin counts (one block of CKB_ORDER_BINS / 2 threads, two bins per thread) */
__global__ void order_scan_kernel(unsigned *__restrict__ bins) {
  __shared__ unsigned s[CKB_ORDER_BINS];
  const int t = threadIdx.x;
  s[2 * t] = bins[2 * t];
  s[2 * t + 1] = bins[2 * t + 1];
  __syncthreads();
  for (int d = 1; d < CKB_ORDER_BINS; d <<= 1) { /* Hillis-Steele inclusive scan, in place with a barrier pair */
    unsigned a = 0, b = 0;
    if (2 * t >= d) a = s[2 * t - d];
    if (2 * t + 1 >= d) b = s[2 * t + 1 - d];
    __syncthreads();
    s[2 * t] += a;
    s[2 * t + 1] += b;
    __syncthreads();
  }
  bins[2 * t] = (2 * t == 0) ? 0u : s[2 * t - 1];
  bins[2 * t + 1] = s[2 * t];
}

/* rank inside the block by shared atomics, one global atomic per non-empty bin and block for the block's base */
__global__ void __launch_bounds__(CKB_ORDER_THREADS)
order_scatter_kernel(const double *__restrict__ T, long long N, unsigned *__restrict__ bins,
                     int *__restrict__ order, int mode) {
  __shared__ unsigned s[CKB_ORDER_BINS];
  for (int b = threadIdx.x; b < CKB_ORDER_BINS; b += CKB_ORDER_THREADS) s[b] = 0u;
  __syncthreads();
  const long long base = (long long)blockIdx.x * (CKB_ORDER_THREADS * CKB_ORDER_ITEMS);
  int bin[CKB_ORDER_ITEMS];
  unsigned rank[CKB_ORDER_ITEMS];
#pragma unroll
  for (int k = 0; k < CKB_ORDER_ITEMS; k++) {
    const long long i = base + k * CKB_ORDER_THREADS + threadIdx.x;
    bin[k] = -1;
    if (i < N) {
      bin[k] = order_bin(T[i], mode);
      rank[k] = atomicAdd(&s[bin[k]], 1u);
    }
  }
  __syncthreads();
  for (int b = threadIdx.x; b < CKB_ORDER_BINS; b += CKB_ORDER_THREADS)
    if (s[b]) s[b] = atomicAdd(&bins[b], s[b]); /* count -> this block's first position in the bin */
  __syncthreads();
#pragma unroll
  for (int k = 0; k < CKB_ORDER_ITEMS; k++)
    if (bin[k] >= 0) order[s[bin[k]] + rank[k]] = (int)(base + k * CKB_ORDER_THREADS + threadIdx.x);
}

}  // namespace ckb

namespace ckb_host {

/* fills m's scratch with the queue order of the N systems whose temperatures are T[0..N); returns the device
 * pointer in *order (NULL: keep index order) */
/* scratch of one slot: order[N], keys[N], bins.  The device entry (ckb_integrate) never allocates: its slot is sized by
 * ckb_mech_load / ckb_mech_reserve and a larger batch is refused (CKB_ECAPACITY); the host entry, which owns its
 * workspace and synchronises anyway, grows its slots (grow = true). */
int queue_scratch(const ckb_mech *m, int slot, long long N, bool grow) {
  ckb_mech::OrderScratch &sc = m->osc[slot];
  if ((size_t)N > sc.cap && !grow) return CKB_ECAPACITY;
  if ((size_t)N > sc.cap) {
    if (sc.d_order) cudaFree(sc.d_order);
    if (sc.d_keys) cudaFree(sc.d_keys);
    sc.d_order = nullptr; sc.d_keys = nullptr; sc.cap = 0;
    CK(cudaMalloc((void **)&sc.d_order, (size_t)N * sizeof(int)));
    CK(cudaMalloc((void **)&sc.d_keys, (size_t)N * sizeof(double)));
    sc.cap = (size_t)N;
  }
  if (!sc.d_bins) CK(cudaMalloc((void **)&sc.d_bins, CKB_ORDER_BINS * sizeof(unsigned)));
  return CKB_OK;
}

/* fills the slot's scratch with the queue order of N systems by their keys; returns the device pointer in *order */
int make_queue_order(const ckb_mech *m, int slot, int mode, const double *keys, long long N, cudaStream_t s,
                     const int **order, bool grow) {
  ckb_mech::OrderScratch &sc = m->osc[slot];
  *order = nullptr;
  if (N > 2147483647LL) return CKB_OK;
  int rc = queue_scratch(m, slot, N, grow);
  if (rc) return rc;
  CK(cudaMemsetAsync(sc.d_bins, 0, CKB_ORDER_BINS * sizeof(unsigned), s));
  const long long per_block = CKB_ORDER_THREADS * CKB_ORDER_ITEMS;
  const unsigned blocks = (unsigned)((N + per_block - 1) / per_block);
  ckb::order_hist_kernel<<<blocks, CKB_ORDER_THREADS, 0, s>>>(keys, N, sc.d_bins, mode);
  ckb::order_scan_kernel<<<1, CKB_ORDER_BINS / 2, 0, s>>>(sc.d_bins);
  ckb::order_scatter_kernel<<<blocks, CKB_ORDER_THREADS, 0, s>>>(keys, N, sc.d_bins, sc.d_order, mode);
  CK(cudaGetLastError());
  *order = sc.d_order;
  return CKB_OK;
}

/* ------------------------------------------------------------------------------------------------
 * The same queue order with its scratch in a file-scope device array (ckb_integrate_static, include/ckb.h): for callers
 * that may not allocate device memory at all -- nothing here or behind it calls cudaMalloc / cudaFree.
 * Layout: keys[MAX] doubles (cost-proxy keys of the RKC order), order[MAX] ints, bins[CKB_ORDER_BINS] unsigned:
 * 12 bytes per system + 8 KB = 6.0 MiB for CKB_STATIC_MAX_BATCH = 524288, held by every GPU that loads the library
 * until the process exits.  Every call shares it and it keeps the last call's contents: the bins are cleared per call,
 * keys and order are overwritten for [0, N) before they are read.  Calls that overlap on the GPU race on it.
 * In host code the array's NAME is a host-side stand-in, not a device address: its address is taken once per device
 * with cudaGetSymbolAddress (that device current) and only that pointer is handed to kernels.
 * ---------------------------------------------------------------------------------------------- */
#define CKB_STATIC_BYTES ((size_t)CKB_STATIC_MAX_BATCH * 12 + (size_t)CKB_ORDER_BINS * 4)
static __device__ __align__(256) unsigned char g_static_scratch[CKB_STATIC_BYTES];

#define CKB_STATIC_MAX_DEVICES 64
static std::atomic<unsigned char *> g_static_ptr[CKB_STATIC_MAX_DEVICES];

/* device pointers of the three parts on the current device */
int static_scratch(double **keys, int **order, unsigned **bins) {
  int dev = 0;
  CK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= CKB_STATIC_MAX_DEVICES) return CKB_EUNSUPPORTED;
  unsigned char *p = g_static_ptr[dev].load(std::memory_order_acquire);
  if (!p) { /* once per device; a second thread racing here gets the same address */
    void *q = nullptr;
    CK(cudaGetSymbolAddress(&q, g_static_scratch));
    if (!q) return CKB_ECUDA;
    p = (unsigned char *)q;
    g_static_ptr[dev].store(p, std::memory_order_release);
  }
  *keys = reinterpret_cast<double *>(p);
  *order = reinterpret_cast<int *>(p + (size_t)CKB_STATIC_MAX_BATCH * 8);
  *bins = reinterpret_cast<unsigned *>(p + (size_t)CKB_STATIC_MAX_BATCH * 12);
  return CKB_OK;
}

/* make_queue_order with the static scratch: N <= CKB_STATIC_MAX_BATCH (checked by the caller as well) */
int static_queue_order(int mode, const double *keys, long long N, cudaStream_t s, const int **order) {
  *order = nullptr;
  if (N < 0 || N > CKB_STATIC_MAX_BATCH) return CKB_ECAPACITY;
  double *d_keys;
  int *d_order;
  unsigned *d_bins;
  int rc = static_scratch(&d_keys, &d_order, &d_bins);
  if (rc) return rc;
  CK(cudaMemsetAsync(d_bins, 0, CKB_ORDER_BINS * sizeof(unsigned), s)); /* the one part that must start at zero */
  const long long per_block = CKB_ORDER_THREADS * CKB_ORDER_ITEMS;
  const unsigned blocks = (unsigned)((N + per_block - 1) / per_block);
  ckb::order_hist_kernel<<<blocks, CKB_ORDER_THREADS, 0, s>>>(keys, N, d_bins, mode);
  ckb::order_scan_kernel<<<1, CKB_ORDER_BINS / 2, 0, s>>>(d_bins);
  ckb::order_scatter_kernel<<<blocks, CKB_ORDER_THREADS, 0, s>>>(keys, N, d_bins, d_order, mode);
  CK(cudaGetLastError());
  *order = d_order;
  return CKB_OK;
}

}  // namespace ckb_host
