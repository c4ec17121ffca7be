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

__device__ __forceinline__ int order_bin(double T) {
  double x = (CKB_ORDER_TMAX - T) * ((double)CKB_ORDER_BINS / (CKB_ORDER_TMAX - CKB_ORDER_TMIN)); /* hot first */
  if (!(x >= 0.0)) x = 0.0; /* also NaN */
  if (x > (double)(CKB_ORDER_BINS - 1)) x = (double)(CKB_ORDER_BINS - 1);
  return (int)x;
}

__global__ void order_hist_kernel(const double *__restrict__ T, long long N, unsigned *__restrict__ bins) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < N) atomicAdd(&bins[order_bin(T[i])], 1u);
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

__global__ void order_scatter_kernel(const double *__restrict__ T, long long N, unsigned *__restrict__ bins,
                                     int *__restrict__ order) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < N) order[atomicAdd(&bins[order_bin(T[i])], 1u)] = (int)i;
}

}  // namespace ckb

namespace ckb_host {

/* fills m's scratch with the queue order of the N systems whose temperatures are T[0..N); returns the device
 * pointer in *order (NULL: keep index order) */
int make_queue_order(const ckb_mech *m, const double *T, long long N, cudaStream_t s, const int **order) {
  *order = nullptr;
  if (N > 2147483647LL) return CKB_OK;
  if ((size_t)N > m->order_cap) {
    if (m->d_order) cudaFree(m->d_order);
    m->d_order = nullptr;
    m->order_cap = 0;
    CK(cudaMalloc((void **)&m->d_order, (size_t)N * sizeof(int)));
    m->order_cap = (size_t)N;
  }
  if (!m->d_bins) CK(cudaMalloc((void **)&m->d_bins, CKB_ORDER_BINS * sizeof(unsigned)));
  CK(cudaMemsetAsync(m->d_bins, 0, CKB_ORDER_BINS * sizeof(unsigned), s));
  const unsigned blocks = (unsigned)((N + 255) / 256);
  ckb::order_hist_kernel<<<blocks, 256, 0, s>>>(T, N, m->d_bins);
  ckb::order_scan_kernel<<<1, CKB_ORDER_BINS / 2, 0, s>>>(m->d_bins);
  ckb::order_scatter_kernel<<<blocks, 256, 0, s>>>(T, N, m->d_bins, m->d_order);
  CK(cudaGetLastError());
  *order = m->d_order;
  return CKB_OK;
}

}  // namespace ckb_host
