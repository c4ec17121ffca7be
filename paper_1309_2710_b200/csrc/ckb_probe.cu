/*
 * ckb_probe.cu -- roofline denominators measured on the device the library runs on:
 * sustained DFMA rate and exp(double) rate of register-resident kernels.
 */
#include "ckb_host.h"

namespace ckb {

/* roofline probes: independent DFMA chains / exp(double) calls, register resident */
__global__ void __launch_bounds__(256) probe_dfma_kernel(double *out, long long iters, double a, double b) {
  double x0 = threadIdx.x * 1e-3, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6,
         x7 = x0 + 7;
  for (long long i = 0; i < iters; i++) {
    x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
    x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
  }
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}

__global__ void __launch_bounds__(256) probe_exp_kernel(double *out, long long iters, double a) {
  double x0 = -1.0 - threadIdx.x * 1e-3, x1 = x0 - 1, x2 = x0 - 2, x3 = x0 - 3;
  double s0 = 0, s1 = 0, s2 = 0, s3 = 0;
  for (long long i = 0; i < iters; i++) {
    s0 += exp(x0); s1 += exp(x1); s2 += exp(x2); s3 += exp(x3);
    x0 += a; x1 += a; x2 += a; x3 += a;
  }
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = (s0 + s1) + (s2 + s3);
}

}  // namespace ckb

extern "C" {

int ckb_fp64_probe(int32_t kind, int64_t iters, double *per_second, void *stream) {
  if (!per_second || iters < 1 || (kind != 0 && kind != 1)) return CKB_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  int dev = 0, sms = 0;
  CK(cudaGetDevice(&dev));
  CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int blocks = sms * 8, threads = 256;
  double *out = nullptr;
  CK(cudaMalloc((void **)&out, (size_t)blocks * threads * 8));
  cudaEvent_t e0, e1;
  CK(cudaEventCreate(&e0));
  CK(cudaEventCreate(&e1));
  float best_ms = 1e30f;
  for (int rep = 0; rep < 4; rep++) { /* first repetition is the warm-up */
    CK(cudaEventRecord(e0, s));
    if (kind == 0) ckb::probe_dfma_kernel<<<blocks, threads, 0, s>>>(out, iters, 0.999999, 1e-7);
    else ckb::probe_exp_kernel<<<blocks, threads, 0, s>>>(out, iters, -1e-6);
    CK(cudaGetLastError());
    CK(cudaEventRecord(e1, s));
    CK(cudaEventSynchronize(e1));
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, e0, e1));
    if (rep > 0 && ms < best_ms) best_ms = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(out);
  const double per_thread = (kind == 0) ? 8.0 * 2.0 * (double)iters : 4.0 * (double)iters;
  *per_second = per_thread * (double)blocks * threads / ((double)best_ms * 1e-3);
  return CKB_OK;
}

} /* extern "C" */
