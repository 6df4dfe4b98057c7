// mhd_peaks.cu -- measured roofline denominators for bench.py: a dependent-chain DFMA kernel
// (fp64 pipe peak at the clocks the run actually sees) and a plain copy (HBM read+write).
// Not part of the time step.
#include <cuda_runtime.h>

#include "../../include/mhd.h"

namespace {

__global__ void __launch_bounds__(256) k_dfma_peak(double *out, int iters, double a, double b) {
  double x0 = threadIdx.x * 1e-3, x1 = x0 + 1.0, x2 = x0 + 2.0, x3 = x0 + 3.0;
  double x4 = x0 + 4.0, x5 = x0 + 5.0, x6 = x0 + 6.0, x7 = x0 + 7.0;
  for (int i = 0; i < iters; i++) {
#pragma unroll
    for (int u = 0; u < 8; u++) {
      x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
      x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
  }
  double s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
  if (s == 12345.678) out[0] = s;  // keep the chains alive
}

__global__ void __launch_bounds__(256) k_copy(double2 *__restrict__ dst, const double2 *__restrict__ src,
                                              long long n) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  long long stride = (long long)gridDim.x * blockDim.x;
  for (; i < n; i += stride) dst[i] = src[i];
}

}  // namespace

extern "C" int mhd_measure_peaks(double *fp64_tflops, double *copy_gbs, double seconds) {
  if (!fp64_tflops || !copy_gbs) return MHD_ERR_ARG;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return MHD_ERR_CUDA;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  double *buf = nullptr;
  const long long nbytes = 1LL << 30;  // 1 GiB source + 1 GiB destination
  if (cudaMalloc(&buf, 2 * nbytes) != cudaSuccess) { cudaGetLastError(); return MHD_ERR_NOMEM; }
  cudaMemset(buf, 0, 2 * nbytes);
  // fp64: 8 independent chains per thread, 8 blocks of 256 threads per SM
  const int iters = 4096, blocks = sms * 8;
  k_dfma_peak<<<blocks, 256>>>(buf, 64, 1.0000001, 1e-9);  // warm-up
  cudaDeviceSynchronize();
  double best_tf = 0.0;
  int reps = seconds > 0.5 ? 40 : 5;
  for (int r = 0; r < reps; r++) {
    cudaEventRecord(e0);
    k_dfma_peak<<<blocks, 256>>>(buf, iters, 1.0000001, 1e-9);
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    double flops = 2.0 * 64.0 * iters * 256.0 * blocks;
    double tf = flops / (ms * 1e-3) / 1e12;
    if (seconds > 0.5) best_tf = (r >= reps / 2) ? best_tf + tf / (reps - reps / 2) : 0.0;  // sustained mean
    else if (tf > best_tf) best_tf = tf;
  }
  *fp64_tflops = best_tf;
  double best_bw = 0.0;
  const long long n2 = nbytes / sizeof(double2);
  for (int r = 0; r < 6; r++) {
    cudaEventRecord(e0);
    k_copy<<<sms * 16, 256>>>((double2 *)((char *)buf + nbytes), (const double2 *)buf, n2);
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    double bw = 2.0 * nbytes / (ms * 1e-3) / 1e9;
    if (r > 0 && bw > best_bw) best_bw = bw;
  }
  *copy_gbs = best_bw;
  cudaFree(buf);
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? MHD_OK : MHD_ERR_CUDA;
}
