// mhd_noalloc.cu -- mhd_max_divb_noalloc: the div B diagnostic for callers that may not
// allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  Self-contained: it needs
// no mhd_init, touches no context and calls no cudaMalloc / cudaFree / allocating library routine.
//
// The reduction's scratch (one partial maximum per block) is a file-scope __device__ array of a fixed,
// modest size: MHD_NOALLOC_MAX_PARTIALS doubles = 512 KiB, held by every GPU that loads the library until
// the process exits.  Every call on a device shares it and it keeps the last call's contents:
//   - nothing in it has to start at zero: pass 1 writes slots [0, nblocks) and pass 2 reads exactly those,
//     both on the caller's stream, so stale partials of an earlier (larger) call are never read;
//   - two calls that overlap on the GPU (different streams, no ordering between them) RACE on it.
//
// In host code the array's name is a host-side stand-in, not a device address; the address a kernel can
// use is obtained once per device, with that device current, by cudaGetSymbolAddress (below).
#include <cuda_runtime.h>

#include <cstdio>
#include <mutex>

#include "../../include/mhd.h"

namespace {

constexpr int kThreads = 256;
constexpr int kMaxDevices = 64;

static __device__ __align__(256) double g_divb_partial[MHD_NOALLOC_MAX_PARTIALS];

char g_noalloc_err[256] = "no error";
std::mutex g_mu;
double *g_partial_ptr[kMaxDevices] = {nullptr};   // device address of g_divb_partial, per device

int nfail(int code, const char *msg) {
  snprintf(g_noalloc_err, sizeof(g_noalloc_err), "%s", msg);
  return code;
}

int ncuda_fail(cudaError_t e, const char *where) {
  snprintf(g_noalloc_err, sizeof(g_noalloc_err), "CUDA error at %s: %s", where, cudaGetErrorString(e));
  return MHD_ERR_CUDA;
}

// set-up, once per device, with that device current
int scratch_address(double **out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return ncuda_fail(e, "cudaGetDevice");
  if (dev < 0 || dev >= kMaxDevices) return nfail(MHD_ERR_ARG, "mhd_max_divb_noalloc: device ordinal out of range");
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_partial_ptr[dev]) {
    double *p = nullptr;
    e = cudaGetSymbolAddress((void **)&p, g_divb_partial);
    if (e != cudaSuccess) return ncuda_fail(e, "cudaGetSymbolAddress(g_divb_partial)");
    if (!p) return nfail(MHD_ERR_CUDA, "cudaGetSymbolAddress returned a null address");
    g_partial_ptr[dev] = p;
  }
  *out = g_partial_ptr[dev];
  return MHD_OK;
}

__device__ __forceinline__ double block_max(double m) {
  __shared__ double wm[kThreads / 32];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0) wm[threadIdx.x >> 5] = m;
  __syncthreads();
  m = (threadIdx.x < kThreads / 32) ? wm[threadIdx.x] : 0.0;
  if (threadIdx.x < 32) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
  }
  return m;   // valid in thread 0
}

// pass 1: one thread per cell of the dense ABI layout (include/mhd.h: bx (nx+1) x ny x nz, by nx x (ny+1) x nz,
// bz nx x ny x (nz+1), i fastest); the same expression, in the same order, as k_divb of mhd_kernels.cuh
__global__ void __launch_bounds__(kThreads) k_divb_partials(const double *__restrict__ bx, const double *__restrict__ by,
                                                            const double *__restrict__ bz, int nx, int ny, int nz,
                                                            double dx, double dy, double dz, double *partial) {
  const long long t = (long long)blockIdx.x * kThreads + threadIdx.x;
  const long long ncell = (long long)nx * ny * nz;
  double m = 0.0;
  if (t < ncell) {
    const int i = (int)(t % nx), j = (int)((t / nx) % ny), k = (int)(t / ((long long)nx * ny));
    const long long ix = i + (long long)(nx + 1) * (j + (long long)ny * k);
    const long long iy = i + (long long)nx * (j + (long long)(ny + 1) * k);
    const long long iz = i + (long long)nx * (j + (long long)ny * k);
    double d = 0.0;
    d += (bx[ix + 1] - bx[ix]) / dx;
    d += (by[iy + nx] - by[iy]) / dy;
    d += (bz[iz + (long long)nx * ny] - bz[iz]) / dz;
    m = fabs(d);
  }
  m = block_max(m);
  if (threadIdx.x == 0) partial[blockIdx.x] = m;
}

// pass 2: one block over the partials of THIS call
__global__ void __launch_bounds__(kThreads) k_divb_finish(const double *partial, int n, double *out) {
  double m = 0.0;
  for (int q = threadIdx.x; q < n; q += kThreads) m = fmax(m, partial[q]);
  m = block_max(m);
  if (threadIdx.x == 0) *out = m;
}

}  // namespace

extern "C" int mhd_max_divb_noalloc(int nx, int ny, int nz, double dx, double dy, double dz, const double *d_bx,
                                    const double *d_by, const double *d_bz, double *d_out, void *stream) {
  if (nx < 1 || ny < 1 || nz < 1 || !(dx > 0.0) || !(dy > 0.0) || !(dz > 0.0))
    return nfail(MHD_ERR_ARG, "mhd_max_divb_noalloc: bad grid size or spacing");
  if (!d_bx || !d_by || !d_bz || !d_out) return nfail(MHD_ERR_ARG, "mhd_max_divb_noalloc: null pointer");
  const long long ncell = (long long)nx * ny * nz;
  if (ncell > MHD_NOALLOC_MAX_CELLS) {
    snprintf(g_noalloc_err, sizeof(g_noalloc_err),
             "mhd_max_divb_noalloc: %lld cells exceed the static scratch (at most %lld cells = %d partial maxima of %d "
             "cells); use mhd_max_divb",
             ncell, (long long)MHD_NOALLOC_MAX_CELLS, MHD_NOALLOC_MAX_PARTIALS, kThreads);
    return MHD_ERR_ARG;
  }
  double *partial = nullptr;
  int rc = scratch_address(&partial);
  if (rc) return rc;
  const int nblocks = (int)((ncell + kThreads - 1) / kThreads);
  cudaStream_t s = (cudaStream_t)stream;
  k_divb_partials<<<nblocks, kThreads, 0, s>>>(d_bx, d_by, d_bz, nx, ny, nz, dx, dy, dz, partial);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return ncuda_fail(e, "k_divb_partials");
  k_divb_finish<<<1, kThreads, 0, s>>>(partial, nblocks, d_out);
  e = cudaGetLastError();
  if (e != cudaSuccess) return ncuda_fail(e, "k_divb_finish");
  return MHD_OK;
}

extern "C" const char *mhd_noalloc_last_error(void) { return g_noalloc_err; }
