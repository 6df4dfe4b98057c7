// mhd_unit.cu -- unit-level entry points of the C ABI: the per-face / per-cell device functions
// of mhd_device.cuh (HLLD, PLMC/PPMC reconstruction, CT edge formula) evaluated on arrays of
// independent inputs.  They exist so that tests can compare the device arithmetic with the
// oracle function by function (branch coverage, degenerate states) instead of only through a
// whole step.  Host pointers in, host pointers out; synchronous; default stream.
#include <cuda_runtime.h>

#include "../../include/mhd.h"
#include "mhd_device.cuh"

using namespace mhd;

namespace {

__device__ __forceinline__ W7 load_W(const double *p) {
  W7 W;
  W.rho = p[0]; W.u = p[1]; W.v = p[2]; W.w = p[3]; W.P = p[4]; W.by = p[5]; W.bz = p[6];
  return W;
}

__device__ __forceinline__ void store_W(double *p, const W7 &W) {
  p[0] = W.rho; p[1] = W.u; p[2] = W.v; p[3] = W.w; p[4] = W.P; p[5] = W.by; p[6] = W.bz;
}

__global__ void k_unit_hlld(int n, double gamma, const double *WL, const double *WR,
                            const double *bx, double *F) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  W7 L = load_W(WL + 7 * t), R = load_W(WR + 7 * t);
  F7 f = hlld(gamma, 1.0 / (gamma - 1.0), L, R, bx[t]);
  double *o = F + 7 * t;
  o[0] = f.m; o[1] = f.mn; o[2] = f.mt1; o[3] = f.mt2; o[4] = f.e; o[5] = f.by; o[6] = f.bz;
}

template <int RC>
__global__ void k_unit_recon(int n, double gamma, const double *Ws, const double *bn0, double *Wlo,
                             double *Whi) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  W7 lo, hi;
  constexpr int R = (RC == 1 || RC == 3) ? 1 : 2;
  const double *s = Ws + (size_t)t * 7 * (2 * R + 1);
  if (RC == 1) plmc(gamma, load_W(s), load_W(s + 7), load_W(s + 14), bn0[t], lo, hi);
  else if (RC == 2) ppmc(gamma, load_W(s), load_W(s + 7), load_W(s + 14), load_W(s + 21), load_W(s + 28), bn0[t], lo, hi);
  else if (RC == 3) plmp(load_W(s), load_W(s + 7), load_W(s + 14), lo, hi);
  else ppmp(load_W(s), load_W(s + 7), load_W(s + 14), load_W(s + 21), load_W(s + 28), lo, hi);
  store_W(Wlo + 7 * t, lo);
  store_W(Whi + 7 * t, hi);
}

__global__ void k_unit_ct(int n, const double *in, double *out) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  const double *p = in + 12 * t;
  out[t] = ct_edge(p[0], p[1], p[2], p[3], p[4], p[5], p[6], p[7], p[8], p[9], p[10], p[11]);
}

__global__ void k_unit_math(int n, int op, const double *x, double *y) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  y[t] = (op == 0) ? rcp(x[t]) : ((op == 1) ? rsqrt_(x[t]) : sqrt_(x[t]));
}

struct DevBuf {
  double *p = nullptr;
  ~DevBuf() { if (p) cudaFree(p); }
  bool alloc(size_t n) { return cudaMalloc(&p, n * sizeof(double)) == cudaSuccess; }
  bool up(const double *h, size_t n) { return cudaMemcpy(p, h, n * sizeof(double), cudaMemcpyHostToDevice) == cudaSuccess; }
  bool down(double *h, size_t n) { return cudaMemcpy(h, p, n * sizeof(double), cudaMemcpyDeviceToHost) == cudaSuccess; }
};

}  // namespace

extern "C" int mhd_unit_hlld(int n, double gamma, const double *WL, const double *WR, const double *bx,
                             double *F) {
  if (n < 0 || !WL || !WR || !bx || !F || !(gamma > 1.0)) return MHD_ERR_ARG;
  if (n == 0) return MHD_OK;
  DevBuf a, b, c, d;
  if (!a.alloc(7 * (size_t)n) || !b.alloc(7 * (size_t)n) || !c.alloc(n) || !d.alloc(7 * (size_t)n)) return MHD_ERR_NOMEM;
  if (!a.up(WL, 7 * (size_t)n) || !b.up(WR, 7 * (size_t)n) || !c.up(bx, n)) return MHD_ERR_CUDA;
  k_unit_hlld<<<(n + 127) / 128, 128>>>(n, gamma, a.p, b.p, c.p, d.p);
  if (cudaGetLastError() != cudaSuccess || !d.down(F, 7 * (size_t)n)) return MHD_ERR_CUDA;
  return MHD_OK;
}

extern "C" int mhd_unit_reconstruct(int n, double gamma, int recon, const double *Ws, const double *bn0,
                                    double *Wlo, double *Whi) {
  if (n < 0 || !Ws || !bn0 || !Wlo || !Whi || !(gamma > 1.0) || recon < 1 || recon > 4) return MHD_ERR_ARG;
  if (n == 0) return MHD_OK;
  const int radius = (recon == 1 || recon == 3) ? 1 : 2;
  const size_t ns = 7 * (size_t)(2 * radius + 1) * n;
  DevBuf a, b, c, d;
  if (!a.alloc(ns) || !b.alloc(n) || !c.alloc(7 * (size_t)n) || !d.alloc(7 * (size_t)n)) return MHD_ERR_NOMEM;
  if (!a.up(Ws, ns) || !b.up(bn0, n)) return MHD_ERR_CUDA;
  if (recon == 1) k_unit_recon<1><<<(n + 127) / 128, 128>>>(n, gamma, a.p, b.p, c.p, d.p);
  else if (recon == 2) k_unit_recon<2><<<(n + 127) / 128, 128>>>(n, gamma, a.p, b.p, c.p, d.p);
  else if (recon == 3) k_unit_recon<3><<<(n + 127) / 128, 128>>>(n, gamma, a.p, b.p, c.p, d.p);
  else k_unit_recon<4><<<(n + 127) / 128, 128>>>(n, gamma, a.p, b.p, c.p, d.p);
  if (cudaGetLastError() != cudaSuccess || !c.down(Wlo, 7 * (size_t)n) || !d.down(Whi, 7 * (size_t)n)) return MHD_ERR_CUDA;
  return MHD_OK;
}

extern "C" int mhd_unit_ct_edge(int n, const double *in12, double *out) {
  if (n < 0 || !in12 || !out) return MHD_ERR_ARG;
  if (n == 0) return MHD_OK;
  DevBuf a, b;
  if (!a.alloc(12 * (size_t)n) || !b.alloc(n)) return MHD_ERR_NOMEM;
  if (!a.up(in12, 12 * (size_t)n)) return MHD_ERR_CUDA;
  k_unit_ct<<<(n + 127) / 128, 128>>>(n, a.p, b.p);
  if (cudaGetLastError() != cudaSuccess || !b.down(out, n)) return MHD_ERR_CUDA;
  return MHD_OK;
}

extern "C" int mhd_unit_math(int n, int op, const double *x, double *y) {
  if (n < 0 || op < 0 || op > 2 || !x || !y) return MHD_ERR_ARG;
  if (n == 0) return MHD_OK;
  DevBuf a, b;
  if (!a.alloc(n) || !b.alloc(n)) return MHD_ERR_NOMEM;
  if (!a.up(x, n)) return MHD_ERR_CUDA;
  k_unit_math<<<(n + 127) / 128, 128>>>(n, op, a.p, b.p);
  if (cudaGetLastError() != cudaSuccess || !b.down(y, n)) return MHD_ERR_CUDA;
  return MHD_OK;
}
