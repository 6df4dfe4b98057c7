// mhd_math.cuh -- fp64 reciprocal, reciprocal square root and square root for the VL+CT kernels.
//
// nvcc's IEEE `/` and sqrt() expand to a MUFU seed, Newton steps, a range test and a call to a
// slow path for denormal / huge operands: ~10 fp64-pipe instructions plus ~8 moves, compares and
// branch bookkeeping each, and the step executes ~110 of them per cell.  Every operand here is a
// physical quantity of ordinary magnitude (densities, speeds, pressures; never denormal, never
// near overflow), so the slow path is dead weight.  These versions take the same hardware seed
// (MUFU.RCP64H / MUFU.RSQ64H through PTX rcp.approx / rsqrt.approx, relative error < 2^-20) and
// ONE step of a cubically convergent iteration in fp64 FMAs (error e -> ~e^3 < 2^-60, below the
// rounding of the last FMA): 3 fp64 instructions for 1/x, 5 for 1/sqrt(x), 6 for sqrt(x), each a
// dependent chain of 3-4 (two Newton steps were 4 / 7 / 8 instructions and chains of 4-7).  The
// results are within 2 ulp of the correctly rounded value (tests/test_gpu_units.py, 200 000 operands
// over 60 decades): full fp64 precision, not -use_fast_math (which would not touch fp64 anyway);
// the parity tolerance (1e-12) is four orders of magnitude looser.
// Not valid for 0, denormal, infinite or NaN operands beyond what is noted per function.
#pragma once
#include <cuda_runtime.h>

namespace mhd {

// 1/x for normal x.  One step of the cubically convergent iteration y <- y (1 + e + e^2), e = 1 - x y:
// the seed's relative error of < 2^-20 goes to e^3 < 2^-60, below the rounding of the last FMA.
__device__ __forceinline__ double rcp(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double e = __fma_rn(-x, y, 1.0);
  double t = __fma_rn(e, e, e);
  return __fma_rn(y, t, y);
}

// 1/sqrt(x) for normal x > 0.  Cubic step y <- y (1 + e/2 + 3 e^2/8), e = 1 - x y^2 (remainder 5 e^3/16).
__device__ __forceinline__ double rsqrt_(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double e = __fma_rn(-(x * y), y, 1.0);
  double t = __fma_rn(0.375, e, 0.5) * e;
  return __fma_rn(y, t, y);
}

// sqrt(x) for normal x > 0, and exactly 0 for x == 0 (x < 0 is the caller's bug).  One Newton step
// on the seed (error 2^-44) and then the coupled correction s += (x - s^2) y / 2, which squares the
// error again: the reciprocal root itself never needs full precision here.  Branch-free: for x == 0
// the seed is +inf and the NaN that follows is discarded by the final select.
__device__ __forceinline__ double sqrt_(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double g = x * y, h = 0.5 * y;
  double r = __fma_rn(-g, h, 0.5);
  g = __fma_rn(g, r, g);
  h = __fma_rn(h, r, h);
  r = __fma_rn(-g, g, x);  // residual x - g^2
  g = __fma_rn(r, h, g);
  // zero test on the exponent bits (integer pipe; the seed instruction flushes denormals anyway)
  return (__double2hiint(x) < 0x00100000) ? 0.0 : g;
}

// sqrt(x) for normal x > 0 only (no zero check): g = x y (y the seed of 1/sqrt(x)), then one cubic step
// g <- g (1 + r + 3 r^2 / 2) with r = 1/2 - g y / 2 = e / 2; remainder 5 e^3 / 16 < 2^-60.
__device__ __forceinline__ double sqrt_nz(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double g = x * y, h = 0.5 * y;
  double r = __fma_rn(-g, h, 0.5);
  double t = __fma_rn(1.5 * r, r, r);
  return __fma_rn(g, t, g);
}

// sqrt(x) for x >= 0 of ANY magnitude, denormals included (the seed instruction flushes them to
// zero): operands below 2^-900 are scaled by 2^200 first.  For the one call site that can meet such
// values -- the slow speed where the normal field is ~1e-160 in the numerical foot of a switch-on
// shock (Ryu & Jones 4d).
__device__ __forceinline__ double sqrt_any(double x) {
  const bool tiny = x < 0x1p-900;
  double s = sqrt_(tiny ? x * 0x1p200 : x);
  return tiny ? s * 0x1p-100 : s;
}

// sqrt(x) and 1/sqrt(x) together, x > 0 (the root as x / sqrt(x): <= 2 ulp).
__device__ __forceinline__ void sqrt_rsqrt(double x, double &s, double &is) {
  double y = rsqrt_(x);
  s = x * y;
  is = y;
}

}  // namespace mhd
