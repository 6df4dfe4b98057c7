// mhd_grid.cuh -- HBM data layout of the VL+CT context and per-cell loads.
//
// Layout: every field is one fp64 array of pitch*N[1]*N[2] values;
// logical cell (i,j,k), i fastest, lives at (i+ox) + pitch*((j+ng) + N[1]*(k+ng)).  ng ghost
// layers on every side (3 + stencil radius of the reconstruction, so one ghost fill per step
// suffices); ox >= ng is rounded up to 4 doubles and the pitch to 8 doubles so
// that every row starts on a 64-byte boundary and cell 0 on a 32-byte sector.  B_a is stored
// on the LOWER a-face of each cell (Eq. 20).
#pragma once
#include "mhd_device.cuh"

namespace mhd {

enum { F_RHO = 0, F_MX, F_MY, F_MZ, F_E, F_BX, F_BY, F_BZ, NFIELD };

struct State8 {
  double *f[NFIELD];
};

struct Flux21 {
  double *f[3][7];  // [sweep axis][mass, mom_n, mom_t1, mom_t2, energy, B_t1 flux, B_t2 flux]
};

struct Edge3 {
  double *f[3];  // E_x, E_y, E_z on the edges (lower corner of the cell in the other two axes)
};

struct Geo {
  int n[3];        // active cells
  int ng;          // ghost layers
  int ox;          // raw x position of cell i = 0
  int N[3];        // allocated extents (N[0] = pitch)
  long long s[3];  // strides
  long long ntot;  // pitch * N[1] * N[2]
  double d[3];     // Delta_a = L_a / n_a (unit box by default)
  double id[3];    // 1 / Delta_a (= n_a exactly on the unit box)
  double gamma;
  double gm1inv;   // 1 / (gamma - 1)
  int bc[3];
  int recon;
};

struct Box {  // inclusive logical index range
  int lo[3], hi[3];
};

__device__ __forceinline__ long long cell_index(const Geo &g, int i, int j, int k) {
  return (long long)(i + g.ox) + g.s[1] * (long long)(j + g.ng) + g.s[2] * (long long)(k + g.ng);
}

struct Prim {
  double rho, ir, v[3], P, B[3];  // ir = 1/rho
};

// P = (gamma-1)(E - rho v^2/2 - B^2/2) with explicit roundings: every inlined copy
// is the same instruction sequence, so bit-identical cells give bit-identical pressures (the
// limiters' "<= 0" tests include equality, O10; reading R8).
__device__ __forceinline__ double pressure(double gm1, double rho, const double v[3], double E,
                                           const double B[3]) {
  double v2 = __fma_rn(v[2], v[2], __fma_rn(v[1], v[1], __dmul_rn(v[0], v[0])));
  double b2 = __fma_rn(B[2], B[2], __fma_rn(B[1], B[1], __dmul_rn(B[0], B[0])));
  double ek = __dmul_rn(__dmul_rn(0.5, rho), v2);
  return __dmul_rn(gm1, __fma_rn(-0.5, b2, __dadd_rn(E, -ek)));
}

// O1 from the CONSERVED state U^n: v = m / rho, cell-centred B = mean of
// the two opposing faces (Eq. 13), P from the total energy.
__device__ __forceinline__ Prim make_prim(double gm1, double rho, double mx, double my, double mz, double E,
                                          double bxl, double bxh, double byl, double byh, double bzl, double bzh) {
  Prim p;
  double ir = rcp(rho);
  p.rho = rho; p.ir = ir;
  p.B[0] = 0.5 * (bxl + bxh); p.B[1] = 0.5 * (byl + byh); p.B[2] = 0.5 * (bzl + bzh);
  p.v[0] = mx * ir; p.v[1] = my * ir; p.v[2] = mz * ir;
  p.P = pressure(gm1, rho, p.v, E, p.B);
  return p;
}

__device__ __forceinline__ Prim load_prim(const State8 &U, const Geo &g, long long idx) {
  return make_prim(g.gamma - 1.0, __ldg(U.f[F_RHO] + idx), __ldg(U.f[F_MX] + idx), __ldg(U.f[F_MY] + idx),
                   __ldg(U.f[F_MZ] + idx), __ldg(U.f[F_E] + idx), __ldg(U.f[F_BX] + idx),
                   __ldg(U.f[F_BX] + idx + g.s[0]), __ldg(U.f[F_BY] + idx), __ldg(U.f[F_BY] + idx + g.s[1]),
                   __ldg(U.f[F_BZ] + idx), __ldg(U.f[F_BZ] + idx + g.s[2]));
}

// The half-step state is held in PRIMITIVE form (rho, v, P at cell centres in slots F_RHO..F_E,
// face B^{n+1/2} in slots F_BX..F_BZ): the three sweep kernels and the CT kernel of the corrector
// read it ready-made instead of each redoing the division and the pressure.
__device__ __forceinline__ Prim load_prim_half(const State8 &Wh, const Geo &g, long long idx) {
  Prim p;
  p.rho = __ldg(Wh.f[F_RHO] + idx);
  p.ir = 0.0;  // not stored; formed where needed
#pragma unroll
  for (int a = 0; a < 3; a++) {
    p.B[a] = 0.5 * (__ldg(Wh.f[F_BX + a] + idx) + __ldg(Wh.f[F_BX + a] + idx + g.s[a]));
    p.v[a] = __ldg(Wh.f[F_MX + a] + idx);
  }
  p.P = __ldg(Wh.f[F_E] + idx);
  return p;
}

// solver-local state for a sweep along axis A: (n, t1, t2) = (A, A+1, A+2) mod 3 (O0)
template <int A>
__device__ __forceinline__ W7 to_W(const Prim &p, double &bn_cc) {
  W7 W;
  W.rho = p.rho; W.u = p.v[A]; W.v = p.v[(A + 1) % 3]; W.w = p.v[(A + 2) % 3];
  W.P = p.P; W.by = p.B[(A + 1) % 3]; W.bz = p.B[(A + 2) % 3];
  bn_cc = p.B[A];
  return W;
}

template <int A>
__device__ __forceinline__ void store_flux(const Flux21 &F, long long idx, const F7 &f) {
  F.f[A][0][idx] = f.m; F.f[A][1][idx] = f.mn; F.f[A][2][idx] = f.mt1; F.f[A][3][idx] = f.mt2;
  F.f[A][4][idx] = f.e; F.f[A][5][idx] = f.by; F.f[A][6][idx] = f.bz;
}

}  // namespace mhd
