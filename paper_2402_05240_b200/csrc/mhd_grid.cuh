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
  double d[3];     // Delta_a = 1/n_a
  double gamma;
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
  double rho, v[3], P, B[3];
};

// O1: v = m / rho, cell-centred B = mean of the two opposing faces
// (Eq. 13), P from the total energy.  Primitives are recomputed wherever needed, never stored
// (PAPER.md:305).
__device__ __forceinline__ Prim load_prim(const State8 &U, const Geo &g, long long idx) {
  Prim p;
  double rho = __ldg(U.f[F_RHO] + idx);
  double ir = 1.0 / rho;
  p.rho = rho;
#pragma unroll
  for (int a = 0; a < 3; a++) {
    p.B[a] = 0.5 * (__ldg(U.f[F_BX + a] + idx) + __ldg(U.f[F_BX + a] + idx + g.s[a]));
    p.v[a] = __ldg(U.f[F_MX + a] + idx) * ir;
  }
  double E = __ldg(U.f[F_E] + idx);
  // explicit roundings: every inlined copy is the same instruction sequence, so bit-identical
  // cells give bit-identical primitives (the limiters' "<= 0" tests include equality, O10)
  double v2 = __fma_rn(p.v[2], p.v[2], __fma_rn(p.v[1], p.v[1], __dmul_rn(p.v[0], p.v[0])));
  double b2 = __fma_rn(p.B[2], p.B[2], __fma_rn(p.B[1], p.B[1], __dmul_rn(p.B[0], p.B[0])));
  double ek = __dmul_rn(__dmul_rn(0.5, rho), v2);
  p.P = __dmul_rn(g.gamma - 1.0, __fma_rn(-0.5, b2, __dadd_rn(E, -ek)));
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
