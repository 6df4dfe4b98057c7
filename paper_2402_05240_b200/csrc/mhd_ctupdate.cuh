// mhd_ctupdate.cuh -- the tail of the corrector (a7 + the face-field part of a8 + a1 of SURVEY.md 8(a))
// in ONE kernel: CT edge fields from the corrector fluxes (Eq. 15-18, Table 1),
// face-field update B^{n+1} = B^n + dt curl-difference of E^{n+1/2} (Eq. 30-32) and
// the CFL signal rate of the finished cell U^{n+1} (Eq. 11-12) with its warp-shuffle /
// block / atomic reduction.  The three edge-field arrays never touch HBM.
//
// Geometry: a block owns 31 x (TY-1) columns (32 x TY threads, x along the warp) and marches along z.
// At plane k every thread forms the three edge fields on the lower corner of its cell (as k_ct), the
// block exchanges E_x and E_z with the row above through shared memory (double-buffered: one barrier per
// plane) and E_y, E_z with the lane above by shuffle; the z face of plane k and the x / y faces of
// plane k-1 -- whose upper edges are now known -- are updated, and cell k-1 gets its CFL rate.  The face
// arithmetic is the stage kernel's (fma_diff, same order), so a face has the same bits wherever it is formed.
#pragma once
#include "mhd_kernels.cuh"

namespace mhd {

#ifndef MHD_CTU_TY
#define MHD_CTU_TY 8
#endif
#ifndef MHD_MINB_CTU
#define MHD_MINB_CTU 2
#endif

template <int C>
__device__ __forceinline__ double ct_at(const Flux21 &F, const Edge3 &Er, const Geo &g, long long idx) {
  constexpr int A = (C + 1) % 3, B = (C + 2) % 3;
  const long long sa = g.s[A], sb = g.s[B];
  double Ea0 = -__ldg(F.f[A][5] + idx), Ea1 = -__ldg(F.f[A][5] + idx - sb);
  double Eb0 = __ldg(F.f[B][6] + idx), Eb1 = __ldg(F.f[B][6] + idx - sa);
  double Ma0 = __ldg(F.f[A][0] + idx), Ma1 = __ldg(F.f[A][0] + idx - sb);
  double Mb0 = __ldg(F.f[B][0] + idx), Mb1 = __ldg(F.f[B][0] + idx - sa);
  const double *er = Er.f[C];
  return ct_edge(Ea0, Ea1, Eb0, Eb1, Ma0, Ma1, Mb0, Mb1, __ldg(er + idx), __ldg(er + idx - sa),
                 __ldg(er + idx - sb), __ldg(er + idx - sa - sb));
}

// indices [0, n] per axis (faces 0..n, cells 0..n-1); grid: x = tiles (ntx per row of tiles), y = z-chunks
// of lz planes.  U: the state whose hydro variables are already U^{n+1} and whose face arrays hold B^n;
// Bout: the face arrays that receive B^{n+1}.
//
// Operand staging: the nine CT flux components and the three reference fields of a plane are copied
// with cp.async into a ring of three plane buffers of shared memory (tile of (TY+1) x 33 values per
// array: the block's columns plus the row and the column below them), two planes ahead of their use;
// every edge operand is then a shared-memory read, and the one barrier per plane that the edge
// exchange needs also publishes the plane that has just landed.  B^n and the hydro variables of the
// cell to finish are requested one plane ahead into registers.
#define MHD_CTU_NF 12
template <int TY>
struct CtuTile {
  static constexpr int W = 33, H = TY + 1, PLANE = W * H, STAGE = MHD_CTU_NF * PLANE;
  static constexpr size_t BYTES = (size_t)3 * STAGE * sizeof(double);
};

__device__ __forceinline__ const double *ctu_field(const Flux21 &F, const Edge3 &Er, int f) {
  // 0..2 = x flux (mass, B_t1, B_t2), 3..5 = y flux, 6..8 = z flux, 9..11 = E_ref x, y, z
  return f < 9 ? F.f[f / 3][(f % 3 == 0) ? 0 : 4 + f % 3] : Er.f[f - 9];
}

template <int TY>
__global__ void __launch_bounds__(32 * TY, MHD_MINB_CTU)
k_ct_update(State8 U, Edge3 Bout, Flux21 F, Edge3 Er, Geo g, Scalars *sc, int ntx, int lz) {
  constexpr int NT = 32 * TY;
  using T = CtuTile<TY>;
  extern __shared__ double ctu_ring[];
  __shared__ double ex_s[2][NT], ez_s[2][NT];
  const int t = threadIdx.x, lane = t & 31, row = t >> 5;
  const int tbx = blockIdx.x % ntx, tby = blockIdx.x / ntx;
  const int n0 = g.n[0], n1 = g.n[1], n2 = g.n[2];
  const int kc0 = (int)blockIdx.y * lz, kc1 = min(kc0 + lz - 1, n2 - 1);   // cell planes of this chunk
  const int i0 = 31 * tbx + lane, j0 = (TY - 1) * tby + row;
  // threads beyond the last face index compute on clamped coordinates; nothing of theirs is used
  const int i = min(i0, n0), j = min(j0, n1);
  const bool own = lane <= 30 && row <= TY - 2 && i0 <= n0 && j0 <= n1;
  const bool inx = i0 < n0, iny = j0 < n1;
  const int tu = (row < TY - 1) ? t + 32 : t;       // upper y neighbour
  const double dt = sc->dt;
  const double dtd0 = dt * g.id[0], dtd1 = dt * g.id[1], dtd2 = dt * g.id[2];
  double rate = 0.0;
  int bad = 0;
  if (kc0 <= kc1) {
    const int o = (row + 1) * T::W + lane + 1, ox = o - 1, oy = o - T::W, oxy = oy - 1;
    const long long sy = g.s[1], sz = g.s[2];
    // request plane k (cell index c of this thread) into ring slot st: every thread its own value; the
    // row below the tile (and the corner) by warp 0, the column below it by the first lanes of warp 1
    // (warp-uniform branches: the other warps issue twelve copies and nothing else)
    const long long d_row = -sy;                                   // warp 0: element (i, j-1)
    // warp 1, lane q: element (x of lane 0 minus one, row q of the tile), as an offset from this thread's cell
    const long long d_col = (long long)(min((TY - 1) * tby + lane, n1) - j) * sy + (31 * tbx - 1 - i);
    const int o_col = (lane + 1) * T::W;                           // tile position (row lane, column -1)
    auto request = [&](int st, long long c) {
      double *base = ctu_ring + st * T::STAGE;
#pragma unroll
      for (int f = 0; f < MHD_CTU_NF; f++) cp_async8(base + f * T::PLANE + o, ctu_field(F, Er, f) + c);
      if (row == 0) {
#pragma unroll
        for (int f = 0; f < MHD_CTU_NF; f++) {
          cp_async8(base + f * T::PLANE + oy, ctu_field(F, Er, f) + c + d_row);
          if (lane == 0) cp_async8(base + f * T::PLANE + oxy, ctu_field(F, Er, f) + c + d_row - 1);
        }
      } else if (row == 1 && lane < TY) {
#pragma unroll
        for (int f = 0; f < MHD_CTU_NF; f++) cp_async8(base + f * T::PLANE + o_col, ctu_field(F, Er, f) + c + d_col);
      }
      cp_async_commit();
    };
    long long c = cell_index(g, i, j, kc0);
    // ring slot of plane k: (k - kc0 + 1) % 3
    request(0, c - sz);
    request(1, c);
    cp_async_wait_all();
    __syncthreads();
    if (kc0 + 1 <= kc1 + 1) request(2, c + sz);
    // register prefetch: B^n of the plane to come, hydro variables of the cell to finish
    double bzn = __ldg(U.f[F_BZ] + c), bxn = __ldg(U.f[F_BX] + c), byn = __ldg(U.f[F_BY] + c);
    double byun = __ldg(U.f[F_BY] + c + sy);
    double rho = 1.0, mx = 0.0, my = 0.0, mz = 0.0, En = 1.0;
    double Ex_p = 0.0, Ey_p = 0.0, Exu_p = 0.0, Bx_part = 0.0, By_part = 0.0, Byu_part = 0.0, Bzh_p = 0.0;
    int sp = 1, sq = 0;   // ring slots of planes k and k-1
    for (int k = kc0; k <= kc1 + 1; k++, c += sz) {
      const int par = (k - kc0) & 1;
      const bool cells = k <= kc1;   // plane k holds cells of this chunk (k = kc1 + 1 only closes plane kc1)
      const bool later = k > kc0;
      const double *P = ctu_ring + sp * T::STAGE, *Q = ctu_ring + sq * T::STAGE;
#define PF(f, off) P[(f) * T::PLANE + (off)]
#define QF(f, off) Q[(f) * T::PLANE + (off)]
      // Eq. 15-17 on the three edges at the lower corner of cell (i, j, k); Table 1 signs as in k_ct
      const double Ex = ct_edge(-PF(4, o), -QF(4, o), PF(8, o), PF(8, oy), PF(3, o), QF(3, o), PF(6, o), PF(6, oy),
                                PF(9, o), PF(9, oy), QF(9, o), QF(9, oy));
      const double Ey = ct_edge(-PF(7, o), -PF(7, ox), PF(2, o), QF(2, o), PF(6, o), PF(6, ox), PF(0, o), QF(0, o),
                                PF(10, o), QF(10, o), PF(10, ox), QF(10, ox));
      const double Ez = ct_edge(-PF(1, o), -PF(1, oy), PF(5, o), PF(5, ox), PF(0, o), PF(0, oy), PF(3, o), PF(3, ox),
                                PF(11, o), PF(11, ox), PF(11, oy), PF(11, oxy));
#undef PF
#undef QF
      ex_s[par][t] = Ex; ez_s[par][t] = Ez;
      cp_async_wait_all();   // plane k+1 (requested one iteration ago) has landed for this thread
      __syncthreads();       // ... and for everybody; the edge fields of this plane are exchanged;
                             // nobody reads plane k-1 any more
      const int sn = 3 - sp - sq;                       // slot of plane k+1; plane k+2 takes over k-1's
      if (k + 2 <= kc1 + 1) request(sq, c + 2 * sz);
      const double Exu = ex_s[par][tu], Ezu = ez_s[par][tu];
      const double Eyr = shfl_dn1(Ey), Ezr = shfl_dn1(Ez), Ezur = shfl_dn1(Ezu);
      // Eq. 32: the z face of plane k needs only the edges of this plane
      const double Bzh = fma_diff(fma_diff(bzn, dtd1, Exu, Ex), -dtd0, Eyr, Ey);
      if (own && inx && iny && (cells || k == n2)) Bout.f[2][c] = Bzh;
      double Bxh = 0.0, Byh = 0.0, Byuh = 0.0;
      if (later) {  // Eq. 30-31 with the edges of planes k-1 and k
        Bxh = fma_diff(Bx_part, dtd2, Ey, Ey_p);
        Byh = fma_diff(By_part, -dtd2, Ex, Ex_p);
        Byuh = fma_diff(Byu_part, -dtd2, Exu, Exu_p);
      }
      const double Bxuh = shfl_dn1(Bxh);
      if (later) {
        const long long cp = c - sz;
        if (own && iny) Bout.f[0][cp] = Bxh;
        if (own && inx) Bout.f[1][cp] = Byh;
        if (own && inx && iny) {  // Eq. 11-12 on the finished cell (i, j, k-1) of U^{n+1}
          Prim p;
          p.rho = rho; p.ir = rcp(rho);
          p.v[0] = mx * p.ir; p.v[1] = my * p.ir; p.v[2] = mz * p.ir;
          p.B[0] = 0.5 * (Bxh + Bxuh); p.B[1] = 0.5 * (Byh + Byuh); p.B[2] = 0.5 * (Bzh_p + Bzh);
          p.P = pressure(g.gamma - 1.0, rho, p.v, En, p.B);
          rate = fmax(rate, cell_rate(g, p, bad));
        }
      }
      if (cells) {
        Bx_part = fma_diff(bxn, -dtd1, Ezu, Ez);
        By_part = fma_diff(byn, dtd0, Ezr, Ez);
        Byu_part = fma_diff(byun, dtd0, Ezur, Ezu);
        // what the next iteration needs from global memory, one plane ahead
        rho = __ldg(U.f[F_RHO] + c); mx = __ldg(U.f[F_MX] + c); my = __ldg(U.f[F_MY] + c);
        mz = __ldg(U.f[F_MZ] + c); En = __ldg(U.f[F_E] + c);
        const long long cn = c + sz;
        bzn = __ldg(U.f[F_BZ] + cn);
        if (k + 1 <= kc1) { bxn = __ldg(U.f[F_BX] + cn); byn = __ldg(U.f[F_BY] + cn); byun = __ldg(U.f[F_BY] + cn + sy); }
      }
      Ex_p = Ex; Ey_p = Ey; Exu_p = Exu; Bzh_p = Bzh;
      sq = sp; sp = sn;
    }
  }
  block_rate_reduce(rate, bad, sc);
}

}  // namespace mhd
