// mhd_stage.cuh -- the whole predictor stage (a2 + a3 + a4 of SURVEY.md 8(a)) in ONE kernel:
// PCM + HLLD on the three lower faces of every cell (Eq. 14), CT edge fields
// (Eq. 15-18, Table 1), and the half-step update of the hydro variables and of the face field
// (Eq. 19-22), from U^n straight to the primitive half state W^{n+1/2} and its reference field.
// The 21 predictor fluxes and the 3 predictor edge fields never touch HBM (SURVEY.md 8(f) row 3:
// stage fusion with halo recompute in shared memory): the kernel reads the 8 arrays of U^n and
// writes the 8 arrays of W^{n+1/2} plus 3 of E_ref, 19 array passes instead of 84.
//
// Geometry: a block owns a tile of 30 x (TY-2) cell columns and carries one halo column on each
// side (32 x TY threads, x along the warp); it marches along z.  At plane k every thread solves
// the x-, y- and z-face below its cell, the block exchanges what the neighbours need through
// shared memory (rows) and warp shuffles (lanes), every thread forms the three edge fields on the
// lower corner of its cell, and the cell of plane k-1 -- whose upper z-face and upper edges are
// now known -- is completed and stored.  Halo columns repeat work of the neighbouring block with
// the same instructions on the same operands, hence the same bits.
#pragma once
#include "mhd_kernels.cuh"

namespace mhd {

#define MHD_STAGE_COLS 54
// rows per block; 0 = the three separate kernels of mhd_kernels.cuh
#ifndef MHD_STAGE_TY
#define MHD_STAGE_TY 12
#endif

// Split-phase block barrier (mbarrier): a thread announces that its shared-memory writes of a
// phase are done (arrive, release), goes on with work that needs nobody else's data, and only then
// waits for the others (acquire).  The three exchanges per plane cost almost no idle issue slots
// this way; __syncthreads() stalled every warp until the slowest one had finished its Riemann solve.
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(unsigned long long *bar) {
  asm volatile("{\n.reg .b64 tok;\nmbarrier.arrive.shared::cta.b64 tok, [%0];\n}" ::"r"((unsigned)__cvta_generic_to_shared(bar))
               : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned phase) {
  asm volatile(
      "{\n.reg .pred p;\nMBAR_WAIT:\nmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@p bra MBAR_DONE;\n"
      "bra MBAR_WAIT;\nMBAR_DONE:\n}" ::"r"((unsigned)__cvta_generic_to_shared(bar)),
      "r"(phase)
      : "memory");
}

template <int NT>
__device__ __forceinline__ void prim_store(double (*P)[NT], int t, const Prim &p) {
  P[0][t] = p.rho; P[1][t] = p.ir; P[2][t] = p.v[0]; P[3][t] = p.v[1]; P[4][t] = p.v[2];
  P[5][t] = p.P; P[6][t] = p.B[0]; P[7][t] = p.B[1]; P[8][t] = p.B[2];
}

template <int NT>
__device__ __forceinline__ Prim prim_fetch(double (*P)[NT], int t) {
  Prim p;
  p.rho = P[0][t]; p.ir = P[1][t]; p.v[0] = P[2][t]; p.v[1] = P[3][t]; p.v[2] = P[4][t];
  p.P = P[5][t]; p.B[0] = P[6][t]; p.B[1] = P[7][t]; p.B[2] = P[8][t];
  return p;
}

template <int A>
__device__ __forceinline__ F7 stage_face(const Geo &g, const Prim &pm, const Prim &pc, double bface) {
  double bn;
  W7 WL = to_W<A>(pm, bn);
  W7 WR = to_W<A>(pc, bn);
  return hlld(g.gamma, g.gm1inv, WL, WR, bface);
}

// hb = cells of the half state, [lo, hi] per axis; faces and edges are produced on [lo, hi+1].
// grid: x = tiles (ntx per row of tiles), y = z-chunks of lz planes.
template <int TY>
__global__ void __launch_bounds__(32 * TY, (TY <= 8) ? 2 : 1)
k_predictor_stage(State8 U, State8 Uh, Edge3 Er, Geo g, Box hb, const Scalars *sc, int ntx, int lz) {
  constexpr int NT = 32 * TY;
  extern __shared__ double stage_sm_[];
  double (*sm)[NT] = reinterpret_cast<double (*)[NT]>(stage_sm_);
  // columns of shared memory (NT doubles each): primitive states of two planes, the next plane's
  // U in flight, values exchanged with neighbours, this thread's own values of the previous plane
  enum { PR = 0, PF = 18, XC = 28, EX = 39, CP = 41, FZ = 49 };
  static_assert(FZ + 5 == MHD_STAGE_COLS, "column count");
  const int t = threadIdx.x, lane = t & 31, row = t >> 5;
  const int tbx = blockIdx.x % ntx, tby = blockIdx.x / ntx;
  const int zc0 = hb.lo[2] + (int)blockIdx.y * lz, zc1 = min(zc0 + lz - 1, hb.hi[2]);
  if (zc0 > hb.hi[2]) return;
  const int kbeg = zc0 - 1, kend = zc1 + 1;
  const int i0 = hb.lo[0] + 30 * tbx - 1 + lane, j0 = hb.lo[1] + (TY - 2) * tby - 1 + row;
  // threads beyond the last face index compute on clamped coordinates; nothing of theirs is used
  const int i = min(i0, hb.hi[0] + 1), j = min(j0, hb.hi[1] + 1);
  const bool own = lane >= 1 && lane <= 30 && row >= 1 && row <= TY - 2 && i0 <= hb.hi[0] + 1 && j0 <= hb.hi[1] + 1;
  const bool inx = i0 <= hb.hi[0], iny = j0 <= hb.hi[1];
  const int tl = lane ? t - 1 : t;                  // lower x neighbour (shared memory)
  const int td = row ? t - 32 : t;                  // lower y neighbour
  const int tdl = (row && lane) ? t - 33 : t;       // lower x, lower y
  const int tu = (row < TY - 1) ? t + 32 : t;       // upper y neighbour
  const double gm1 = g.gamma - 1.0;
  const double dts = 0.5 * sc->dt;                  // half step (G8)
  const double dtd0 = dts * g.id[0], dtd1 = dts * g.id[1], dtd2 = dts * g.id[2];

  long long c = cell_index(g, i, j, kbeg);
  // U^n is read THROUGH the boundary map (a0: periodic wrap / outflow clamp; the composed per-axis map that
  // k_fill_ghosts applies, with the normal field's own rule for its faces), so the ghost layers of U^n are
  // not filled between steps: cell (i, j, k) comes from (src_x(i), src_y(j), src_z(k)).  Per thread: the
  // offset of the source column from its own (hydro variables; lower / upper x face; lower / upper y face);
  // the z part is the same for the whole block and advances with the plane.
  const int xs = ghost_src(i, g.n[0], g.bc[0], false), ys = ghost_src(j, g.n[1], g.bc[1], false);
  const int s1 = (int)g.s[1];
  const int o_c = (xs - i) + (ys - j) * s1;
  const int o_xl = o_c + ghost_src(i, g.n[0], g.bc[0], true) - xs;
  const int o_xu = o_c + ghost_src(i + 1, g.n[0], g.bc[0], true) - xs;
  const int o_yl = o_c + (ghost_src(j, g.n[1], g.bc[1], true) - ys) * s1;
  const int o_yu = o_c + (ghost_src(j + 1, g.n[1], g.bc[1], true) - ys) * s1;
  const bool zper = g.bc[2] == MHD_BC_PERIODIC;
  auto znext = [&](int src, int knext, bool face) {   // source index of plane / face knext, given that of knext - 1
    if (zper) return (src + 1 >= g.n[2]) ? 0 : src + 1;
    const int top = face ? g.n[2] : g.n[2] - 1;
    return knext < 0 ? 0 : (knext > top ? top : knext);
  };
  // q = this thread's own column at plane k; zo, zfo = (source plane - k) * stride for cells and for face k + 1
  auto prefetch = [&](long long q, long long zo, long long zfo) {
    const long long qc = q + zo + o_c;
    cp_async8(&sm[PF + 0][t], U.f[F_RHO] + qc); cp_async8(&sm[PF + 1][t], U.f[F_MX] + qc);
    cp_async8(&sm[PF + 2][t], U.f[F_MY] + qc); cp_async8(&sm[PF + 3][t], U.f[F_MZ] + qc);
    cp_async8(&sm[PF + 4][t], U.f[F_E] + qc);
    cp_async8(&sm[PF + 5][t], U.f[F_BX] + q + zo + o_xl); cp_async8(&sm[PF + 6][t], U.f[F_BX] + q + zo + o_xu);
    cp_async8(&sm[PF + 7][t], U.f[F_BY] + q + zo + o_yl); cp_async8(&sm[PF + 8][t], U.f[F_BY] + q + zo + o_yu);
    cp_async8(&sm[PF + 9][t], U.f[F_BZ] + q + zfo + o_c);
    cp_async_commit();
  };
  __shared__ unsigned long long bar[3];
  if (t == 0) { mbar_init(&bar[0], NT); mbar_init(&bar[1], NT); mbar_init(&bar[2], NT); }
  __syncthreads();
  int zs = ghost_src(kbeg, g.n[2], g.bc[2], false);        // source plane of the cells of plane k
  int zf = ghost_src(kbeg, g.n[2], g.bc[2], true);         // source of face k, then of face k + 1
  double bzl = __ldg(U.f[F_BZ] + c + (long long)(zf - kbeg) * g.s[2] + o_c);
  zf = ghost_src(kbeg + 1, g.n[2], g.bc[2], true);
  prefetch(c, (long long)(zs - kbeg) * g.s[2], (long long)(zf - kbeg) * g.s[2]);
  // carried from plane k-1: edge fields, partly updated faces, the cell's hydro variables after
  // the x and y differences
  double Ex_p = 0.0, Ey_p = 0.0, Exu_p = 0.0, Bx_part = 0.0, By_part = 0.0, Byu_part = 0.0, Bzh_p = 0.0;
  double acc[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
  int par = 0;
  for (int k = kbeg; k <= kend; k++, c += g.s[2], par ^= 1) {
    const unsigned ph = (unsigned)(k - kbeg) & 1u;   // every barrier completes once per plane
    const bool later = k > kbeg;   // block-uniform: the first plane only primes the carried values
    cp_async_wait_all();
    double accn[5];
#pragma unroll
    for (int q = 0; q < 5; q++) accn[q] = sm[PF + q][t];
    const double bxl = sm[PF + 5][t], bxu = sm[PF + 6][t], byl = sm[PF + 7][t], byu = sm[PF + 8][t];
    const double bzu = sm[PF + 9][t];
    asm volatile("" ::: "memory");   // the reads above stay ahead of the copies that refill the columns
    if (k < kend) {
      zs = znext(zs, k + 1, false); zf = znext(zf, k + 2, true);
      prefetch(c + g.s[2], (long long)(zs - (k + 1)) * g.s[2], (long long)(zf - (k + 1)) * g.s[2]);
    }
    const Prim pc = make_prim(gm1, accn[0], accn[1], accn[2], accn[3], accn[4], bxl, bxu, byl, byu, bzl, bzu);
    double (*P)[NT] = sm + PR + 9 * par;
    double (*Pp)[NT] = sm + PR + 9 * (par ^ 1);
    prim_store<NT>(P, t, pc);
    const double erx = -(pc.v[1] * pc.B[2] - pc.v[2] * pc.B[1]);   // Eq. 18
    const double ery = -(pc.v[2] * pc.B[0] - pc.v[0] * pc.B[2]);
    const double erz = -(pc.v[0] * pc.B[1] - pc.v[1] * pc.B[0]);
    sm[XC + 4][t] = erx; sm[XC + 5][t] = erz;
    mbar_arrive(&bar[0]);
    double Fx0, Fx6, Fy0, Fy5, Fy6, Fz0 = 0.0, Fz5 = 0.0, Fz6 = 0.0;
    if (later) {  // z face (own column only); completes the hydro variables of the cell below
      F7 f = stage_face<2>(g, prim_fetch<NT>(Pp, t), pc, bzl);
      acc[0] -= dtd2 * (f.m - sm[FZ + 0][t]);
      acc[3] -= dtd2 * (f.mn - sm[FZ + 1][t]);
      acc[1] -= dtd2 * (f.mt1 - sm[FZ + 2][t]);
      acc[2] -= dtd2 * (f.mt2 - sm[FZ + 3][t]);
      acc[4] -= dtd2 * (f.e - sm[FZ + 4][t]);
      sm[FZ + 0][t] = f.m; sm[FZ + 1][t] = f.mn; sm[FZ + 2][t] = f.mt1; sm[FZ + 3][t] = f.mt2; sm[FZ + 4][t] = f.e;
      sm[XC + 2][t] = f.m; sm[XC + 3][t] = f.bz;
      Fz0 = f.m; Fz5 = f.by; Fz6 = f.bz;
    }
    mbar_wait(&bar[0], ph);   // the neighbours' primitive states are in place
    {  // x face: Eq. 19 differences in x for this plane's cell
      F7 f = stage_face<0>(g, prim_fetch<NT>(P, tl), pc, bxl);
      accn[0] -= dtd0 * (shfl_dn1(f.m) - f.m);
      accn[1] -= dtd0 * (shfl_dn1(f.mn) - f.mn);
      accn[2] -= dtd0 * (shfl_dn1(f.mt1) - f.mt1);
      accn[3] -= dtd0 * (shfl_dn1(f.mt2) - f.mt2);
      accn[4] -= dtd0 * (shfl_dn1(f.e) - f.e);
      sm[XC + 0][t] = f.m; sm[XC + 1][t] = f.by;
      Fx0 = f.m; Fx6 = f.bz;
    }
    double Fyh[5];
    {  // y face.  The lowest row only lends its x and z faces and nobody reads its y face (its lower
       // neighbour is itself: a uniform problem); it is solved all the same, because without a branch
       // between them the x and y solves are one basic block and their instructions interleave
       // (stage kernel 1.89 -> 1.85 ms at 256^3 in spite of the extra solves)
      F7 f = stage_face<1>(g, prim_fetch<NT>(P, td), pc, byl);
      Fyh[0] = f.m; Fyh[1] = f.mn; Fyh[2] = f.mt1; Fyh[3] = f.mt2; Fyh[4] = f.e;
      Fy5 = f.by; Fy6 = f.bz;
    }
#pragma unroll
    for (int q = 0; q < 5; q++) sm[XC + 6 + q][t] = Fyh[q];
    Fy0 = Fyh[0];
    mbar_arrive(&bar[1]);
    // Eq. 15-17 on the three edges at the lower corner of cell (i, j, k); Table 1 signs as in k_ct.
    // E_y needs the x neighbour only (shuffles) ...
    const double ery_l = shfl_up1(ery);
    double Ex = 0.0, Ey = 0.0, Ez = 0.0;
    if (later)
      Ey = ct_edge(-Fz5, -shfl_up1(Fz5), Fx6, sm[CP + 2][t], Fz0, shfl_up1(Fz0), Fx0, sm[CP + 3][t],
                   ery, sm[CP + 5][t], ery_l, sm[CP + 7][t]);
    mbar_wait(&bar[1], ph);   // the neighbours' fluxes and reference fields are in place
    const double erx_d = sm[XC + 4][td];
    if (later) {  // ... E_x and E_z the row below
      Ex = ct_edge(-Fy5, -sm[CP + 0][t], Fz6, sm[XC + 3][td], Fy0, sm[CP + 1][t], Fz0, sm[XC + 2][td],
                   erx, erx_d, sm[CP + 4][t], sm[CP + 6][t]);
      Ez = ct_edge(-sm[XC + 1][t], -sm[XC + 1][td], Fy6, shfl_up1(Fy6), Fx0, sm[XC + 0][td], Fy0, shfl_up1(Fy0),
                   erz, shfl_up1(erz), sm[XC + 5][td], sm[XC + 5][tdl]);
      sm[EX + 0][t] = Ex; sm[EX + 1][t] = Ez;
    }
    mbar_arrive(&bar[2]);   // also: nobody reads columns XC+0..5 of another thread beyond this point
    // Eq. 19 differences in y for this plane's cell
    accn[0] -= dtd1 * (sm[XC + 6][tu] - Fyh[0]);
    accn[2] -= dtd1 * (sm[XC + 7][tu] - Fyh[1]);
    accn[3] -= dtd1 * (sm[XC + 8][tu] - Fyh[2]);
    accn[1] -= dtd1 * (sm[XC + 9][tu] - Fyh[3]);
    accn[4] -= dtd1 * (sm[XC + 10][tu] - Fyh[4]);
    // this plane's values for the edges of the next one
    sm[CP + 0][t] = Fy5; sm[CP + 1][t] = Fy0; sm[CP + 2][t] = Fx6; sm[CP + 3][t] = Fx0;
    sm[CP + 4][t] = erx; sm[CP + 5][t] = ery; sm[CP + 6][t] = erx_d; sm[CP + 7][t] = ery_l;
    // what the cell below can already have: velocity, and the x face of Eq. 20
    Prim p;
    p.rho = acc[0]; p.ir = rcp(acc[0]);
    p.v[0] = acc[1] * p.ir; p.v[1] = acc[2] * p.ir; p.v[2] = acc[3] * p.ir;
    const double Bxh = fma_diff(Bx_part, dtd2, Ey, Ey_p);
    const double Bxuh = shfl_dn1(Bxh);
    const double Eyr = shfl_dn1(Ey), Ezr = shfl_dn1(Ez);
    mbar_wait(&bar[2], ph);   // the upper row's edge fields are in place
    if (later) {
      const double Exu = sm[EX + 0][tu], Ezu = sm[EX + 1][tu];
      const double Ezur = shfl_dn1(Ezu);
      // Eq. 22: the z face of plane k needs only the edges of this plane
      const double Bzh = fma_diff(fma_diff(bzl, dtd1, Exu, Ex), -dtd0, Eyr, Ey);
      if (own && inx && iny && (k <= zc1 || k == hb.hi[2] + 1)) Uh.f[F_BZ][c] = Bzh;
      if (k - 1 >= zc0) {  // complete cell (i, j, k-1): Eq. 20-21 with the edges of planes k-1 and k
        const long long cp = c - g.s[2];
        const double Byh = fma_diff(By_part, -dtd2, Ex, Ex_p);
        const double Byuh = fma_diff(Byu_part, -dtd2, Exu, Exu_p);
        p.B[0] = 0.5 * (Bxh + Bxuh); p.B[1] = 0.5 * (Byh + Byuh); p.B[2] = 0.5 * (Bzh_p + Bzh);
        p.P = pressure(gm1, p.rho, p.v, acc[4], p.B);
        if (own) {
          if (inx && iny) {
            Uh.f[F_RHO][cp] = p.rho; Uh.f[F_MX][cp] = p.v[0]; Uh.f[F_MY][cp] = p.v[1];
            Uh.f[F_MZ][cp] = p.v[2]; Uh.f[F_E][cp] = p.P;
            store_eref(Er, cp, p);
          }
          if (iny) Uh.f[F_BX][cp] = Bxh;
          if (inx) Uh.f[F_BY][cp] = Byh;
        }
      }
      Bx_part = fma_diff(bxl, -dtd1, Ezu, Ez);
      By_part = fma_diff(byl, dtd0, Ezr, Ez);
      Byu_part = fma_diff(byu, dtd0, Ezur, Ezu);
      Ex_p = Ex; Ey_p = Ey; Exu_p = Exu; Bzh_p = Bzh;
    }
#pragma unroll
    for (int q = 0; q < 5; q++) acc[q] = accn[q];
    bzl = bzu;
  }
}

}  // namespace mhd
