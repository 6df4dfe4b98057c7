// mhd_small.cuh -- launch-bound grids (32^3, 256 x 16 x 16: a step is eight kernels of a few
// microseconds each): the WHOLE of mhd_advance -- n steps of { dt = CFL / max rate; VL+CT step }
// -- as ONE cooperative kernel.  The stages of a step are the same device
// functions as in the large-grid kernels (hlld, plmc / ppmc, ct_edge, pressure, cell_rate, ...), one
// thread per cell / face / edge in grid-stride loops (no marching, no tiles: at these sizes the whole
// state sits in L2 and parallelism is what is scarce), separated by grid-wide barriers instead of
// kernel boundaries: 7 barriers per step instead of 8 launches.  All fluxes and edge fields go
// through the flux / edge arrays, as in the oracle.
#pragma once
#include <cooperative_groups.h>

#include "mhd_kernels.cuh"

namespace mhd {

struct SmallArgs {
  State8 U, Uh;
  Flux21 F;
  Edge3 E, Er, Bnext;
  Geo g;
  Scalars *sc;
  int n_steps;
  double cfl;      // dt = cfl / max rate, every step ...
  double dt_fixed; // ... or this dt for every step when > 0 (mhd_step)
  unsigned long long *dbg;   // optional: globaltimer stamps of thread 0 at every barrier of the last step
};

// Versions of the per-cell loads for data that OTHER blocks rewrite between the phases of one kernel:
// neither the non-coherent read-only path (__ldg) of the large-grid kernels nor a line that this SM's L1
// cached in an earlier phase may serve them, so every such load is ld.global.cg (L2, where the state of a
// launch-bound grid lives anyway).
#define LD(x) __ldcg(&(x))
__device__ __forceinline__ Prim s_load_prim(const State8 &U, const Geo &g, long long idx) {
  return make_prim(g.gamma - 1.0, LD(U.f[F_RHO][idx]), LD(U.f[F_MX][idx]), LD(U.f[F_MY][idx]), LD(U.f[F_MZ][idx]),
                   LD(U.f[F_E][idx]), LD(U.f[F_BX][idx]), LD(U.f[F_BX][idx + g.s[0]]), LD(U.f[F_BY][idx]),
                   LD(U.f[F_BY][idx + g.s[1]]), LD(U.f[F_BZ][idx]), LD(U.f[F_BZ][idx + g.s[2]]));
}
__device__ __forceinline__ Prim s_load_prim_half(const State8 &Wh, const Geo &g, long long idx) {
  Prim p;
  p.rho = LD(Wh.f[F_RHO][idx]);
  p.ir = 0.0;
#pragma unroll
  for (int a = 0; a < 3; a++) {
    p.B[a] = 0.5 * (LD(Wh.f[F_BX + a][idx]) + LD(Wh.f[F_BX + a][idx + g.s[a]]));
    p.v[a] = LD(Wh.f[F_MX + a][idx]);
  }
  p.P = LD(Wh.f[F_E][idx]);
  return p;
}
template <int C>
__device__ __forceinline__ void s_ct_one(const Flux21 &F, const Edge3 &Er, const Edge3 &E, const Geo &g, long long idx) {
  constexpr int A = (C + 1) % 3, B = (C + 2) % 3;
  const long long sa = g.s[A], sb = g.s[B];
  const double *er = Er.f[C];
  E.f[C][idx] = ct_edge(-LD(F.f[A][5][idx]), -LD(F.f[A][5][idx - sb]), LD(F.f[B][6][idx]), LD(F.f[B][6][idx - sa]),
                        LD(F.f[A][0][idx]), LD(F.f[A][0][idx - sb]), LD(F.f[B][0][idx]), LD(F.f[B][0][idx - sa]),
                        LD(er[idx]), LD(er[idx - sa]), LD(er[idx - sb]), LD(er[idx - sa - sb]));
}
template <int A>
__device__ __forceinline__ double s_face_update(const State8 &U, const Edge3 &E, const Geo &g, long long idx,
                                                const double dtd[3]) {  // Eq. 20-22 / 30-32
  constexpr int B = (A + 1) % 3, C = (A + 2) % 3;
  return LD(U.f[F_BX + A][idx]) + dtd[C] * (LD(E.f[B][idx + g.s[C]]) - LD(E.f[B][idx])) -
         dtd[B] * (LD(E.f[C][idx + g.s[B]]) - LD(E.f[C][idx]));
}

__device__ __forceinline__ void small_decode(long long t, const Box &b, int &i, int &j, int &k) {
  const int lx = b.hi[0] - b.lo[0] + 1, ly = b.hi[1] - b.lo[1] + 1;
  i = b.lo[0] + (int)(t % lx); j = b.lo[1] + (int)((t / lx) % ly); k = b.lo[2] + (int)(t / ((long long)lx * ly));
}
__device__ __forceinline__ long long box_count(const Box &b) {
  return (long long)(b.hi[0] - b.lo[0] + 1) * (b.hi[1] - b.lo[1] + 1) * (b.hi[2] - b.lo[2] + 1);
}

// a0: every index of the padded arrays with a ghost coordinate takes the value of its boundary image
__device__ __forceinline__ void small_fill_ghosts(const State8 &U, const Geo &g, long long t0, long long nt) {
  const int ng = g.ng;
  Box all;
  for (int a = 0; a < 3; a++) { all.lo[a] = -ng; all.hi[a] = g.n[a] + ng - 1; }
  const long long N = box_count(all);
  for (long long t = t0; t < N; t += nt) {
    int i, j, k;
    small_decode(t, all, i, j, k);
    // strictly interior indices (also not the upper boundary face of a normal field) have nothing to do
    if (i >= 0 && i < g.n[0] && j >= 0 && j < g.n[1] && k >= 0 && k < g.n[2]) continue;
    const long long dst = cell_index(g, i, j, k);
    // the cell-centred map serves every field except the normal component of B on an outflow axis
    const int si = ghost_src(i, g.n[0], g.bc[0], false), sj = ghost_src(j, g.n[1], g.bc[1], false);
    const int sk = ghost_src(k, g.n[2], g.bc[2], false);
    const long long src = cell_index(g, si, sj, sk);
#pragma unroll
    for (int f = 0; f < NFIELD; f++) {
      long long s = src;
      if (f >= F_BX && g.bc[f - F_BX] != MHD_BC_PERIODIC) {
        const int a = f - F_BX;
        const int x = (a == 0) ? i : ((a == 1) ? j : k);
        const int sx = ghost_src(x, g.n[a], g.bc[a], true);
        s = (a == 0) ? cell_index(g, sx, sj, sk) : ((a == 1) ? cell_index(g, si, sx, sk) : cell_index(g, si, sj, sx));
      }
      if (s != dst) U.f[f][dst] = LD(U.f[f][s]);
    }
  }
}

// a2: PCM + HLLD on the three lower faces of every cell of `box` (Eq. 14), E_ref of U^n
template <int A>
__device__ __forceinline__ void small_pcm_face(const State8 &U, const Flux21 &F, const Geo &g, long long idx,
                                               const Prim &pc) {
  const Prim pm = s_load_prim(U, g, idx - g.s[A]);
  double bn;
  const W7 WL = to_W<A>(pm, bn);
  const W7 WR = to_W<A>(pc, bn);
  store_flux<A>(F, idx, hlld(g.gamma, g.gm1inv, WL, WR, LD(U.f[F_BX + A][idx])));
}

__device__ __forceinline__ void small_predictor_flux(const SmallArgs &a, const State8 &U, const Box &box, long long t0, long long nt) {
  const long long N = box_count(box);
  for (long long t = t0; t < N; t += nt) {
    int i, j, k;
    small_decode(t, box, i, j, k);
    const long long idx = cell_index(a.g, i, j, k);
    const Prim pc = s_load_prim(U, a.g, idx);
    store_eref(a.Er, idx, pc);
    if (i > box.lo[0]) small_pcm_face<0>(U, a.F, a.g, idx, pc);
    if (j > box.lo[1]) small_pcm_face<1>(U, a.F, a.g, idx, pc);
    if (k > box.lo[2]) small_pcm_face<2>(U, a.F, a.g, idx, pc);
  }
}

// a3 / a7: the three edge fields on the lower corner of every index of `box` (Eq. 15-18)
__device__ __forceinline__ void small_ct(const SmallArgs &a, const Box &box, long long t0, long long nt) {
  const long long N = box_count(box);
  for (long long t = t0; t < N; t += nt) {
    int i, j, k;
    small_decode(t, box, i, j, k);
    const long long idx = cell_index(a.g, i, j, k);
    s_ct_one<0>(a.F, a.Er, a.E, a.g, idx);
    s_ct_one<1>(a.F, a.Er, a.E, a.g, idx);
    s_ct_one<2>(a.F, a.Er, a.E, a.g, idx);
  }
}


// a4 / a8 (O7): out = base - dts/Delta * flux differences (x, then y, then z; reading R2), face field from
// the edge fields.  One index of [lo, hi+1] per thread; cells are updated for indices <= hi in all axes,
// the lower a-face where the two transverse indices are <= hi.
// HALF: the result is stored in primitive form (rho, v, P, face B) with its reference field (Eq. 18).
// else: rho, m, E in place, face B to Bout, CFL rate of the new cell (Eq. 11-12) into `rate`.
template <bool HALF>
__device__ __forceinline__ void small_update(const SmallArgs &a, const State8 &Ubase, const State8 &Uout, const Box &box,
                                             double dts, long long t0, long long nt, double &rate, int &bad) {
  const Geo &g = a.g;
  Box ext = box;
  for (int x = 0; x < 3; x++) ext.hi[x] += 1;
  double dtd[3];
#pragma unroll
  for (int x = 0; x < 3; x++) dtd[x] = dts * g.id[x];
  const long long N = box_count(ext);
  for (long long t = t0; t < N; t += nt) {
    int i, j, k;
    small_decode(t, ext, i, j, k);
    const bool inx = i <= box.hi[0], iny = j <= box.hi[1], inz = k <= box.hi[2];
    const long long idx = cell_index(g, i, j, k);
    double Bl[3];
    Bl[0] = s_face_update<0>(Ubase, a.E, g, idx, dtd);
    Bl[1] = s_face_update<1>(Ubase, a.E, g, idx, dtd);
    Bl[2] = s_face_update<2>(Ubase, a.E, g, idx, dtd);
    if (inx && iny && inz) {
      double rho = LD(Ubase.f[F_RHO][idx]), En = LD(Ubase.f[F_E][idx]);
      double m[3] = {LD(Ubase.f[F_MX][idx]), LD(Ubase.f[F_MY][idx]), LD(Ubase.f[F_MZ][idx])};
#pragma unroll
      for (int x = 0; x < 3; x++) {   // Eq. 19 / 29
        const long long up = idx + g.s[x];
        rho -= dtd[x] * (LD(a.F.f[x][0][up]) - LD(a.F.f[x][0][idx]));
        m[x] -= dtd[x] * (LD(a.F.f[x][1][up]) - LD(a.F.f[x][1][idx]));
        m[(x + 1) % 3] -= dtd[x] * (LD(a.F.f[x][2][up]) - LD(a.F.f[x][2][idx]));
        m[(x + 2) % 3] -= dtd[x] * (LD(a.F.f[x][3][up]) - LD(a.F.f[x][3][idx]));
        En -= dtd[x] * (LD(a.F.f[x][4][up]) - LD(a.F.f[x][4][idx]));
      }
      Prim p;
      p.rho = rho; p.ir = rcp(rho);
      p.B[0] = 0.5 * (Bl[0] + s_face_update<0>(Ubase, a.E, g, idx + g.s[0], dtd));
      p.B[1] = 0.5 * (Bl[1] + s_face_update<1>(Ubase, a.E, g, idx + g.s[1], dtd));
      p.B[2] = 0.5 * (Bl[2] + s_face_update<2>(Ubase, a.E, g, idx + g.s[2], dtd));
#pragma unroll
      for (int x = 0; x < 3; x++) p.v[x] = m[x] * p.ir;
      p.P = pressure(g.gamma - 1.0, rho, p.v, En, p.B);
      if (HALF) {
        Uout.f[F_RHO][idx] = rho; Uout.f[F_MX][idx] = p.v[0]; Uout.f[F_MY][idx] = p.v[1];
        Uout.f[F_MZ][idx] = p.v[2]; Uout.f[F_E][idx] = p.P;
        store_eref(a.Er, idx, p);
      } else {
        Uout.f[F_RHO][idx] = rho; Uout.f[F_MX][idx] = m[0]; Uout.f[F_MY][idx] = m[1];
        Uout.f[F_MZ][idx] = m[2]; Uout.f[F_E][idx] = En;
        rate = fmax(rate, cell_rate(g, p, bad));
      }
    }
    // the face arrays of Uout are never those of Ubase (the upper-face reads above would race)
    if (iny && inz) Uout.f[F_BX][idx] = Bl[0];
    if (inz && inx) Uout.f[F_BY][idx] = Bl[1];
    if (inx && iny) Uout.f[F_BZ][idx] = Bl[2];
  }
}

// a5 + a6: reconstruction of the two cells next to a face + HLLD, every face of `fb` (faces lo..hi along A)
template <int A, int RC>
__device__ __forceinline__ void small_face_flux(const SmallArgs &a, const Box &fb, long long t0, long long nt) {
  constexpr int R = recon_radius(RC);
  const Geo &g = a.g;
  const long long N = box_count(fb), sA = g.s[A];
  for (long long t = t0; t < N; t += nt) {
    int i, j, k;
    small_decode(t, fb, i, j, k);
    const long long idx = cell_index(g, i, j, k);
    W7 WL, WR, lo, hi;
    // one reconstruction call site (reading R8): first the cell below the face (its upper state), then
    // the cell above it (its lower state)
#pragma unroll
    for (int side = 0; side < 2; side++) {
      const long long c = idx - (1 - side) * sA;
      W7 win[2 * R + 1];
      double bnc[2 * R + 1];
#pragma unroll
      for (int s = 0; s < 2 * R + 1; s++) win[s] = to_W<A>(s_load_prim_half(a.Uh, g, c + (long long)(s - R) * sA), bnc[s]);
      reconstruct<RC>(g.gamma, win, bnc[R], lo, hi);
      if (side == 0) WL = hi; else WR = lo;
    }
    store_flux<A>(a.F, idx, hlld(g.gamma, g.gm1inv, WL, WR, LD(a.Uh.f[F_BX + A][idx])));
  }
}

#ifndef MHD_SMALL_MINB
#define MHD_SMALL_MINB 2
#endif
template <int RC>
__global__ void __launch_bounds__(256, MHD_SMALL_MINB) k_small_steps(SmallArgs a) {
  namespace cg = cooperative_groups;
  cg::grid_group grid = cg::this_grid();
  const long long t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x, nt = (long long)gridDim.x * blockDim.x;
  const Geo &g = a.g;
  const int r = recon_radius(RC);
  State8 U = a.U;
  Edge3 Bnext = a.Bnext;
  Box pb, hb, eb, ab, cb, fx, fy, fz;
  for (int x = 0; x < 3; x++) {
    pb.lo[x] = -2 - r; pb.hi[x] = g.n[x] + r + 1;   // predictor fluxes (R1)
    hb.lo[x] = -1 - r; hb.hi[x] = g.n[x] + r;       // half-step state
    eb.lo[x] = hb.lo[x]; eb.hi[x] = hb.hi[x] + 1;   // predictor edges
    ab.lo[x] = 0; ab.hi[x] = g.n[x] - 1;            // active cells
    cb.lo[x] = 0; cb.hi[x] = g.n[x];                // corrector edges
    fx.lo[x] = fy.lo[x] = fz.lo[x] = -1; fx.hi[x] = fy.hi[x] = fz.hi[x] = g.n[x];
  }
  fx.lo[0] = 0; fy.lo[1] = 0; fz.lo[2] = 0;         // faces 0..n along the sweep, transverse -1..n
  volatile unsigned long long *rate_bits = &a.sc->rate_bits;
  int nstamp = 0;
  auto stamp = [&]() {
    if (a.dbg && t0 == 0) { unsigned long long tm; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(tm)); a.dbg[nstamp++ & 15] = tm; }
  };
  for (int s = 0; s < a.n_steps; s++) {
    // Eq. 11: every thread forms the same dt from the reduced rate of the current state
    nstamp = 0; stamp();
    const double dt = a.dt_fixed > 0.0 ? a.dt_fixed : a.cfl / __longlong_as_double((long long)*rate_bits);
    small_fill_ghosts(U, g, t0, nt);                                   // a0
    grid.sync(); stamp();
    if (t0 == 0) {   // (everybody has read the rate: re-arm the reduction)
      a.sc->dt = dt;
      if (!(a.dt_fixed > 0.0)) a.sc->t_accum += dt;
      *rate_bits = 0ull;
    }
    small_predictor_flux(a, U, pb, t0, nt);                            // a2
    grid.sync(); stamp();
    small_ct(a, eb, t0, nt);                                           // a3
    grid.sync(); stamp();
    double rate = 0.0;
    int bad = 0;
    small_update<true>(a, U, a.Uh, hb, 0.5 * dt, t0, nt, rate, bad);   // a4 (G8: dt/2)
    grid.sync(); stamp();
    small_face_flux<0, RC>(a, fx, t0, nt);                             // a5 + a6
    small_face_flux<1, RC>(a, fy, t0, nt);
    small_face_flux<2, RC>(a, fz, t0, nt);
    grid.sync(); stamp();
    small_ct(a, cb, t0, nt);                                           // a7 (G12)
    grid.sync(); stamp();
    State8 out = U;
    for (int x = 0; x < 3; x++) out.f[F_BX + x] = Bnext.f[x];
    small_update<false>(a, U, out, ab, dt, t0, nt, rate, bad);         // a8 + a1 of the new state
    block_rate_reduce(rate, bad, a.sc);
    for (int x = 0; x < 3; x++) { Bnext.f[x] = U.f[F_BX + x]; U.f[F_BX + x] = out.f[F_BX + x]; }
    grid.sync(); stamp();
  }
}

#undef LD

}  // namespace mhd
