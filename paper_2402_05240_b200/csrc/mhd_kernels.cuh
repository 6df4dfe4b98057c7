// mhd_kernels.cuh -- the CUDA kernels of one VL+CT step, sm_100a, fp64.
//
//   k_fill_ghosts<AXIS>   a0  periodic / outflow ghost layers (O12)
//   k_cfl                 a1  Eq. 11-12 + warp-shuffle/block/atomic min
//   k_predictor_flux      a2  PCM + HLLD on the three lower faces of a cell
//   k_ct                  a3/a7  CT edge fields, Eq. 15-18
//   k_update              a4/a8  Eq. 19-22 / 29-32
//   k_flux_x / k_flux_march<A>  a5+a6  PLMC/PPMC reconstruction fused with HLLD per sweep
//                               direction
#pragma once
#include "../../include/mhd.h"
#include "mhd_grid.cuh"

namespace mhd {

// ---------------------------------------------------------------------------------------
// a0: ghost fill along one axis over the full raw extent of the other two (so edges and
// corners are filled by the x, y, z sequence).  Thread = (ghost slot, p, q); blockIdx.z = field.
// ---------------------------------------------------------------------------------------
template <int AXIS>
__global__ void k_fill_ghosts(State8 U, Geo g) {
  constexpr int A1 = (AXIS + 1) % 3, A2 = (AXIS + 2) % 3;
  const int f = blockIdx.z;
  const int ng = g.ng, na = g.n[AXIS];
  // fastest thread index runs along x whenever x is not the fill axis
  int e0, e1, e2;  // extents of (fast, mid, slow) loop
  if (AXIS == 0) { e0 = 2 * ng; e1 = g.N[1]; e2 = g.N[2]; }
  else if (AXIS == 1) { e0 = g.N[0]; e1 = 2 * ng; e2 = g.N[2]; }
  else { e0 = g.N[0]; e1 = g.N[1]; e2 = 2 * ng; }
  long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  long long tot = (long long)e0 * e1 * e2;
  if (t >= tot) return;
  int c0 = (int)(t % e0);
  int c1 = (int)((t / e0) % e1);
  int c2 = (int)(t / ((long long)e0 * e1));
  int slot, r1, r2;  // ghost slot along AXIS, raw positions along A1, A2
  if (AXIS == 0) { slot = c0; r1 = c1; r2 = c2; }
  else if (AXIS == 1) { slot = c1; r2 = c0; r1 = c2; }   // A1 = z, A2 = x
  else { slot = c2; r1 = c0; r2 = c1; }                 // A1 = x, A2 = y
  int i = (slot < ng) ? slot - ng : na + (slot - ng);   // logical index along AXIS
  const bool normalB = (f == F_BX + AXIS);
  int src;
  if (g.bc[AXIS] == MHD_BC_PERIODIC) {
    src = i % na;
    if (src < 0) src += na;
  } else {
    if (normalB) {  // faces 0..na are active
      if (i == na) return;
      src = (i < 0) ? 0 : na;
    } else {
      src = (i < 0) ? 0 : na - 1;
    }
  }
  const int off = (AXIS == 0) ? g.ox : ng;
  long long base = (long long)r1 * g.s[A1] + (long long)r2 * g.s[A2];
  double *p = U.f[f];
  p[base + (long long)(i + off) * g.s[AXIS]] = p[base + (long long)(src + off) * g.s[AXIS]];
}

// ---------------------------------------------------------------------------------------
// host <-> padded layout: dense array of extent (ex, ey, ez) <-> interior of a field
// ---------------------------------------------------------------------------------------
__global__ void k_unpack(double *__restrict__ dst, const double *__restrict__ src, Geo g, int ex,
                         int ey, int ez) {
  long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  long long tot = (long long)ex * ey * ez;
  if (t >= tot) return;
  int i = (int)(t % ex);
  int j = (int)((t / ex) % ey);
  int k = (int)(t / ((long long)ex * ey));
  dst[cell_index(g, i, j, k)] = src[t];
}

__global__ void k_pack(double *__restrict__ dst, const double *__restrict__ src, Geo g, int ex,
                       int ey, int ez) {
  long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  long long tot = (long long)ex * ey * ez;
  if (t >= tot) return;
  int i = (int)(t % ex);
  int j = (int)((t / ex) % ey);
  int k = (int)(t / ((long long)ex * ey));
  dst[t] = src[cell_index(g, i, j, k)];
}

// ---------------------------------------------------------------------------------------
// a1: CFL.  Positive doubles order like their bit patterns, so the grid-wide minimum is an
// unsigned 64-bit atomicMin (the integer-encoding idea of PAPER.md:325, without the sign
// handling the paper's max needs).  Scalars: sc[0] = bits of the running minimum,
// sc[1] = dt, sc[2] = accumulated time, sc[3] = bad-state flag (as double bits != 0).
// ---------------------------------------------------------------------------------------
struct Scalars {
  unsigned long long min_bits;
  double dt;
  double t_accum;
  unsigned long long bad;
};

__device__ __forceinline__ double warp_min(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

__global__ void __launch_bounds__(256) k_cfl(State8 U, Geo g, Scalars *sc) {
  __shared__ double wmin[8];
  __shared__ int wbad[8];
  const int plane = g.n[0] * g.n[1];
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  const int k = blockIdx.y;
  double tmin = INFINITY;
  int bad = 0;
  if (t < plane) {
    int i = t % g.n[0], j = t / g.n[0];
    Prim p = load_prim(U, g, cell_index(g, i, j, k));
    bad = !(p.rho > 0.0) || !(p.P > 0.0) || !isfinite(p.rho) || !isfinite(p.P);
#pragma unroll
    for (int a = 0; a < 3; a++) {
      double cf = sqrt(fast_speed_sq(g.gamma, p.rho, p.P, p.B[a], p.B[(a + 1) % 3], p.B[(a + 2) % 3]));
      double tt = g.d[a] / (fabs(p.v[a]) + cf);
      if (!isfinite(tt)) bad = 1;
      tmin = fmin(tmin, tt);
    }
  }
  tmin = warp_min(tmin);
  bad = __any_sync(0xffffffffu, bad);
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  if (l == 0) { wmin[w] = tmin; wbad[w] = bad; }
  __syncthreads();
  if (w == 0) {
    int nw = blockDim.x >> 5;
    tmin = (l < nw) ? wmin[l] : INFINITY;
    bad = (l < nw) ? wbad[l] : 0;
    tmin = warp_min(tmin);
    bad = __any_sync(0xffffffffu, bad);
    if (l == 0) {
      if (tmin > 0.0 && tmin < INFINITY)
        atomicMin(&sc->min_bits, (unsigned long long)__double_as_longlong(tmin));
      if (bad) atomicOr(&sc->bad, 1ull);
    }
  }
}

__global__ void k_reset_min(Scalars *sc) {
  sc->min_bits = (unsigned long long)__double_as_longlong(INFINITY);
}

// dt = cfl * min; accumulate time; re-arm the reduction
__global__ void k_finish_dt(Scalars *sc, double cfl) {
  double m = __longlong_as_double((long long)sc->min_bits);
  sc->dt = cfl * m;
  sc->t_accum += sc->dt;
  sc->min_bits = (unsigned long long)__double_as_longlong(INFINITY);
}

__global__ void k_set_dt(Scalars *sc, double dt) { sc->dt = dt; }

// ---------------------------------------------------------------------------------------
// a2: predictor.  One thread per cell of `box`; it forms the PCM states (Eq. 14)
// of its own cell and of its three lower neighbours and solves HLLD on its three lower faces
// (fused PCM+HLLD, the paper's K1).  B_n is the face value.
// Face a is skipped where the lower neighbour lies outside the box.
// ---------------------------------------------------------------------------------------
template <int A>
__device__ __forceinline__ void pcm_face(const State8 &U, const Flux21 &F, const Geo &g,
                                         long long idx, const Prim &pc) {
  Prim pm = load_prim(U, g, idx - g.s[A]);
  double bn;
  W7 WL = to_W<A>(pm, bn);
  W7 WR = to_W<A>(pc, bn);
  F7 f = hlld(g.gamma, WL, WR, __ldg(U.f[F_BX + A] + idx));
  store_flux<A>(F, idx, f);
}

#ifndef MHD_MINB_PRED
#define MHD_MINB_PRED 1
#endif
#ifndef MHD_MINB_FX
#define MHD_MINB_FX 1
#endif
#ifndef MHD_MINB_FM
#define MHD_MINB_FM 1
#endif
__global__ void __launch_bounds__(128, MHD_MINB_PRED) k_predictor_flux(State8 U, Flux21 F, Geo g, Box box) {
  const int lx = box.hi[0] - box.lo[0] + 1, ly = box.hi[1] - box.lo[1] + 1;
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= lx * ly) return;
  int i = box.lo[0] + t % lx, j = box.lo[1] + t / lx, k = box.lo[2] + blockIdx.y;
  long long idx = cell_index(g, i, j, k);
  Prim pc = load_prim(U, g, idx);
  if (i > box.lo[0]) pcm_face<0>(U, F, g, idx, pc);
  if (j > box.lo[1]) pcm_face<1>(U, F, g, idx, pc);
  if (k > box.lo[2]) pcm_face<2>(U, F, g, idx, pc);
}

// ---------------------------------------------------------------------------------------
// a3 / a7: CT.  One thread per index of `box`; it evaluates the three edges on the lower
// corner of its cell.  Face E from the magnetic fluxes per Table 1 (O5):
// on an a-face E_c = -F_a[B_t1], on a b-face E_c = +F_b[B_t2], (a,b,c) cyclic.  The
// cell-centred reference field is Eq. 18 from the state `U` handed in (U^n or U^{n+1/2}).
// ---------------------------------------------------------------------------------------
struct VB {
  double v[3], B[3];
};

__device__ __forceinline__ VB load_vb(const State8 &U, const Geo &g, long long idx) {
  VB q;
  double ir = 1.0 / __ldg(U.f[F_RHO] + idx);
#pragma unroll
  for (int a = 0; a < 3; a++) {
    q.v[a] = __ldg(U.f[F_MX + a] + idx) * ir;
    q.B[a] = 0.5 * (__ldg(U.f[F_BX + a] + idx) + __ldg(U.f[F_BX + a] + idx + g.s[a]));
  }
  return q;
}

template <int C>
__device__ __forceinline__ double eref(const VB &q) {  // Eq. 18: -(v x B)_c
  constexpr int A = (C + 1) % 3, B = (C + 2) % 3;
  return -(q.v[A] * q.B[B] - q.v[B] * q.B[A]);
}

template <int C>
__device__ __forceinline__ void ct_one(const Flux21 &F, const Edge3 &E, const Geo &g, long long idx,
                                       const VB &q00, const VB &q10, const VB &q01, const VB &q11) {
  constexpr int A = (C + 1) % 3, B = (C + 2) % 3;
  const long long sa = g.s[A], sb = g.s[B];
  double Ea0 = -__ldg(F.f[A][5] + idx), Ea1 = -__ldg(F.f[A][5] + idx - sb);
  double Eb0 = __ldg(F.f[B][6] + idx), Eb1 = __ldg(F.f[B][6] + idx - sa);
  double Ma0 = __ldg(F.f[A][0] + idx), Ma1 = __ldg(F.f[A][0] + idx - sb);
  double Mb0 = __ldg(F.f[B][0] + idx), Mb1 = __ldg(F.f[B][0] + idx - sa);
  E.f[C][idx] = ct_edge(Ea0, Ea1, Eb0, Eb1, Ma0, Ma1, Mb0, Mb1, eref<C>(q00), eref<C>(q10),
                        eref<C>(q01), eref<C>(q11));
}

__global__ void __launch_bounds__(128) k_ct(State8 U, Flux21 F, Edge3 E, Geo g, Box box) {
  const int lx = box.hi[0] - box.lo[0] + 1, ly = box.hi[1] - box.lo[1] + 1;
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= lx * ly) return;
  int i = box.lo[0] + t % lx, j = box.lo[1] + t / lx, k = box.lo[2] + blockIdx.y;
  long long idx = cell_index(g, i, j, k);
  const long long sx = g.s[0], sy = g.s[1], sz = g.s[2];
  VB c = load_vb(U, g, idx);
  VB cx = load_vb(U, g, idx - sx), cy = load_vb(U, g, idx - sy), cz = load_vb(U, g, idx - sz);
  VB cxy = load_vb(U, g, idx - sx - sy), cyz = load_vb(U, g, idx - sy - sz),
     czx = load_vb(U, g, idx - sz - sx);
  // E_x: (a,b) = (y,z);  E_y: (z,x);  E_z: (x,y);   args: cells (0,0), (-a,0), (0,-b), (-a,-b)
  ct_one<0>(F, E, g, idx, c, cy, cz, cyz);
  ct_one<1>(F, E, g, idx, c, cz, cx, czx);
  ct_one<2>(F, E, g, idx, c, cx, cy, cxy);
}

// ---------------------------------------------------------------------------------------
// a4 / a8: update (O7).  Uout = Ubase - dts/Delta * flux differences (x, then y, then z);
// face B from the edge fields.  One thread per index of [lo, hi+1]; cells are updated for
// indices <= hi in all axes, the lower a-face where the two transverse indices are <= hi.
// dts = scale * sc->dt (scale 1/2 for the half step, G8).
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_update(State8 Ubase, State8 Uout, Flux21 F, Edge3 E, Geo g,
                                                Box box, const Scalars *sc, double scale) {
  const int lx = box.hi[0] - box.lo[0] + 2, ly = box.hi[1] - box.lo[1] + 2;
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= lx * ly) return;
  int i = box.lo[0] + t % lx, j = box.lo[1] + t / lx, k = box.lo[2] + blockIdx.y;
  const bool inx = i <= box.hi[0], iny = j <= box.hi[1], inz = k <= box.hi[2];
  long long idx = cell_index(g, i, j, k);
  const double dts = scale * sc->dt;
  double dtd[3];
#pragma unroll
  for (int a = 0; a < 3; a++) dtd[a] = dts / g.d[a];
  if (inx && iny && inz) {
    double rho = Ubase.f[F_RHO][idx], En = Ubase.f[F_E][idx];
    double m[3] = {Ubase.f[F_MX][idx], Ubase.f[F_MY][idx], Ubase.f[F_MZ][idx]};
#pragma unroll
    for (int a = 0; a < 3; a++) {
      long long up = idx + g.s[a];
      rho -= dtd[a] * (__ldg(F.f[a][0] + up) - __ldg(F.f[a][0] + idx));
      m[a] -= dtd[a] * (__ldg(F.f[a][1] + up) - __ldg(F.f[a][1] + idx));
      m[(a + 1) % 3] -= dtd[a] * (__ldg(F.f[a][2] + up) - __ldg(F.f[a][2] + idx));
      m[(a + 2) % 3] -= dtd[a] * (__ldg(F.f[a][3] + up) - __ldg(F.f[a][3] + idx));
      En -= dtd[a] * (__ldg(F.f[a][4] + up) - __ldg(F.f[a][4] + idx));
    }
    Uout.f[F_RHO][idx] = rho; Uout.f[F_MX][idx] = m[0]; Uout.f[F_MY][idx] = m[1];
    Uout.f[F_MZ][idx] = m[2]; Uout.f[F_E][idx] = En;
  }
  const bool in[3] = {inx, iny, inz};
#pragma unroll
  for (int a = 0; a < 3; a++) {  // Eq. 20-22 / 30-32
    const int b = (a + 1) % 3, c = (a + 2) % 3;
    if (in[b] && in[c]) {
      Uout.f[F_BX + a][idx] = Ubase.f[F_BX + a][idx] +
                              dtd[c] * (__ldg(E.f[b] + idx + g.s[c]) - __ldg(E.f[b] + idx)) -
                              dtd[b] * (__ldg(E.f[c] + idx + g.s[b]) - __ldg(E.f[c] + idx));
    }
  }
}

// max |div B| over the active cells (diagnostic)
__global__ void __launch_bounds__(256) k_divb(State8 U, Geo g, unsigned long long *out_bits) {
  const int plane = g.n[0] * g.n[1];
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  double m = 0.0;
  if (t < plane) {
    int i = t % g.n[0], j = t / g.n[0];
    long long idx = cell_index(g, i, j, blockIdx.y);
    double d = 0.0;
#pragma unroll
    for (int a = 0; a < 3; a++) d += (U.f[F_BX + a][idx + g.s[a]] - U.f[F_BX + a][idx]) / g.d[a];
    m = fabs(d);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0 && m > 0.0)
    atomicMax(out_bits, (unsigned long long)__double_as_longlong(m));
}

// ---------------------------------------------------------------------------------------
// a5 + a6: high-order reconstruction fused with HLLD, one kernel per sweep direction.
// The interface states never touch HBM (the paper wrote them out and read them back,
// PAPER.md:307): each cell is reconstructed once, its upper-face state W_{L,i+1/2} is handed
// to the thread / iteration that owns face i+1/2.
// ---------------------------------------------------------------------------------------
template <int R>
__device__ __forceinline__ void reconstruct(double gamma, const W7 *win, double bn0, W7 &lo, W7 &hi) {
  if (R == 0) { lo = win[0]; hi = win[0]; }                                   // Eq. 14
  else if (R == 1) plmc(gamma, win[0], win[1], win[2], bn0, lo, hi);          // Eq. 23-28
  else ppmc(gamma, win[0], win[1], win[2], win[3], win[4], bn0, lo, hi);      // O10
}

// x sweep: one thread per cell of an x pencil; the stencil and the hand-over of W_L go
// through shared memory.  Block b owns cells c0 + b*(BX-1) + [0, BX) and faces 1..BX-1 of them.
#define MHD_BX 128
template <int R>
__global__ void __launch_bounds__(MHD_BX, MHD_MINB_FX) k_flux_x(State8 Uh, Flux21 F, Geo g, Box fb) {
  __shared__ double sW[7][MHD_BX + 2 * R + 1];
  __shared__ double sH[7][MHD_BX];
  const int t = threadIdx.x;
  const int cbase = fb.lo[0] - 1 + blockIdx.x * (MHD_BX - 1);
  const int c = cbase + t;
  const int j = fb.lo[1] + blockIdx.y, k = fb.lo[2] + blockIdx.z;
  const int cmax = fb.hi[0];  // last cell to reconstruct (= last face index)
  const long long row = cell_index(g, 0, j, k);
  double bn0 = 0.0;
  W7 W0;
  if (c <= cmax + R) {
    Prim p = load_prim(Uh, g, row + c);
    W0 = to_W<0>(p, bn0);
    sW[0][t + R] = W0.rho; sW[1][t + R] = W0.u; sW[2][t + R] = W0.v; sW[3][t + R] = W0.w;
    sW[4][t + R] = W0.P; sW[5][t + R] = W0.by; sW[6][t + R] = W0.bz;
  }
  if (R > 0 && t < 2 * R) {  // halo: R cells below the block, R above
    int slot = (t < R) ? t : MHD_BX + t;
    int ch = cbase - R + slot;
    if (ch <= cmax + R) {
      double bnh;
      Prim p = load_prim(Uh, g, row + ch);
      W7 Wh = to_W<0>(p, bnh);
      sW[0][slot] = Wh.rho; sW[1][slot] = Wh.u; sW[2][slot] = Wh.v; sW[3][slot] = Wh.w;
      sW[4][slot] = Wh.P; sW[5][slot] = Wh.by; sW[6][slot] = Wh.bz;
    }
  }
  __syncthreads();
  const bool active = (c <= cmax);
  W7 lo, hi;
  if (active) {
    W7 win[2 * R + 1];
#pragma unroll
    for (int s = 0; s < 2 * R + 1; s++) {
      if (s == R) { win[s] = W0; continue; }
      win[s].rho = sW[0][t + s]; win[s].u = sW[1][t + s]; win[s].v = sW[2][t + s];
      win[s].w = sW[3][t + s]; win[s].P = sW[4][t + s]; win[s].by = sW[5][t + s];
      win[s].bz = sW[6][t + s];
    }
    reconstruct<R>(g.gamma, win, bn0, lo, hi);
    sH[0][t] = hi.rho; sH[1][t] = hi.u; sH[2][t] = hi.v; sH[3][t] = hi.w; sH[4][t] = hi.P;
    sH[5][t] = hi.by; sH[6][t] = hi.bz;
  }
  __syncthreads();
  if (active && t >= 1) {
    W7 WL;
    WL.rho = sH[0][t - 1]; WL.u = sH[1][t - 1]; WL.v = sH[2][t - 1]; WL.w = sH[3][t - 1];
    WL.P = sH[4][t - 1]; WL.by = sH[5][t - 1]; WL.bz = sH[6][t - 1];
    F7 f = hlld(g.gamma, WL, lo, __ldg(Uh.f[F_BX] + row + c));
    store_flux<0>(F, row + c, f);
  }
}

// y / z sweep: a thread owns one x position (warps run along x, so every load and store is
// coalesced) and marches along the sweep axis over a chunk of J faces with a rolling window
// of 2R+1 primitive states in registers; each cell's primitives are formed once per chunk.
template <int A, int R>
__global__ void __launch_bounds__(128, MHD_MINB_FM) k_flux_march(State8 Uh, Flux21 F, Geo g, Box fb, int J) {
  constexpr int O = (A == 1) ? 2 : 1;  // the other transverse axis
  const int lx = fb.hi[0] - fb.lo[0] + 1, lo_ = fb.hi[O] - fb.lo[O] + 1;
  long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (long long)lx * lo_) return;
  const int i = fb.lo[0] + (int)(t % lx), o = fb.lo[O] + (int)(t / lx);
  const int f0 = fb.lo[A] + blockIdx.y * J;
  const int f1 = min(f0 + J - 1, fb.hi[A]);
  const long long sA = g.s[A];
  long long idx = (A == 1) ? cell_index(g, i, f0, o) : cell_index(g, i, o, f0);  // cell f0
  W7 win[2 * R + 1];
  double bnc[2 * R + 1];
  // window centred on cell f0-2 (slot 0 is never used): the loop below first shifts it
#pragma unroll
  for (int s = 1; s < 2 * R + 1; s++) {
    Prim p = load_prim(Uh, g, idx + (long long)(s - R - 2) * sA);
    win[s] = to_W<A>(p, bnc[s]);
  }
  win[0] = win[1]; bnc[0] = bnc[1];
  W7 WL = win[1], lo, hi;
  idx -= sA;
  // One reconstruct() call site per kernel: iteration f0-1 only produces W_L of face f0; every
  // cell is then reconstructed by the same instruction sequence, so mirror-image cells give
  // mirror-image states bit for bit.
  for (int f = f0 - 1; f <= f1; f++, idx += sA) {
#pragma unroll
    for (int s = 0; s < 2 * R; s++) { win[s] = win[s + 1]; bnc[s] = bnc[s + 1]; }
    {
      Prim p = load_prim(Uh, g, idx + (long long)R * sA);
      win[2 * R] = to_W<A>(p, bnc[2 * R]);
    }
    reconstruct<R>(g.gamma, win, bnc[R], lo, hi);
    if (f >= f0) {
      F7 fl = hlld(g.gamma, WL, lo, __ldg(Uh.f[F_BX + A] + idx));
      store_flux<A>(F, idx, fl);
    }
    WL = hi;
  }
}

}  // namespace mhd
