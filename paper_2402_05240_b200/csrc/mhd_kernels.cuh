// mhd_kernels.cuh -- the CUDA kernels of one VL+CT step, sm_100a, fp64.
//
//   k_fill_ghosts         a0  periodic / outflow ghost layers (O12)
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
// a0: ghost fill (O12), all three axes in one launch.  Filling x, then y, then z
// over the full extent of the other two axes gives every ghost cell the value of the cell at
// (src_x(i), src_y(j), src_z(k)), where src_a is the per-axis boundary map; this kernel applies the
// composed map directly.  Periodic: src = i mod n (so the upper boundary face of the normal field
// copies face 0).  Outflow: nearest active cell, or nearest active face 0..n for the normal field.
// blockIdx.z = field; blockIdx.y = a row of the ghost region, decoded once per block (no per-thread
// divisions): rows [0, R0) = (j, z slot) of the z ghost slabs over all (i, j); [R0, R0 + R1) = (y slot,
// k) of the y ghost slabs over all i and active k -- one thread per i along the row, coalesced; the
// remaining block rows cover the x ghost columns over active (j, k), 2 ng values per grid row and
// blockDim.x / (2 ng) grid rows per block.  Disjoint, together every index with a ghost coordinate.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ int ghost_src(int i, int n, int bc, bool normalB) {
  if (bc == MHD_BC_PERIODIC) { int s = i % n; return s < 0 ? s + n : s; }
  if (normalB) return i < 0 ? 0 : (i > n ? n : i);
  return i < 0 ? 0 : (i >= n ? n - 1 : i);
}

__device__ __forceinline__ int ghost_slot(int slot, int ng, int n) {  // slot 0..2ng-1 -> logical index
  return slot < ng ? slot - ng : n + (slot - ng);
}

#define MHD_GHOST_RPB 8   // rows per block (blocks of one short row each are bound by the block launch rate)

__global__ void __launch_bounds__(1024) k_fill_ghosts(State8 U, Geo g) {
  const int f = blockIdx.z;
  const int ng = g.ng, n0 = g.n[0], n1 = g.n[1], n2 = g.n[2];
  const int L0 = n0 + 2 * ng, L1 = n1 + 2 * ng;
  const int R0 = L1 * 2 * ng, R1 = 2 * ng * n2;
  const int per = blockDim.x / (2 * ng);                      // grid rows per block row in the x-column part
  const long long nrow2 = (long long)n1 * n2;
  const int R2 = (int)((nrow2 + per - 1) / per);
  double *p = U.f[f];
  double v[MHD_GHOST_RPB];
  long long dst[MHD_GHOST_RPB];
#pragma unroll
  for (int u = 0; u < MHD_GHOST_RPB; u++) {
    int r = blockIdx.y * MHD_GHOST_RPB + u;
    dst[u] = -1;
    if (r >= R0 + R1 + R2) continue;
    int i, j, k;
    if (r < R0 + R1) {
      i = (int)(blockIdx.x * blockDim.x + threadIdx.x);
      if (i >= L0) continue;
      i -= ng;
      if (r < R0) { j = r % L1 - ng; k = ghost_slot(r / L1, ng, n2); }
      else { r -= R0; j = ghost_slot(r % (2 * ng), ng, n1); k = r / (2 * ng); }
    } else {
      if (blockIdx.x != 0) continue;
      const int q = (int)threadIdx.x / (2 * ng);
      if (q >= per) continue;
      const long long row = (long long)(r - R0 - R1) * per + q;   // (j, k) = row % n1, row / n1
      if (row >= nrow2) continue;
      i = ghost_slot((int)threadIdx.x - q * 2 * ng, ng, n0);
      j = (int)(row % n1); k = (int)(row / n1);
    }
    const int si = ghost_src(i, n0, g.bc[0], f == F_BX);
    const int sj = ghost_src(j, n1, g.bc[1], f == F_BY);
    const int sk = ghost_src(k, n2, g.bc[2], f == F_BZ);
    if (si == i && sj == j && sk == k) continue;  // an active face of the normal field on an outflow side
    dst[u] = cell_index(g, i, j, k);
    v[u] = p[cell_index(g, si, sj, sk)];
  }
#pragma unroll
  for (int u = 0; u < MHD_GHOST_RPB; u++)
    if (dst[u] >= 0) p[dst[u]] = v[u];
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
// a1: CFL.  Each thread forms the largest signal rate (|v_a| + c_f,a) / Delta_a of its cell; the
// grid-wide maximum goes through warp shuffles, shared memory and one atomic per block
// (PAPER.md:317-327).  Positive doubles order like their bit patterns, so the atomic is an
// unsigned 64-bit atomicMax (the integer-encoding idea of PAPER.md:325 without the sign
// handling).  dt = cfl / max rate  (= cfl * min Delta_a / (|v_a| + c_f,a), Eq. 11).
// ---------------------------------------------------------------------------------------
struct Scalars {
  unsigned long long rate_bits;  // running maximum of the signal rate
  double dt;
  double t_accum;
  unsigned long long bad;
};

__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = max_(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

__device__ __forceinline__ double cell_rate(const Geo &g, const Prim &p, int &bad) {
  bad |= !(p.rho > 0.0) || !(p.P > 0.0) || !isfinite(p.rho) || !isfinite(p.P);
  double r = 0.0;
#pragma unroll
  for (int a = 0; a < 3; a++) {
    double cf = sqrt_(fast_speed_sq(g.gamma, p.ir, p.P, p.B[a], p.B[(a + 1) % 3], p.B[(a + 2) % 3]));
    r = max_(r, (fabs(p.v[a]) + cf) * g.id[a]);
  }
  bad |= !isfinite(r) || !(r > 0.0);
  return r;
}

__device__ __forceinline__ void block_rate_reduce(double r, int bad, Scalars *sc) {
  __shared__ double wmax[32];
  __shared__ int wbad[32];
  r = warp_max(r);
  bad = __any_sync(0xffffffffu, bad);
  const int t = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
  const int nt = blockDim.x * blockDim.y * blockDim.z;
  const int w = t >> 5, l = t & 31;
  if (l == 0) { wmax[w] = r; wbad[w] = bad; }
  __syncthreads();
  if (w == 0) {
    int nw = (nt + 31) >> 5;
    r = (l < nw) ? wmax[l] : 0.0;
    bad = (l < nw) ? wbad[l] : 0;
    r = warp_max(r);
    bad = __any_sync(0xffffffffu, bad);
    if (l == 0) {
      if (r > 0.0 && r < INFINITY) atomicMax(&sc->rate_bits, (unsigned long long)__double_as_longlong(r));
      if (bad) atomicOr(&sc->bad, 1ull);
    }
  }
}

__global__ void __launch_bounds__(256) k_cfl(State8 U, Geo g, Scalars *sc) {
  const int plane = g.n[0] * g.n[1];
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  const int k = blockIdx.y;
  double r = 0.0;
  int bad = 0;
  if (t < plane) {
    int i = t % g.n[0], j = t / g.n[0];
    Prim p = load_prim(U, g, cell_index(g, i, j, k));
    r = cell_rate(g, p, bad);
  }
  block_rate_reduce(r, bad, sc);
}

// new state (mhd_set_state, mhd_set_domain): the running maximum and the non-physical-state flag
// belong to the state they were computed on
__global__ void k_reset_rate(Scalars *sc) { sc->rate_bits = 0ull; sc->bad = 0ull; }

// dt = cfl / max rate; accumulate time; re-arm the reduction
__global__ void k_finish_dt(Scalars *sc, double cfl) {
  double m = __longlong_as_double((long long)sc->rate_bits);
  sc->dt = cfl / m;
  sc->t_accum += sc->dt;
  sc->rate_bits = 0ull;
}

// dt given by the caller; re-arm the reduction (the full update accumulates the next rate)
__global__ void k_set_dt(Scalars *sc, double dt) { sc->dt = dt; sc->rate_bits = 0ull; }

// Eq. 18: cell-centred reference field E = -(v x B)
__device__ __forceinline__ void store_eref(const Edge3 &Er, long long idx, const Prim &p) {
  Er.f[0][idx] = -(p.v[1] * p.B[2] - p.v[2] * p.B[1]);
  Er.f[1][idx] = -(p.v[2] * p.B[0] - p.v[0] * p.B[2]);
  Er.f[2][idx] = -(p.v[0] * p.B[1] - p.v[1] * p.B[0]);
}

// Asynchronous 8-byte global -> shared copies (LDGSTS) into a per-thread column of shared memory:
// operands that are needed later (the neighbour cells of the predictor, the fused hydro update of
// the z sweep) are requested early, and their HBM latency hides behind a Riemann solve or a whole
// reconstruction at no cost in registers.
__device__ __forceinline__ void cp_async8(double *smem, const double *gmem) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
// all groups but the most recently committed one are complete
__device__ __forceinline__ void cp_async_wait_but_last() { asm volatile("cp.async.wait_group 1;" ::: "memory"); }

// ---------------------------------------------------------------------------------------
// a2: predictor.  One thread per cell of `box`; it forms the PCM states (Eq. 14)
// of its own cell and of its three lower neighbours and solves HLLD on its three lower faces
// (fused PCM+HLLD, the paper's K1).  B_n is the face value.
// Face a is skipped where the lower neighbour lies outside the box.  The thread also leaves
// the reference field of its cell (Eq. 18) for the CT kernel.
// ---------------------------------------------------------------------------------------
#define MHD_PRED_T 128
// neighbour cell `slot` (0, 1, 2 = lower x, y, z neighbour) of the calling thread, staged by cp.async
__device__ __forceinline__ void stage_cell(double (*st)[MHD_PRED_T], int slot, const State8 &U, const Geo &g,
                                           long long c) {
  const int t = threadIdx.x, o = 11 * slot;
  cp_async8(&st[o + 0][t], U.f[F_RHO] + c); cp_async8(&st[o + 1][t], U.f[F_MX] + c);
  cp_async8(&st[o + 2][t], U.f[F_MY] + c); cp_async8(&st[o + 3][t], U.f[F_MZ] + c);
  cp_async8(&st[o + 4][t], U.f[F_E] + c);
#pragma unroll
  for (int b = 0; b < 3; b++) {
    cp_async8(&st[o + 5 + 2 * b][t], U.f[F_BX + b] + c);
    cp_async8(&st[o + 6 + 2 * b][t], U.f[F_BX + b] + c + g.s[b]);
  }
}

template <int A>
__device__ __forceinline__ void pcm_face(double (*st)[MHD_PRED_T], const State8 &U, const Flux21 &F, const Geo &g,
                                         long long idx, const Prim &pc) {
  const int t = threadIdx.x, o = 11 * A;
  Prim pm = make_prim(g.gamma - 1.0, st[o][t], st[o + 1][t], st[o + 2][t], st[o + 3][t], st[o + 4][t], st[o + 5][t],
                      st[o + 6][t], st[o + 7][t], st[o + 8][t], st[o + 9][t], st[o + 10][t]);
  double bn;
  W7 WL = to_W<A>(pm, bn);
  W7 WR = to_W<A>(pc, bn);
  F7 f = hlld(g.gamma, g.gm1inv, WL, WR, __ldg(U.f[F_BX + A] + idx));
  store_flux<A>(F, idx, f);
}

// minimum resident blocks per SM asked of ptxas (register caps), tuned on B200 at 256^3:
// the fp64-bound kernels want warps (128 registers), the HBM-bound ones want loads in flight
#ifndef MHD_MINB_UPD
#define MHD_MINB_UPD 2
#endif
// (6 blocks = 40 registers spilled 16 B once the CFL rate's roots became cubic steps; 4 blocks, 60 registers:
// 0.43 -> 0.40 ms at 256^3; 3 and 5 blocks 0.42, 0.40; 8 blocks 0.46)
#ifndef MHD_MINB_UPDB
#define MHD_MINB_UPDB 4
#endif
#ifndef MHD_MINB_CT
#define MHD_MINB_CT 3
#endif
#ifndef MHD_MINB_PRED
#define MHD_MINB_PRED 5
#endif
#ifndef MHD_MINB_FX
#define MHD_MINB_FX 5
#endif
#ifndef MHD_MINB_FM
#define MHD_MINB_FM 3
#endif
#ifndef MHD_MINB_FMZ
#define MHD_MINB_FMZ 3
#endif
#ifndef MHD_MINB_FM_PPM
#define MHD_MINB_FM_PPM 3
#endif
#ifndef MHD_MINB_FX_PPM
#define MHD_MINB_FX_PPM 4
#endif
// the 5-cell z sweep with the update wants 212 registers (2.08 -> 2.00 ms at 256^3 against 3 blocks of 168)
#ifndef MHD_MINB_FMZ_PPM
#define MHD_MINB_FMZ_PPM 2
#endif
__global__ void __launch_bounds__(MHD_PRED_T, MHD_MINB_PRED) k_predictor_flux(State8 U, Flux21 F, Edge3 Er, Geo g, Box box) {
  __shared__ double st[33][MHD_PRED_T];
  const int lx = box.hi[0] - box.lo[0] + 1, ly = box.hi[1] - box.lo[1] + 1;
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= lx * ly) return;
  int i = box.lo[0] + t % lx, j = box.lo[1] + t / lx, k = box.lo[2] + blockIdx.y;
  long long idx = cell_index(g, i, j, k);
  // the three lower neighbours are requested first (they lie inside the arrays even for the first
  // layer of the box, whose faces are not solved); the thread's own cell goes through registers
  stage_cell(st, 0, U, g, idx - g.s[0]);
  stage_cell(st, 1, U, g, idx - g.s[1]);
  stage_cell(st, 2, U, g, idx - g.s[2]);
  cp_async_commit();
  Prim pc = load_prim(U, g, idx);
  store_eref(Er, idx, pc);
  cp_async_wait_all();
  if (i > box.lo[0]) pcm_face<0>(st, U, F, g, idx, pc);
  if (j > box.lo[1]) pcm_face<1>(st, U, F, g, idx, pc);
  if (k > box.lo[2]) pcm_face<2>(st, U, F, g, idx, pc);
}

// ---------------------------------------------------------------------------------------
// a3 / a7: CT.  One thread per index of `box`; it evaluates the three edges on the lower
// corner of its cell.  Face E from the magnetic fluxes per Table 1 (O5):
// on an a-face E_c = -F_a[B_t1], on a b-face E_c = +F_b[B_t2], (a,b,c) cyclic.  The
// cell-centred reference field (Eq. 18) was left in `Er` by the kernel that produced the state
// (predictor: U^n; half update: U^{n+1/2}), so this kernel is pure stencil traffic.
// ---------------------------------------------------------------------------------------
template <int C>
__device__ __forceinline__ void ct_one(const Flux21 &F, const Edge3 &Er, const Edge3 &E, const Geo &g,
                                       long long idx) {
  constexpr int A = (C + 1) % 3, B = (C + 2) % 3;
  const long long sa = g.s[A], sb = g.s[B];
  double Ea0 = -__ldg(F.f[A][5] + idx), Ea1 = -__ldg(F.f[A][5] + idx - sb);
  double Eb0 = __ldg(F.f[B][6] + idx), Eb1 = __ldg(F.f[B][6] + idx - sa);
  double Ma0 = __ldg(F.f[A][0] + idx), Ma1 = __ldg(F.f[A][0] + idx - sb);
  double Mb0 = __ldg(F.f[B][0] + idx), Mb1 = __ldg(F.f[B][0] + idx - sa);
  const double *er = Er.f[C];
  E.f[C][idx] = ct_edge(Ea0, Ea1, Eb0, Eb1, Ma0, Ma1, Mb0, Mb1, __ldg(er + idx), __ldg(er + idx - sa),
                        __ldg(er + idx - sb), __ldg(er + idx - sa - sb));
}

__global__ void __launch_bounds__(256, MHD_MINB_CT) k_ct(Flux21 F, Edge3 Er, Edge3 E, Geo g, Box box) {
  const int lx = box.hi[0] - box.lo[0] + 1, ly = box.hi[1] - box.lo[1] + 1;
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= lx * ly) return;
  int i = box.lo[0] + t % lx, j = box.lo[1] + t / lx, k = box.lo[2] + blockIdx.y;
  long long idx = cell_index(g, i, j, k);
  ct_one<0>(F, Er, E, g, idx);
  ct_one<1>(F, Er, E, g, idx);
  ct_one<2>(F, Er, E, g, idx);
}

// ---------------------------------------------------------------------------------------
// a4 / a8: update (O7).  U_out = U^n - dts/Delta * flux differences (x, then y, then z);
// face B from the edge fields.  HALF = false: the hydro variables of U^{n+1} were already written by
// the z sweep (k_flux_march<2,R,true>); this kernel updates the face field (Eq. 30-32) and forms the
// CFL rate of the new state.  One thread per index of [lo, hi+1]; cells are updated for
// indices <= hi in all axes, the lower a-face where the two transverse indices are <= hi.
// dts = scale * sc->dt (scale 1/2 for the half step, G8).
// HALF = true: the result is stored in primitive form (rho, v, P, face B; see load_prim_half)
// together with its reference field (Eq. 18); the thread then also needs its three UPPER faces
// for the cell-centred field (Eq. 13), which it updates itself (same expression, same bits as the
// owner of that face stores).
// ---------------------------------------------------------------------------------------
template <int A>
__device__ __forceinline__ double face_update(const State8 &U, const Edge3 &E, const Geo &g, long long idx,
                                              const double dtd[3]) {  // Eq. 20-22 / 30-32
  constexpr int B = (A + 1) % 3, C = (A + 2) % 3;
  return __ldg(U.f[F_BX + A] + idx) + dtd[C] * (__ldg(E.f[B] + idx + g.s[C]) - __ldg(E.f[B] + idx)) -
         dtd[B] * (__ldg(E.f[C] + idx + g.s[B]) - __ldg(E.f[C] + idx));
}

template <bool HALF>
__global__ void __launch_bounds__(256, HALF ? MHD_MINB_UPD : MHD_MINB_UPDB) k_update(State8 Ubase, State8 Uout, Flux21 F, Edge3 E, Edge3 Er,
                                                Geo g, Box box, Scalars *sc, double scale) {
  const int lx = box.hi[0] - box.lo[0] + 2, ly = box.hi[1] - box.lo[1] + 2;
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  const bool valid = t < lx * ly;
  if (!valid) t = 0;
  int i = box.lo[0] + t % lx, j = box.lo[1] + t / lx, k = box.lo[2] + blockIdx.y;
  const bool inx = valid && i <= box.hi[0], iny = valid && j <= box.hi[1], inz = valid && k <= box.hi[2];
  long long idx = cell_index(g, i, j, k);
  const double dts = scale * sc->dt;
  double dtd[3];
#pragma unroll
  for (int a = 0; a < 3; a++) dtd[a] = dts * g.id[a];
  // evaluated unconditionally (every operand lies inside the padded arrays; results of indices
  // that do not own the face are simply not stored): no branch ahead of the loads, so all of the
  // kernel's ~60 loads go out in one batch -- this kernel lives on loads in flight
  double Bl[3];
  Bl[0] = face_update<0>(Ubase, E, g, idx, dtd);
  Bl[1] = face_update<1>(Ubase, E, g, idx, dtd);
  Bl[2] = face_update<2>(Ubase, E, g, idx, dtd);
  double rate = 0.0;
  int bad = 0;
  const bool in_cell = inx && iny && inz;
  {
    double rho = __ldg(Ubase.f[F_RHO] + idx), En = __ldg(Ubase.f[F_E] + idx);
    double m[3] = {__ldg(Ubase.f[F_MX] + idx), __ldg(Ubase.f[F_MY] + idx), __ldg(Ubase.f[F_MZ] + idx)};
    if (HALF) {  // Eq. 19; in the full step the z sweep has already applied Eq. 29 to these five
#pragma unroll
      for (int a = 0; a < 3; a++) {
        long long up = idx + g.s[a];
        rho -= dtd[a] * (__ldg(F.f[a][0] + up) - __ldg(F.f[a][0] + idx));
        m[a] -= dtd[a] * (__ldg(F.f[a][1] + up) - __ldg(F.f[a][1] + idx));
        m[(a + 1) % 3] -= dtd[a] * (__ldg(F.f[a][2] + up) - __ldg(F.f[a][2] + idx));
        m[(a + 2) % 3] -= dtd[a] * (__ldg(F.f[a][3] + up) - __ldg(F.f[a][3] + idx));
        En -= dtd[a] * (__ldg(F.f[a][4] + up) - __ldg(F.f[a][4] + idx));
      }
    }
    // primitives of the updated cell: the half step stores them; the full step needs them for the
    // next step's CFL rate (Eq. 11), folded in here so that the state is not read once more
    Prim p;
    p.rho = rho; p.ir = rcp(rho);
    p.B[0] = 0.5 * (Bl[0] + face_update<0>(Ubase, E, g, idx + g.s[0], dtd));
    p.B[1] = 0.5 * (Bl[1] + face_update<1>(Ubase, E, g, idx + g.s[1], dtd));
    p.B[2] = 0.5 * (Bl[2] + face_update<2>(Ubase, E, g, idx + g.s[2], dtd));
#pragma unroll
    for (int a = 0; a < 3; a++) p.v[a] = m[a] * p.ir;
    p.P = pressure(g.gamma - 1.0, rho, p.v, En, p.B);
    if (in_cell) {
      if (HALF) {
        Uout.f[F_RHO][idx] = rho; Uout.f[F_MX][idx] = p.v[0]; Uout.f[F_MY][idx] = p.v[1];
        Uout.f[F_MZ][idx] = p.v[2]; Uout.f[F_E][idx] = p.P;
        store_eref(Er, idx, p);
      } else {
        rate = cell_rate(g, p, bad);
      }
    }
  }
  // the face arrays of Uout are never those of Ubase (the upper-face reads above would race)
  if (iny && inz) Uout.f[F_BX][idx] = Bl[0];
  if (inz && inx) Uout.f[F_BY][idx] = Bl[1];
  if (inx && iny) Uout.f[F_BZ][idx] = Bl[2];
  if (!HALF) block_rate_reduce(rate, bad, sc);
}

// mhd_get_half_state: primitive half state -> conserved variables of the ABI
__global__ void k_half_to_cons(State8 Wh, State8 Out, Geo g, Box box) {
  const int lx = box.hi[0] - box.lo[0] + 1, ly = box.hi[1] - box.lo[1] + 1;
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= lx * ly) return;
  int i = box.lo[0] + t % lx, j = box.lo[1] + t / lx, k = box.lo[2] + blockIdx.y;
  long long idx = cell_index(g, i, j, k);
  Prim p = load_prim_half(Wh, g, idx);
  double v2 = p.v[0] * p.v[0] + p.v[1] * p.v[1] + p.v[2] * p.v[2];
  double b2 = p.B[0] * p.B[0] + p.B[1] * p.B[1] + p.B[2] * p.B[2];
  Out.f[F_RHO][idx] = p.rho;
  Out.f[F_MX][idx] = p.rho * p.v[0]; Out.f[F_MY][idx] = p.rho * p.v[1]; Out.f[F_MZ][idx] = p.rho * p.v[2];
  Out.f[F_E][idx] = p.P * g.gm1inv + 0.5 * p.rho * v2 + 0.5 * b2;
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
// recon code RC (include/mhd.h MHD_RECON_*) -> stencil radius: PCM 0, PLMC/PLMP 1, PPMC/PPMP 2
__host__ __device__ constexpr int recon_radius(int rc) { return rc == 0 ? 0 : ((rc == 1 || rc == 3) ? 1 : 2); }

template <int RC>
__device__ __forceinline__ void reconstruct(double gamma, const W7 *win, double bn0, W7 &lo, W7 &hi) {
  if (RC == 0) { lo = win[0]; hi = win[0]; }                                   // Eq. 14
  else if (RC == 1) plmc(gamma, win[0], win[1], win[2], bn0, lo, hi);          // Eq. 23-28
  else if (RC == 2) ppmc(gamma, win[0], win[1], win[2], win[3], win[4], bn0, lo, hi);  // O10
  else if (RC == 3) plmp(win[0], win[1], win[2], lo, hi);
  else ppmp(win[0], win[1], win[2], win[3], win[4], lo, hi);
}

// x sweep: one WARP per 31 consecutive faces of an x pencil.  Lane l reconstructs cell c0 + l
// (its stencil comes straight from global memory / L1: neighbouring lanes read the same lines);
// the upper-face state W_{L,i+1/2} is handed to lane l+1 by warp shuffle, lanes 1..31 solve the
// Riemann problem on their lower face.  No shared memory, no block barrier; consecutive warps
// overlap by one cell (1/31 of the reconstructions are done twice).
__device__ __forceinline__ double shfl_up1(double v) { return __shfl_up_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ double shfl_dn1(double v) { return __shfl_down_sync(0xffffffffu, v, 1); }

// B + c (hi - lo) with one rounding per operation, identical wherever it is inlined
__device__ __forceinline__ double fma_diff(double B, double c, double hi, double lo) {
  return __fma_rn(c, __dadd_rn(hi, -lo), B);
}

template <int RC>
__global__ void __launch_bounds__(128, RC == 2 ? MHD_MINB_FX_PPM : MHD_MINB_FX) k_flux_x(State8 Uh, Flux21 F, Geo g, Box fb, int nwx) {
  constexpr int R = recon_radius(RC);
  const int lane = threadIdx.x & 31;
  const long long wid = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const int ly = fb.hi[1] - fb.lo[1] + 1, lz = fb.hi[2] - fb.lo[2] + 1;
  if (wid >= (long long)nwx * ly * lz) return;  // whole warps only
  const int wx = (int)(wid % nwx);
  const long long row_id = wid / nwx;
  const int j = fb.lo[1] + (int)(row_id % ly), k = fb.lo[2] + (int)(row_id / ly);
  const int c = fb.lo[0] - 1 + wx * 31 + lane;  // cell of this lane
  const bool active = (c <= fb.hi[0]);          // cells lo-1 .. hi are reconstructed
  const long long idx = cell_index(g, c, j, k);
  W7 lo, hi;
  if (active) {
    W7 win[2 * R + 1];
    double bnc[2 * R + 1];
#pragma unroll
    for (int s = 0; s < 2 * R + 1; s++) {
      Prim p = load_prim_half(Uh, g, idx + (s - R));
      win[s] = to_W<0>(p, bnc[s]);
    }
    reconstruct<RC>(g.gamma, win, bnc[R], lo, hi);
  } else {
    hi.rho = hi.u = hi.v = hi.w = hi.P = hi.by = hi.bz = 0.0;
    lo = hi;
  }
  W7 WL;
  WL.rho = shfl_up1(hi.rho); WL.u = shfl_up1(hi.u); WL.v = shfl_up1(hi.v); WL.w = shfl_up1(hi.w);
  WL.P = shfl_up1(hi.P); WL.by = shfl_up1(hi.by); WL.bz = shfl_up1(hi.bz);
  if (active && lane >= 1) {
    F7 f = hlld(g.gamma, g.gm1inv, WL, lo, __ldg(Uh.f[F_BX] + idx));
    store_flux<0>(F, idx, f);
  }
}

#define MHD_WSM_BYTES (5 * 8 * 128 * 8)
// the PLM y march is unrolled by two: the carried cell, difference and face state (24 doubles) then change
// names instead of registers (45 moves less per iteration; 0.715 -> 0.696 ms at 256^3); the z march with the
// update loses with it (0.88 -> 0.92 ms)
#ifndef MHD_MARCH_UNROLL
#define MHD_MARCH_UNROLL 2
#endif
#define MHD_PRAGMA_(x) _Pragma(#x)
#define MHD_UNROLL(n) MHD_PRAGMA_(unroll n)
// y / z sweep: a thread owns one x position (warps run along x, so every load and store is
// coalesced) and marches along the sweep axis over a chunk of J faces with a rolling window
// of 2R+1 primitive states in registers; each cell's primitives are formed once per chunk.
//
// UPDATE (z sweep only, the last of the three): the thread holds the z fluxes on both faces of cell
// f-1, and the x and y fluxes are already in memory, so it applies Eq. 29 to the hydro variables of
// that cell on the spot (U^n -> U^{n+1} in place; nothing else reads U^n's hydro fields any more).
// The four momentum / energy z fluxes then never go to memory (the mass and magnetic fluxes still
// do, for the CT kernel), and the full update that follows only has the face field left to do.
// A chunk then also solves face f1+1 (its last cell needs it; 1/J more Riemann solves).
template <int A, int RC, bool UPDATE>
__global__ void __launch_bounds__(128, recon_radius(RC) == 2 ? (UPDATE ? MHD_MINB_FMZ_PPM : MHD_MINB_FM_PPM) : (UPDATE ? MHD_MINB_FMZ : MHD_MINB_FM)) k_flux_march(State8 Uh, Flux21 F, Geo g, Box fb, int J,
                                                                  State8 U, const Scalars *sc) {
  static_assert(!UPDATE || A == 2, "the fused hydro update rides on the z sweep");
  constexpr int R = recon_radius(RC);
  constexpr int O = (A == 1) ? 2 : 1;  // the other transverse axis
  const int lx = fb.hi[0] - fb.lo[0] + 1, lo_ = fb.hi[O] - fb.lo[O] + 1;
  long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (long long)lx * lo_) return;
  const int i = fb.lo[0] + (int)(t % lx), o = fb.lo[O] + (int)(t / lx);
  const int f0 = fb.lo[A] + blockIdx.y * J;
  const int f1 = min(f0 + J - 1, fb.hi[A]);
  const int fend = (UPDATE && f1 < fb.hi[A]) ? f1 + 1 : f1;
  const long long sA = g.s[A];
  long long idx = (A == 1) ? cell_index(g, i, f0, o) : cell_index(g, i, o, f0);  // cell f0
  const bool upd_col = UPDATE && i >= 0 && i < g.n[0] && o >= 0 && o < g.n[O];  // an active column
  double dtd[3] = {0.0, 0.0, 0.0};
  if (UPDATE) {
    const double dt = sc->dt;
#pragma unroll
    for (int a = 0; a < 3; a++) dtd[a] = dt * g.id[a];
  }
  W7 win[2 * R + 1];
  double bnc[2 * R + 1];
  // 5-cell (PPM) sweeps: the window lives in this thread's column of shared memory (ring of 5 slots)
  // between iterations, so that its 40 doubles do not sit in registers across the projections
  // (dynamic shared memory, MHD_WSM_BYTES per block: with the update operands of the z sweep the
  // total exceeds the 48 KB static limit).
  // 3-cell (PLM) sweeps carry cell f and its lower one-sided difference dL = W_f - W_{f-1} (Eq. 23);
  // dR = W_{f+1} - W_f (Eq. 24) becomes the next cell's dL.
  constexpr bool WSM = (R == 2);
  constexpr bool PLM = (R == 1);
  extern __shared__ double wsm_[];
  auto wput = [&](int slot, const W7 &W, double bn) {
    double *q = wsm_ + slot * 8 * 128 + threadIdx.x;
    q[0] = W.rho; q[128] = W.u; q[256] = W.v; q[384] = W.w; q[512] = W.P; q[640] = W.by; q[768] = W.bz; q[896] = bn;
  };
  auto wget = [&](int slot, W7 &W, double &bn) {
    const double *q = wsm_ + slot * 8 * 128 + threadIdx.x;
    W.rho = q[0]; W.u = q[128]; W.v = q[256]; W.w = q[384]; W.P = q[512]; W.by = q[640]; W.bz = q[768]; bn = q[896];
  };
  W7 W0c, dLc;
  double bn0c = 0.0;
  [[maybe_unused]] double bface = 0.0, bface_next = 0.0;   // normal field on faces f, f+1 (PLM: from the prefetched cells)
  if constexpr (PLM) {
    double bnm;
    const W7 Wm = to_W<A>(load_prim_half(Uh, g, idx - 2 * sA), bnm);
    W0c = to_W<A>(load_prim_half(Uh, g, idx - sA), bn0c);
    dLc = w7_diff(W0c, Wm);
  } else {
    // window centred on cell f0-2 (slot 0 is never used): the loop below first shifts it
#pragma unroll
    for (int s = 1; s < 2 * R + 1; s++) {
      Prim p = load_prim_half(Uh, g, idx + (long long)(s - R - 2) * sA);
      win[s] = to_W<A>(p, bnc[s]);
      if (WSM) wput(s, win[s], bnc[s]);   // ring position of window slot s at "time" 0
    }
    if constexpr (R > 0) { win[0] = win[1]; bnc[0] = bnc[1]; }
    if (WSM) wput(0, win[0], bnc[0]);
  }
  int ring = 0;  // ring slot that holds window slot 0
  W7 WL, lo, hi;
  WL.rho = WL.P = 1.0; WL.u = WL.v = WL.w = WL.by = WL.bz = 0.0;  // (replaced before its first use)
  F7 fprev;
  fprev.m = fprev.mn = fprev.mt1 = fprev.mt2 = fprev.e = fprev.by = fprev.bz = 0.0;
  // staging column of this thread: slots 0..4 = U (rho, mx, my, mz, E) of the cell to update,
  // 5 + 10 a + 2 q + {0, 1} = flux component q of sweep a (x, y) on its lower / upper face
  __shared__ double stage[UPDATE ? 25 : 1][UPDATE ? 128 : 1];
  const int tid = threadIdx.x;
  const int last_cell = min(f1, g.n[A] - 1);
  idx -= sA;
  // The cell that enters the window in iteration f (cell f + R) is requested one iteration earlier
  // into this thread's column of `pre` (double-buffered): rho, v, P and the six faces around it.
  // cp.async groups complete in order and every iteration commits exactly two (the prefetch, then
  // the update operands -- either may be empty), so "all but the last group" is always the right wait.
  // Used by the 3-cell (PLM) sweeps and, since the 5-cell window moved to shared memory, by the PPM ones
  // (PPMC 256^3: y 1.57 -> 1.51 ms, z 2.00 -> 1.84 ms).
#ifndef MHD_PPM_PREF
#define MHD_PPM_PREF 1
#endif
  constexpr bool PREF = (R == 1) || (R == 2 && MHD_PPM_PREF);
  __shared__ double pre[PREF ? 2 : 1][PREF ? 11 : 1][PREF ? 128 : 1];
  auto prefetch = [&](int buf, long long c) {
    cp_async8(&pre[buf][0][tid], Uh.f[F_RHO] + c); cp_async8(&pre[buf][1][tid], Uh.f[F_MX] + c);
    cp_async8(&pre[buf][2][tid], Uh.f[F_MY] + c); cp_async8(&pre[buf][3][tid], Uh.f[F_MZ] + c);
    cp_async8(&pre[buf][4][tid], Uh.f[F_E] + c);
#pragma unroll
    for (int b = 0; b < 3; b++) {
      cp_async8(&pre[buf][5 + 2 * b][tid], Uh.f[F_BX + b] + c);
      cp_async8(&pre[buf][6 + 2 * b][tid], Uh.f[F_BX + b] + c + g.s[b]);
    }
  };
  if (PREF) prefetch((f0 - 1) & 1, idx + (long long)R * sA);
  cp_async_commit();
  cp_async_commit();  // (empty: keeps the two-groups-per-iteration count from the start)
  // One reconstruct() call site per kernel: iteration f0-1 only produces W_L of face f0; every
  // cell is then reconstructed by the same instruction sequence, so mirror-image cells give
  // mirror-image states bit for bit.
  MHD_UNROLL((PLM && !UPDATE) ? MHD_MARCH_UNROLL : 1)
  for (int f = f0 - 1; f <= fend; f++, idx += sA) {
    if constexpr (PLM) {
      cp_async_wait_but_last();  // the prefetch of cell f+1 (the newer group is the update's)
      const int b = f & 1;
      Prim p;
      p.rho = pre[b][0][tid]; p.ir = 0.0;
      p.v[0] = pre[b][1][tid]; p.v[1] = pre[b][2][tid]; p.v[2] = pre[b][3][tid];
      p.P = pre[b][4][tid];
      p.B[0] = 0.5 * (pre[b][5][tid] + pre[b][6][tid]);
      p.B[1] = 0.5 * (pre[b][7][tid] + pre[b][8][tid]);
      p.B[2] = 0.5 * (pre[b][9][tid] + pre[b][10][tid]);
      bface = bface_next;                        // face f: the lower A-face of cell f, seen one iteration ago
      bface_next = pre[b][5 + 2 * A][tid];       // lower A-face of the entering cell f+1 = face f+1
      if (f < fend) prefetch(b ^ 1, idx + (long long)(R + 1) * sA);
      cp_async_commit();
      double bnp;
      const W7 Wp = to_W<A>(p, bnp);
      const W7 dR = w7_diff(Wp, W0c);
      if (RC == 1) plmc_d(g.gamma, W0c, dLc, dR, bn0c, lo, hi);   // Eq. 23-28
      else plmp_d(W0c, dLc, dR, lo, hi);
      dLc = dR; W0c = Wp; bn0c = bnp;
    } else {
      if constexpr (PREF) {
        cp_async_wait_but_last();  // the prefetch of cell f+R (the newer group is the update's)
        const int b = f & 1;
        Prim p;
        p.rho = pre[b][0][tid]; p.ir = 0.0;
        p.v[0] = pre[b][1][tid]; p.v[1] = pre[b][2][tid]; p.v[2] = pre[b][3][tid];
        p.P = pre[b][4][tid];
        p.B[0] = 0.5 * (pre[b][5][tid] + pre[b][6][tid]);
        p.B[1] = 0.5 * (pre[b][7][tid] + pre[b][8][tid]);
        p.B[2] = 0.5 * (pre[b][9][tid] + pre[b][10][tid]);
        if (f < fend) prefetch(b ^ 1, idx + (long long)(R + 1) * sA);
        cp_async_commit();
        win[2 * R] = to_W<A>(p, bnc[2 * R]);
      } else {
        win[2 * R] = to_W<A>(load_prim_half(Uh, g, idx + (long long)R * sA), bnc[2 * R]);
        cp_async_commit();
      }
      if (WSM) {  // the oldest ring slot takes the new cell; the window is re-read slot by slot
        wput(ring, win[2 * R], bnc[2 * R]);
        ring = (ring + 1 == 5) ? 0 : ring + 1;
#pragma unroll
        for (int s = 0; s < 2 * R; s++) {
          int slot = ring + s; slot = (slot >= 5) ? slot - 5 : slot;
          wget(slot, win[s], bnc[s]);
        }
      }
      reconstruct<RC>(g.gamma, win, bnc[R], lo, hi);
    }
    if (f >= f0) {
      F7 fl = hlld(g.gamma, g.gm1inv, WL, lo, PLM ? bface : __ldg(Uh.f[F_BX + A] + idx));
      if (!UPDATE) {
        store_flux<A>(F, idx, fl);
      } else {
        if (f <= f1) { F.f[A][0][idx] = fl.m; F.f[A][5][idx] = fl.by; F.f[A][6][idx] = fl.bz; }
        if (upd_col && f > f0 && f - 1 <= last_cell) {  // cell f-1: Eq. 29, x then y then z (R2)
          const long long c = idx - sA;
          cp_async_wait_but_last();  // its operands (the newer group is the next cell's prefetch)
          double rho = stage[0][tid], En = stage[4][tid];
          double m[3] = {stage[1][tid], stage[2][tid], stage[3][tid]};
#pragma unroll
          for (int a = 0; a < 2; a++) {
            const double *q = &stage[5 + 10 * a][tid];
            rho -= dtd[a] * (q[1 * 128] - q[0 * 128]);
            m[a] -= dtd[a] * (q[3 * 128] - q[2 * 128]);
            m[(a + 1) % 3] -= dtd[a] * (q[5 * 128] - q[4 * 128]);
            m[(a + 2) % 3] -= dtd[a] * (q[7 * 128] - q[6 * 128]);
            En -= dtd[a] * (q[9 * 128] - q[8 * 128]);
          }
          rho -= dtd[2] * (fl.m - fprev.m);
          m[2] -= dtd[2] * (fl.mn - fprev.mn);
          m[0] -= dtd[2] * (fl.mt1 - fprev.mt1);
          m[1] -= dtd[2] * (fl.mt2 - fprev.mt2);
          En -= dtd[2] * (fl.e - fprev.e);
          U.f[F_RHO][c] = rho; U.f[F_MX][c] = m[0]; U.f[F_MY][c] = m[1]; U.f[F_MZ][c] = m[2];
          U.f[F_E][c] = En;
        }
        fprev = fl;
      }
    }
    if (UPDATE && upd_col && f >= f0 && f <= last_cell) {  // fetch what cell f's update will need
      cp_async8(&stage[0][tid], U.f[F_RHO] + idx); cp_async8(&stage[1][tid], U.f[F_MX] + idx);
      cp_async8(&stage[2][tid], U.f[F_MY] + idx); cp_async8(&stage[3][tid], U.f[F_MZ] + idx);
      cp_async8(&stage[4][tid], U.f[F_E] + idx);
#pragma unroll
      for (int a = 0; a < 2; a++)
#pragma unroll
        for (int q = 0; q < 5; q++) {
          cp_async8(&stage[5 + 10 * a + 2 * q][tid], F.f[a][q] + idx);
          cp_async8(&stage[5 + 10 * a + 2 * q + 1][tid], F.f[a][q] + idx + g.s[a]);
        }
    }
    cp_async_commit();  // always: one update group per iteration, possibly empty
    WL = hi;
  }
}

}  // namespace mhd
