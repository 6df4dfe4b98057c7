// mhd_device.cuh -- per-cell / per-face device arithmetic of the VL+CT step (sm_100a, fp64).
//
// Everything here is register-resident scalar code, written from the paper
// (/root/reference/PAPER.md, cited as PAPER.md:<line>) and the readings O0..O12 listed in
// DESIGN.md.  No fast-math; FMA contraction is left to nvcc (default --fmad=true).
// Solver-local 1-D state for a sweep along axis a (O0): W = (rho, u, v, w, P, By, Bz) with
// (u,v,w) = (v_a, v_{a+1}, v_{a+2}), (By,Bz) = (B_{a+1}, B_{a+2}) (indices mod 3); the normal
// field Bn is carried separately.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

#include "mhd_math.cuh"

namespace mhd {

struct W7 {
  double rho, u, v, w, P, by, bz;
};

struct F7 {  // mass, mom_n, mom_t1, mom_t2, energy, By-flux, Bz-flux
  double m, mn, mt1, mt2, e, by, bz;
};

// Eq. 12: c_f^2 along the direction whose field component is bn; irho = 1/rho.
// The discriminant is clamped at 0 against round-off (reading R3).
__device__ __forceinline__ double fast_speed_sq(double gamma, double irho, double P, double bn,
                                                double bt1, double bt2) {
  double gp = gamma * P;
  double b2 = bn * bn + bt1 * bt1 + bt2 * bt2;
  double s = gp + b2;
  double disc = s * s - 4.0 * gp * bn * bn;
  disc = disc < 0.0 ? 0.0 : disc;
  return (s + sqrt_(disc)) * (0.5 * irho);
}

// ---------------------------------------------------------------------------------------
// HLLD (Miyoshi & Kusano 2005, cited PAPER.md:149; reading O4, wave speeds G15).
//
// The flux in every region of the fan is evaluated as the physical flux function of that region's
// state with the fan's total pressure p_T* in place of p_T:
//     F*_a = F_a + S_a (U*_a - U_a)            == Eq. 8 applied to (rho*, S_M, v*, w*, B*, e*; p_T*)
//     F**_a = F*_a + S*_a (U**_a - U*_a)       == Eq. 8 applied to (rho*, S_M, v**, w**, B**, e**; p_T*)
// These are identities, not approximations: U*_a is DEFINED by the jump conditions across S_a
// (M&K Eq. 43-48) and U** by those across S*_a (Eq. 59-63).  The one exception is M&K's degenerate
// case (|D| < eps p_T*: the tangential components are left unchanged, which is not a solution of the
// jump conditions for B_t): there F_a + S_a (U*_a - U_a) has the extra terms B_t,a (u_a - S_M) in
// the two induction components, which are added explicitly.  One flux evaluation instead of three,
// only the side that bounds the face gets its energy, the other side's star state is formed only
// where the double-star state is needed, and no reciprocal of rho_L, rho_R is taken at all
// (the larger fast speed is found by cross-multiplication).  ~200 fp64 instructions per solve.
// ---------------------------------------------------------------------------------------
#ifndef MHD_DBL_ALWAYS
#define MHD_DBL_ALWAYS 0   // 1: form the double-star state on every face and select (one larger basic block)
#endif
__device__ __forceinline__ int hi32(double x) { return __double2hiint(x); }
__device__ __forceinline__ double xor_sign(double x, int signbit) {
  return __hiloint2double(__double2hiint(x) ^ signbit, __double2loint(x));
}

// x, or +tiny where x is negative, zero or denormal (round-off guard R3 of the discriminant of
// Eq. 12: it is >= 0 analytically; 2^-1000 keeps the seed instruction of the root off 0)
__device__ __forceinline__ double floor_tiny(double x) { return (hi32(x) < 0x00100000) ? 0x1p-1000 : x; }

// minimum / maximum of two numbers by one compare and one select.  fmin() / fmax() also order NaNs
// (a predicate pair, two moves, a quiet-bit LOP3 and two selects per call on sm_100a: 7 instructions);
// their operands here are magnitudes of finite numbers, where both give the same bits.
__device__ __forceinline__ double min_(double a, double b) { return (a < b) ? a : b; }
__device__ __forceinline__ double max_(double a, double b) { return (a > b) ? a : b; }
// the operand of smaller / larger magnitude, sign and all: |x| is free as an operand modifier of the
// compare but costs an instruction as a value, and every use below ends in copysign() or fabs()
__device__ __forceinline__ double amin_(double a, double b) { return (fabs(a) < fabs(b)) ? a : b; }
__device__ __forceinline__ double amax_(double a, double b) { return (fabs(a) > fabs(b)) ? a : b; }

struct HlldSide {
  double rho, u, v, w, P, by, bz;
  double hb2, pT;   // B^2 / 2, total pressure
  double X;         // gamma P + B^2 + sqrt(disc) = 2 rho c_f^2   (Eq. 12)
};

__device__ __forceinline__ void hlld_side_init(HlldSide &s, const W7 &W, double gamma, double bx2, double bx2x4) {
  s.rho = W.rho; s.u = W.u; s.v = W.v; s.w = W.w; s.P = W.P; s.by = W.by; s.bz = W.bz;
  double b2 = (W.by * W.by + W.bz * W.bz) + bx2;
  s.hb2 = 0.5 * b2;
  s.pT = W.P + s.hb2;
  double gp = gamma * W.P;
  double sm = gp + b2;
  double disc = floor_tiny(sm * sm - gp * bx2x4);
  s.X = sm + sqrt_nz(disc);
}

// Eq. 8 without the zero row, for the state (rho, u, v, w, by, bz, e) under the
// total pressure pT; vb = u bx + v by + w bz
__device__ __forceinline__ F7 flux_of(double rho, double u, double v, double w, double by, double bz, double e,
                                      double pT, double vb, double bx, double bx2) {
  F7 F;
  double m = rho * u;
  F.m = m;
  F.mn = m * u + (pT - bx2);
  F.mt1 = m * v - bx * by;
  F.mt2 = m * w - bx * bz;
  F.e = u * (e + pT) - bx * vb;
  F.by = by * u - bx * v;
  F.bz = bz * u - bx * w;
  return F;
}

__device__ __forceinline__ double total_energy(double gm1inv, double rho, double u, double v, double w, double P,
                                               double hb2) {
  return (0.5 * rho) * (u * u + v * v + w * w) + (P * gm1inv + hb2);
}

// single-star state of one side (M&K Eq. 43-47): S = outer speed, sdu = rho (S - u), dua = S_M - u.
// With g = (S_M - u) / D:  v* = v - B_y B_x g,  B_y* = B_y + B_y rho (S - u) g   (the same as
// M&K's (rho (S-u)^2 - B_x^2) / D, written as 1 + ...), so the degenerate case is g = 0.
struct Star {
  double rhos, vs, ws, bys, bzs, iSSm;
  bool degen;
};

__device__ __forceinline__ Star hlld_star(double S, double SM, double sdu, double dua, double v, double w,
                                          double by, double bz, double pTs, double bx, double bx2) {
  Star q;
  const double SSm = S - SM;
  const double D = sdu * SSm - bx2;
  q.degen = fabs(D) < 1e-8 * pTs;                // degenerate 0/0: no jump in the tangential fields
  const double t = q.degen ? 1.0 : D;
  const double inv = rcp(t * SSm);               // one reciprocal for 1/D and 1/(S - S_M)
  q.iSSm = inv * t;
  const double g = q.degen ? 0.0 : (inv * SSm) * dua;
  const double fv = bx * g, fb = sdu * g;
  q.vs = v - by * fv;
  q.ws = w - bz * fv;
  q.bys = by + by * fb;
  q.bzs = bz + bz * fb;
  q.rhos = sdu * q.iSSm;
  return q;
}

__device__ __forceinline__ F7 hlld(double gamma, double gm1inv, const W7 &WL, const W7 &WR, double bx) {
  const double bx2 = bx * bx, bx2x4 = 4.0 * bx2;
  HlldSide L, R;
  hlld_side_init(L, WL, gamma, bx2, bx2x4);
  hlld_side_init(R, WR, gamma, bx2, bx2x4);
  // G15: S_L = min(u_L, u_R) - max(c_fL, c_fR), S_R = max(u_L, u_R) + max(c_fL, c_fR), with
  // c_f^2 = X / (2 rho): the larger one by cross-multiplication, its root as X rsqrt(2 rho X)
  const bool lbig = L.X * R.rho > R.X * L.rho;
  const double Xw = lbig ? L.X : R.X, rw = lbig ? L.rho : R.rho;
  const double cfmax = Xw * rsqrt_((2.0 * rw) * Xw);
  const bool ul = L.u < R.u;
  const double SL = (ul ? L.u : R.u) - cfmax;
  const double SR = (ul ? R.u : L.u) + cfmax;

  // the state whose flux is the answer, and the total pressure it is under
  double frho, fu, fv, fw, fby, fbz, fe, fpT, fvb, cb, cby, cbz;
  const bool super = (SL > 0.0 || SR < 0.0);
  {
    // middle wave (M&K Eq. 38).  rho_R (S_R - u_R) > 0 > rho_L (S_L - u_L) always, so this block is
    // well defined on supersonic faces too (its result is replaced below): no branch ahead of it
    const double sduL = (SL - L.u) * L.rho;
    const double sduR = (SR - R.u) * R.rho;
    const double SM = (sduR * R.u - sduL * L.u - R.pT + L.pT) * rcp(sduR - sduL);
    // side a bounds the face: left if S_M >= 0 (S*_L >= 0 implies S_M >= 0); b is the other one
    const bool left = (SM >= 0.0);
    const double a_rho = left ? L.rho : R.rho, a_u = left ? L.u : R.u, a_v = left ? L.v : R.v;
    const double a_w = left ? L.w : R.w, a_P = left ? L.P : R.P, a_by = left ? L.by : R.by;
    const double a_bz = left ? L.bz : R.bz, a_hb2 = left ? L.hb2 : R.hb2, a_pT = left ? L.pT : R.pT;
    const double a_S = left ? SL : SR, a_sdu = left ? sduL : sduR;
    const double dua = SM - a_u;
    // total pressure of the fan from the jump across S_a (M&K Eq. 23; Eq. 41 is the same quantity)
    const double pTs = a_pT + a_sdu * dua;
    const Star A = hlld_star(a_S, SM, a_sdu, dua, a_v, a_w, a_by, a_bz, pTs, bx, bx2);
    const double a_e = total_energy(gm1inv, a_rho, a_u, a_v, a_w, a_P, a_hb2);
    const double vb = a_u * bx + a_v * a_by + a_w * a_bz;
    const double vbs = SM * bx + A.vs * A.bys + A.ws * A.bzs;
    const double es = ((a_S - a_u) * a_e - a_pT * a_u + pTs * SM + bx * (vb - vbs)) * A.iSSm;  // M&K Eq. 48
    cb = A.degen ? -dua : 0.0;
    cby = a_by; cbz = a_bz;
    frho = A.rhos; fu = SM; fpT = pTs;
    fv = A.vs; fw = A.ws; fby = A.bys; fbz = A.bzs; fe = es; fvb = vbs;
    // double-star region: |S_M| < |B_x| / sqrt(rho*_a)   (S*_L < 0 <= S_M, or S_M < 0 < S*_R)
    const bool dbl = SM * SM * A.rhos < bx2;
    if (MHD_DBL_ALWAYS || dbl) {
      const double b_u = left ? R.u : L.u, b_v = left ? R.v : L.v, b_w = left ? R.w : L.w;
      const double b_by = left ? R.by : L.by, b_bz = left ? R.bz : L.bz;
      const double b_S = left ? SR : SL, b_sdu = left ? sduR : sduL;
      const Star B = hlld_star(b_S, SM, b_sdu, SM - b_u, b_v, b_w, b_by, b_bz, pTs, bx, bx2);
      // M&K Eq. 59-63, written for (a, b) with s' = sgn(B_x) for a = L and -sgn(B_x) for a = R
      const double ra = sqrt_nz(A.rhos), rb = sqrt_nz(B.rhos);
      const double sg = (bx > 0.0) ? 1.0 : ((bx < 0.0) ? -1.0 : 0.0);
      const double sp = left ? sg : -sg;
      const double inv = rcp(ra + rb);
      const double rr = (ra * rb) * sp;
      const double vss = (ra * A.vs + rb * B.vs + (B.bys - A.bys) * sp) * inv;
      const double wss = (ra * A.ws + rb * B.ws + (B.bzs - A.bzs) * sp) * inv;
      const double byss = (ra * B.bys + rb * A.bys + rr * (B.vs - A.vs)) * inv;
      const double bzss = (ra * B.bzs + rb * A.bzs + rr * (B.ws - A.ws)) * inv;
      const double vbss = SM * bx + vss * byss + wss * bzss;
      const double ess = es - (ra * sp) * (vbs - vbss);
      if (dbl) { fv = vss; fw = wss; fby = byss; fbz = bzss; fvb = vbss; fe = ess; }
    }
  }
  if (super) {   // S_L > 0: F_L; S_R < 0: F_R (rare; after the main block so that it stays in one piece)
    const bool l = SL > 0.0;
    frho = l ? L.rho : R.rho; fu = l ? L.u : R.u; fv = l ? L.v : R.v; fw = l ? L.w : R.w;
    fby = l ? L.by : R.by; fbz = l ? L.bz : R.bz; fpT = l ? L.pT : R.pT;
    fe = total_energy(gm1inv, frho, fu, fv, fw, l ? L.P : R.P, l ? L.hb2 : R.hb2);
    fvb = fu * bx + fv * fby + fw * fbz;
    cb = 0.0;
  }
  F7 F = flux_of(frho, fu, fv, fw, fby, fbz, fe, fpT, fvb, bx, bx2);
  F.by += cby * cb;   // degenerate star state of side a only (see the header); cb = 0 otherwise
  F.bz += cbz * cb;
  // reading R6: a contact slower than 1e-13 of the fast speed is at rest -- the mass flux, whose
  // sign upwinds the CT terms (Eq. 16, G6), is then exactly zero ("otherwise" branch: average)
  if (fabs(F.m) <= 1e-13 * (L.rho + R.rho) * cfmax) F.m = 0.0;
  return F;
}

// ---------------------------------------------------------------------------------------
// Eigen-system of the primitive-variable equations (Stone et al. 2008 App. A, cited
// PAPER.md:249; reading O9, degenerate normalisation G16), held as the dozen scalars the
// 7x7 matrices are built from.  Wave order u-cf, u-ca, u-cs, u, u+cs, u+ca, u+cf.
// The left/right projections below are the matrix-vector products L.x and R.a written out
// with the structural zeros removed and the transverse components rotated into the
// (parallel, perpendicular)-to-B_perp frame: xp = by*X_y + bz*X_z, xq = by*X_z - bz*X_y.
// ---------------------------------------------------------------------------------------
struct Eig {
  double rho, irho, a2, ia2, N;
  double betay, betaz, alf, als;
  double Cff, Css, Qf, Qs, Af, As;
  double Ssr;   // S * sqrt(rho)
  double Sisr;  // S / sqrt(rho)
  // rows of L with their common factors folded in (N = 1/(2 a^2), 1/rho, 1/2): each projection is 24
  // fp64 instructions instead of 32, and PLMC makes three of them per cell, PPMC five
  double NCff, NCss, NQf, NQs, Naf, Nas, NAf, NAs, hSisr;
};

struct C7 {  // characteristic amplitudes
  double c0, c1, c2, c3, c4, c5, c6;
};

__device__ __forceinline__ void eig_setup(Eig &e, double gamma, const W7 &W, double bx) {
  double rho = W.rho;
  double sr, isr;
  sqrt_rsqrt(rho, sr, isr);
  double irho = isr * isr;
  double gp = gamma * W.P;
  double a2 = gp * irho;
  double a, ia;
  sqrt_rsqrt(a2, a, ia);
  double ia2 = ia * ia;
  double by = W.by, bz = W.bz;
  double bx2 = bx * bx;
  double s = gp + (bx2 + (by * by + bz * bz));
  double disc = floor_tiny(s * s - 4.0 * gp * bx2);  // reading R3
  double cf2 = (s + sqrt_nz(disc)) * (0.5 * irho);   // Eq. 12
  // c_s = a c_a / c_f: no cancellation (O9), and no square of B_n, which can be ~1e-160 in the
  // numerical foot of a switch-on shock (Ryu & Jones 4d, reading R12)
  double icf = rsqrt_(cf2);
  double cf = cf2 * icf;
  double cs = (a * fabs(bx)) * (isr * icf);
  double cs2 = cs * cs;
  // direction of B_perp; (1, 0) when it vanishes (G16).  The same foot carries transverse fields
  // down to 1e-180: rescale before squaring so that the seed instruction never sees a denormal
  // (exponent test on the integer pipe)
  int mag = max(hi32(by) & 0x7fffffff, hi32(bz) & 0x7fffffff);
  if (mag < 0x20b00000) {  // max(|by|, |bz|) < 2^-500
    by *= 0x1p600; bz *= 0x1p600;
    if (by == 0.0 && bz == 0.0) by = 1.0;
  }
  double ib = rsqrt_(by * by + bz * bz);
  e.betay = by * ib; e.betaz = bz * ib;
  double dfs = cf2 - cs2;
  if (hi32(dfs) < 0x00100000) { e.alf = 1.0; e.als = 0.0; }  // c_f = c_s (G16)
  else {
    double idfs = rcp(dfs);
    double af2 = (a2 - cs2) * idfs;
    double as2 = (cf2 - a2) * idfs;
    // clip to [0, 1] on the exponent bits: negative -> 0, >= 1 -> 1
    af2 = hi32(af2) < 0 ? 0.0 : (hi32(af2) >= 0x3ff00000 ? 1.0 : af2);
    as2 = hi32(as2) < 0 ? 0.0 : (hi32(as2) >= 0x3ff00000 ? 1.0 : as2);
    e.alf = sqrt_(af2); e.als = sqrt_(as2);
  }
  // S = sgn(B_n), +1 at 0 (O9): multiplication by S is a flip of the sign bit
  const int sflip = (bx >= 0.0) ? 0 : (int)0x80000000;
  e.rho = rho; e.irho = irho; e.a2 = a2; e.ia2 = ia2; e.N = 0.5 * ia2;
  e.Cff = cf * e.alf; e.Css = cs * e.als;
  e.Qf = xor_sign(e.Cff, sflip); e.Qs = xor_sign(e.Css, sflip);
  e.Af = a * e.alf * sr; e.As = a * e.als * sr;
  e.Ssr = xor_sign(sr, sflip); e.Sisr = xor_sign(isr, sflip);
  const double Nir = e.N * irho;
  e.NCff = e.N * e.Cff; e.NCss = e.N * e.Css;
  e.NQf = xor_sign(e.NCff, sflip); e.NQs = xor_sign(e.NCss, sflip);
  e.Naf = Nir * e.alf; e.Nas = Nir * e.als; e.NAf = Nir * e.Af; e.NAs = Nir * e.As;
  e.hSisr = 0.5 * e.Sisr;
}

// a = L . x   (x in the component order of W7).  Written with explicit rounding intrinsics so
// that every inlined copy is the same instruction sequence: PPMC projects the five stencil
// states separately, and the limiter's tests (reading O10: "<= 0" includes equality) must see
// bit-identical amplitudes for bit-identical states (an exact plateau next to a jump).
__device__ __forceinline__ C7 eig_left(const Eig &e, const W7 &x) {
  double xp = __fma_rn(e.betay, x.v, __dmul_rn(e.betaz, x.w));
  double xq = __fma_rn(e.betay, x.w, -__dmul_rn(e.betaz, x.v));
  double bp = __fma_rn(e.betay, x.by, __dmul_rn(e.betaz, x.bz));
  double bq = __fma_rn(e.betay, x.bz, -__dmul_rn(e.betaz, x.by));
  double f1 = __fma_rn(e.NCff, x.u, -__dmul_rn(e.NQs, xp));   // N (C_ff u - Q_s x_p)
  double f2 = __fma_rn(e.Naf, x.P, __dmul_rn(e.NAs, bp));     // N (alpha_f P + A_s b_p) / rho
  double s1 = __fma_rn(e.NCss, x.u, __dmul_rn(e.NQf, xp));
  double s2 = __fma_rn(e.Nas, x.P, -__dmul_rn(e.NAf, bp));
  double hxq = __dmul_rn(0.5, xq);
  C7 c;
  c.c0 = __dadd_rn(f2, -f1);
  c.c6 = __dadd_rn(f2, f1);
  c.c2 = __dadd_rn(s2, -s1);
  c.c4 = __dadd_rn(s2, s1);
  c.c1 = __fma_rn(e.hSisr, bq, hxq);
  c.c5 = __fma_rn(e.hSisr, bq, -hxq);
  c.c3 = __fma_rn(-x.P, e.ia2, x.rho);
  return c;
}

// x = R . a   (explicit roundings for the same reason: the two faces of a cell whose limited
// amplitudes are bit-identical must get bit-identical states, so that a face between mirror-image
// cells at rest sees W_L == W_R and an exactly zero mass flux -- the "average" branch of Eq. 16)
__device__ __forceinline__ W7 eig_right(const Eig &e, const C7 &c) {
  double fs = __dadd_rn(c.c0, c.c6), fd = __dadd_rn(c.c6, -c.c0);
  double ss = __dadd_rn(c.c2, c.c4), sd = __dadd_rn(c.c4, -c.c2);
  double as_ = __dadd_rn(c.c1, c.c5), ad = __dadd_rn(c.c1, -c.c5);
  double comp = __fma_rn(e.alf, fs, __dmul_rn(e.als, ss));
  double tp = __fma_rn(e.Qf, sd, -__dmul_rn(e.Qs, fd));   // transverse velocity along B_perp
  double bp = __fma_rn(e.As, fs, -__dmul_rn(e.Af, ss));   // transverse field along B_perp
  double bq = __dmul_rn(e.Ssr, as_);                      // transverse field across B_perp
  W7 x;
  x.rho = __fma_rn(e.rho, comp, c.c3);
  x.u = __fma_rn(e.Cff, fd, __dmul_rn(e.Css, sd));
  x.v = __fma_rn(e.betay, tp, -__dmul_rn(e.betaz, ad));
  x.w = __fma_rn(e.betaz, tp, __dmul_rn(e.betay, ad));
  x.P = __dmul_rn(__dmul_rn(e.rho, e.a2), comp);
  x.by = __fma_rn(e.betay, bp, -__dmul_rn(e.betaz, bq));
  x.bz = __fma_rn(e.betaz, bp, __dmul_rn(e.betay, bq));
  return x;
}

// ---------------------------------------------------------------------------------------
// PLMC, Eq. 23-28 (reading O8).  Out: Wlo = W_{R,i-1/2}, Whi = W_{L,i+1/2}.
// ---------------------------------------------------------------------------------------
// Sign tests and selections of the limiters run on the integer pipe (the sign of a double is
// bit 63, its magnitude orders like the bit pattern); only the minima themselves are fp64 compares.
__device__ __forceinline__ double min_pos(double a, double b) { return a < b ? a : b; }  // no NaN handling needed

__device__ __forceinline__ double vl_slope(double dl, double dr) {  // Eq. 26 (G10)
  // dl dr > 0 <=> the product is a positive normal number (a product that underflows gives a slope
  // below 1e-300: zero for every purpose)
  double pr = dl * dr;
  return (hi32(pr) >= 0x00100000) ? 2.0 * pr * rcp(dl + dr) : 0.0;
}

__device__ __forceinline__ double plm_limit(double aL, double aR, double aC, double aVL) {  // Eq. 27
  // min(2|aL|, 2|aR|, |aC|, |aVL|) with the sign of aC where aL aR > 0, else 0.  If either of aL, aR
  // is zero the minimum is zero by itself, so only "opposite signs" needs a test: the xor of the
  // sign bits.  Where aL aR > 0, aC = (aL + aR)/2 has their sign: the sign transfer is a bit operation.
  double m = min_pos(2.0 * min_pos(fabs(aL), fabs(aR)), min_pos(fabs(aC), fabs(aVL)));
  return ((hi32(aL) ^ hi32(aR)) < 0) ? 0.0 : copysign(m, aC);
}

// from the one-sided differences dL = W_i - W_{i-1} (Eq. 23), dR = W_{i+1} - W_i (Eq. 24): a marching
// sweep carries dR over as the next cell's dL
__device__ __forceinline__ void plmc_d(double gamma, const W7 &W0, const W7 &dL, const W7 &dR, double bx0,
                                       W7 &Wlo, W7 &Whi) {
  Eig e;
  eig_setup(e, gamma, W0, bx0);
  W7 dV;
  dV.rho = vl_slope(dL.rho, dR.rho); dV.u = vl_slope(dL.u, dR.u); dV.v = vl_slope(dL.v, dR.v);
  dV.w = vl_slope(dL.w, dR.w); dV.P = vl_slope(dL.P, dR.P); dV.by = vl_slope(dL.by, dR.by);
  dV.bz = vl_slope(dL.bz, dR.bz);
  // L is linear and dC = (dL + dR)/2, so the centred amplitudes are the mean of the one-sided ones
  C7 aL = eig_left(e, dL), aR = eig_left(e, dR), aV = eig_left(e, dV);
  C7 am;
  am.c0 = plm_limit(aL.c0, aR.c0, 0.5 * (aL.c0 + aR.c0), aV.c0);
  am.c1 = plm_limit(aL.c1, aR.c1, 0.5 * (aL.c1 + aR.c1), aV.c1);
  am.c2 = plm_limit(aL.c2, aR.c2, 0.5 * (aL.c2 + aR.c2), aV.c2);
  am.c3 = plm_limit(aL.c3, aR.c3, 0.5 * (aL.c3 + aR.c3), aV.c3);
  am.c4 = plm_limit(aL.c4, aR.c4, 0.5 * (aL.c4 + aR.c4), aV.c4);
  am.c5 = plm_limit(aL.c5, aR.c5, 0.5 * (aL.c5 + aR.c5), aV.c5);
  am.c6 = plm_limit(aL.c6, aR.c6, 0.5 * (aL.c6 + aR.c6), aV.c6);
  W7 dW = eig_right(e, am);
#define MHD_O(f) Whi.f = W0.f + dW.f / 2.0; Wlo.f = W0.f - dW.f / 2.0;
  MHD_O(rho) MHD_O(u) MHD_O(v) MHD_O(w) MHD_O(P) MHD_O(by) MHD_O(bz)
#undef MHD_O
}

// PLMP (limiting in the primitive variables = Eq. 23-28 without the projections)
__device__ __forceinline__ void plmp_d(const W7 &W0, const W7 &dL, const W7 &dR, W7 &Wlo, W7 &Whi) {
#define MHD_P1(f)                                                                        \
  {                                                                                      \
    double dl = dL.f, dr = dR.f;                                                         \
    double dm = plm_limit(dl, dr, 0.5 * (dl + dr), vl_slope(dl, dr));                    \
    Whi.f = W0.f + 0.5 * dm; Wlo.f = W0.f - 0.5 * dm;                                    \
  }
  MHD_P1(rho) MHD_P1(u) MHD_P1(v) MHD_P1(w) MHD_P1(P) MHD_P1(by) MHD_P1(bz)
#undef MHD_P1
}

__device__ __forceinline__ W7 w7_diff(const W7 &a, const W7 &b) {
  W7 d;
  d.rho = a.rho - b.rho; d.u = a.u - b.u; d.v = a.v - b.v; d.w = a.w - b.w; d.P = a.P - b.P;
  d.by = a.by - b.by; d.bz = a.bz - b.bz;
  return d;
}

__device__ __forceinline__ void plmc(double gamma, const W7 &Wm, const W7 &W0, const W7 &Wp,
                                     double bx0, W7 &Wlo, W7 &Whi) {
  plmc_d(gamma, W0, w7_diff(W0, Wm), w7_diff(Wp, W0), bx0, Wlo, Whi);
}

__device__ __forceinline__ void plmp(const W7 &Wm, const W7 &W0, const W7 &Wp, W7 &Wlo, W7 &Whi) {
  plmp_d(W0, w7_diff(W0, Wm), w7_diff(Wp, W0), Wlo, Whi);
}

// ---------------------------------------------------------------------------------------
// PPMC (reading O10 / G17 of Felker & Stone 2018, cited PAPER.md:231, 431).
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ double sgn3(double x) { return (x > 0.0) ? 1.0 : ((x < 0.0) ? -1.0 : 0.0); }

// limited 4th-order value on the face between cells j and j+1; qa..qd = q_{j-1..j+2}
// "D_f and the cell curvatures share a sign" is tested with products (a fp64 multiply and a compare
// each, instead of three-way sign extraction), and sgn * min(C|D_a|, C|D_b|, |D_f|) is formed as
// copysign(min(C min(|D_a|, |D_b|), |D_f|), D_f): multiplication by C = 1.25 is monotone, so the
// value is bit for bit the oracle's.  The minima pick the operand of smaller magnitude with its sign
// (amin_), which copysign() replaces at the end.
#ifndef MHD_PPM_BRANCHY
#define MHD_PPM_BRANCHY 0
#endif
#if MHD_PPM_BRANCHY
__device__ __forceinline__ double ppm_face(double qa, double qb, double qc, double qd) {
  const double C = 1.25;
  double qf = (7.0 / 12.0) * (qb + qc) - (1.0 / 12.0) * (qa + qd);
  if ((qf - qb) * (qc - qf) < 0.0) {
    double Df = 3.0 * (qb - 2.0 * qf + qc);
    double Dj = qa - 2.0 * qb + qc;
    double Dj1 = qb - 2.0 * qc + qd;
    double Dlim = 0.0;
    if (Df * Dj > 0.0 && Df * Dj1 > 0.0)
      Dlim = copysign(amin_(C * amin_(Dj, Dj1), Df), Df);
    qf = 0.5 * (qb + qc) - Dlim * (1.0 / 6.0);
  }
  return qf;
}

__device__ __forceinline__ void ppm_scalar(double q0, double q1, double q2, double q3, double q4,
                                           double &qlo, double &qhi) {
  const double C = 1.25;
  double qm = ppm_face(q0, q1, q2, q3);
  double qp = ppm_face(q1, q2, q3, q4);
  double qi = q2;
  // reading R7: differences that are zero to round-off count as zero in the extremum test
  double tau = 1e-12 * fabs(amax_(q1, amax_(q2, q3)));
  double dm = qi - qm, dp = qp - qi, e3 = q3 - qi, e1 = qi - q1;
  dm = (fabs(dm) <= tau) ? 0.0 : dm;
  dp = (fabs(dp) <= tau) ? 0.0 : dp;
  e3 = (fabs(e3) <= tau) ? 0.0 : e3;
  e1 = (fabs(e1) <= tau) ? 0.0 : e1;
  if (dm * dp <= 0.0 || e3 * e1 <= 0.0) {
    double Df = 6.0 * (qm - 2.0 * qi + qp);
    double Dm1 = q0 - 2.0 * q1 + q2;
    double D0 = q1 - 2.0 * q2 + q3;
    double Dp1 = q2 - 2.0 * q3 + q4;
    double Dlim = 0.0, r = 0.0;
    if (Df * Dm1 > 0.0 && Df * D0 > 0.0 && Df * Dp1 > 0.0)
      Dlim = copysign(amin_(C * amin_(Dm1, amin_(D0, Dp1)), Df), Df);
    if (fabs(Df) > max_(tau, 1e-290)) r = Dlim * rcp(Df);  // (the floor keeps rcp off denormals)
    if (r <= 1.0 - 1e-12) { qm = qi - r * dm; qp = qi + r * dp; }
  } else {
    if (fabs(dm) >= 2.0 * fabs(dp)) qm = qi - 2.0 * dp;
    if (fabs(dp) >= 2.0 * fabs(dm)) qp = qi + 2.0 * dm;
  }
  qlo = qm; qhi = qp;
}

#else
// Branch-free: every candidate value is formed and the tests select among them.  The seven
// characteristic fields of a cell are then one basic block, whose independent dependency chains the
// instruction scheduler interleaves (with a branch per test each field was a chain of its own: 2.3-2.5
// warps waiting on a fixed-latency result per issued instruction, 0.3 on a branch, 0.4-0.6 on instruction
// fetch); the curvatures D shared by the two faces and by the extremum test are formed once.
// c ? a : b as one select the compiler cannot turn back into a branch around the evaluation of a
__device__ __forceinline__ double select_(bool c, double a, double b) {
  double r;
  asm("{\n.reg .pred p;\nsetp.ne.s32 p, %3, 0;\nselp.f64 %0, %1, %2, p;\n}" : "=d"(r) : "d"(a), "d"(b), "r"((int)c));
  return r;
}

// "D_f and the cell curvatures share a sign" on the sign bits (one LOP3 and one integer compare instead of a
// fp64 multiply and a fp64 compare per curvature).  Zeros need no test of their own: with a zero among them
// the limited curvature min(C |D|, |D_f|) is zero whichever way the test goes.
#ifndef MHD_PPM_SIGN_INT
#define MHD_PPM_SIGN_INT 1
#endif
__device__ __forceinline__ bool same_sign(double f, double a, double b) {
  if (MHD_PPM_SIGN_INT) return ((hi32(f) ^ hi32(a)) | (hi32(f) ^ hi32(b))) >= 0;
  return (f * a > 0.0) && (f * b > 0.0);
}
__device__ __forceinline__ bool same_sign(double f, double a, double b, double c) {
  if (MHD_PPM_SIGN_INT) return ((hi32(f) ^ hi32(a)) | (hi32(f) ^ hi32(b)) | (hi32(f) ^ hi32(c))) >= 0;
  return (f * a > 0.0) && (f * b > 0.0) && (f * c > 0.0);
}

__device__ __forceinline__ double ppm_face(double qa, double qb, double qc, double qd) {
  const double C = 1.25;
  const double sbc = qb + qc;
  const double qf = (7.0 / 12.0) * sbc - (1.0 / 12.0) * (qa + qd);
  const double Df = 3.0 * (qb - 2.0 * qf + qc);
  const double Dj = qa - 2.0 * qb + qc;
  const double Dj1 = qb - 2.0 * qc + qd;
  const bool same = same_sign(Df, Dj, Dj1);
  const double Dlim = select_(same, copysign(amin_(C * amin_(Dj, Dj1), Df), Df), 0.0);
  const double qlim = 0.5 * sbc - Dlim * (1.0 / 6.0);
  return ((qf - qb) * (qc - qf) < 0.0) ? qlim : qf;
}

__device__ __forceinline__ void ppm_scalar(double q0, double q1, double q2, double q3, double q4,
                                           double &qlo, double &qhi) {
  const double C = 1.25;
  const double qm = ppm_face(q0, q1, q2, q3);
  const double qp = ppm_face(q1, q2, q3, q4);
  const double qi = q2;
  // reading R7: differences that are zero to round-off count as zero in the extremum test
  const double tau = 1e-12 * fabs(amax_(q1, amax_(q2, q3)));
  double dm = qi - qm, dp = qp - qi, e3 = q3 - qi, e1 = qi - q1;
  const bool zm = fabs(dm) <= tau, zp = fabs(dp) <= tau, z3 = fabs(e3) <= tau, z1 = fabs(e1) <= tau;
  dm = zm ? 0.0 : dm;
  dp = zp ? 0.0 : dp;
  // "dm dp <= 0 or e3 e1 <= 0": a flushed difference, or a pair of opposite sign (the flush predicates are
  // the zero tests; the sign bits of the unflushed differences do the rest)
  const bool extremum = MHD_PPM_SIGN_INT
                            ? (zm || zp || z3 || z1 || ((hi32(dm) ^ hi32(dp)) | (hi32(e3) ^ hi32(e1))) < 0)
                            : (dm * dp <= 0.0) || ((z3 ? 0.0 : e3) * (z1 ? 0.0 : e1) <= 0.0);
  // at an extremum: the parabola's curvature limited against the cell curvatures
  const double Df = 6.0 * (qm - 2.0 * qi + qp);
  const double Dm1 = q0 - 2.0 * q1 + q2;
  const double D0 = q1 - 2.0 * q2 + q3;
  const double Dp1 = q2 - 2.0 * q3 + q4;
  const bool same = same_sign(Df, Dm1, D0, Dp1);
  const double Dlim = select_(same, copysign(amin_(C * amin_(Dm1, amin_(D0, Dp1)), Df), Df), 0.0);
  const bool big = fabs(Df) > max_(tau, 1e-290);          // (the floor keeps rcp off denormals)
  const double r = big ? Dlim * rcp(big ? Df : 1.0) : 0.0;
  const bool shrink = r <= 1.0 - 1e-12;
  const double qmE = shrink ? qi - r * dm : qm, qpE = shrink ? qi + r * dp : qp;
  // elsewhere: no overshoot of the parabola inside the cell
  const double qmM = (fabs(dm) >= 2.0 * fabs(dp)) ? qi - 2.0 * dp : qm;
  const double qpM = (fabs(dp) >= 2.0 * fabs(dm)) ? qi + 2.0 * dm : qp;
  qlo = extremum ? qmE : qmM;
  qhi = extremum ? qpE : qpM;
}
#endif

// Wm2..Wp2 = W_{i-2..i+2}; bx0 = cell-centred normal field of cell i
__device__ __forceinline__ void ppmc(double gamma, const W7 &Wm2, const W7 &Wm1, const W7 &W0,
                                     const W7 &Wp1, const W7 &Wp2, double bx0, W7 &Wlo, W7 &Whi) {
  Eig e;
  eig_setup(e, gamma, W0, bx0);
  C7 q0 = eig_left(e, Wm2), q1 = eig_left(e, Wm1), q2 = eig_left(e, W0), q3 = eig_left(e, Wp1),
     q4 = eig_left(e, Wp2);
  C7 lo, hi;
  ppm_scalar(q0.c0, q1.c0, q2.c0, q3.c0, q4.c0, lo.c0, hi.c0);
  ppm_scalar(q0.c1, q1.c1, q2.c1, q3.c1, q4.c1, lo.c1, hi.c1);
  ppm_scalar(q0.c2, q1.c2, q2.c2, q3.c2, q4.c2, lo.c2, hi.c2);
  ppm_scalar(q0.c3, q1.c3, q2.c3, q3.c3, q4.c3, lo.c3, hi.c3);
  ppm_scalar(q0.c4, q1.c4, q2.c4, q3.c4, q4.c4, lo.c4, hi.c4);
  ppm_scalar(q0.c5, q1.c5, q2.c5, q3.c5, q4.c5, lo.c5, hi.c5);
  ppm_scalar(q0.c6, q1.c6, q2.c6, q3.c6, q4.c6, lo.c6, hi.c6);
  Wlo = eig_right(e, lo);
  Whi = eig_right(e, hi);
}

// PPMP (PAPER.md:263 applied to the PPM of O10): the limited parabola per primitive variable
__device__ __forceinline__ void ppmp(const W7 &Wm2, const W7 &Wm1, const W7 &W0, const W7 &Wp1, const W7 &Wp2,
                                     W7 &Wlo, W7 &Whi) {
  ppm_scalar(Wm2.rho, Wm1.rho, W0.rho, Wp1.rho, Wp2.rho, Wlo.rho, Whi.rho);
  ppm_scalar(Wm2.u, Wm1.u, W0.u, Wp1.u, Wp2.u, Wlo.u, Whi.u);
  ppm_scalar(Wm2.v, Wm1.v, W0.v, Wp1.v, Wp2.v, Wlo.v, Whi.v);
  ppm_scalar(Wm2.w, Wm1.w, W0.w, Wp1.w, Wp2.w, Wlo.w, Whi.w);
  ppm_scalar(Wm2.P, Wm1.P, W0.P, Wp1.P, Wp2.P, Wlo.P, Whi.P);
  ppm_scalar(Wm2.by, Wm1.by, W0.by, Wp1.by, Wp2.by, Wlo.by, Whi.by);
  ppm_scalar(Wm2.bz, Wm1.bz, W0.bz, Wp1.bz, Wp2.bz, Wlo.bz, Whi.bz);
}

// ---------------------------------------------------------------------------------------
// CT edge field, Eq. 15-18 (readings O6, G5-G7).  Edge along c at
// (ia-1/2, ib-1/2), (a,b,c) cyclic.  Ea0/Ea1 = E_c on the a-faces (ia-1/2, ib) / (ia-1/2, ib-1);
// Eb0/Eb1 = E_c on the b-faces (ia, ib-1/2) / (ia-1, ib-1/2); M* the mass fluxes on those
// faces; Er00, Er10, Er01, Er11 = reference field of cells (ia,ib), (ia-1,ib), (ia,ib-1),
// (ia-1,ib-1).  All Delta factors of Eq. 15 and 17 cancel.
// ---------------------------------------------------------------------------------------
// Eq. 16 (G6): upwind by the sign of the interface mass flux, average where it is zero.  Every mass
// flux comes out of hlld(), which returns either +0.0 (reading R6) or a normal number, so the sign
// and the zero are read off the upper word on the integer pipe.
__device__ __forceinline__ double upwind(double M, double from_lower, double from_upper) {
  const int h = hi32(M);
  const double avg = 0.5 * (from_lower + from_upper);
  return (h >= 0x00100000) ? from_lower : ((h < 0 && h != (int)0x80000000) ? from_upper : avg);
}

__device__ __forceinline__ double ct_edge(double Ea0, double Ea1, double Eb0, double Eb1, double Ma0,
                                          double Ma1, double Mb0, double Mb1, double Er00,
                                          double Er10, double Er01, double Er11) {
  double T1 = upwind(Ma0, Eb1 - Er10, Eb0 - Er00);
  double T2 = upwind(Ma1, Eb1 - Er11, Eb0 - Er01);
  double T3 = upwind(Mb0, Ea1 - Er01, Ea0 - Er00);
  double T4 = upwind(Mb1, Ea1 - Er11, Ea0 - Er10);
  return 0.25 * (Ea0 + Ea1 + Eb0 + Eb1) + 0.25 * (T1 + T2 + T3 + T4);
}

}  // namespace mhd
