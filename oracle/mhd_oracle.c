/*
 * oracle/mhd_oracle.c  --  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * A plain, slow, fp64 CPU statement of the Van Leer + Constrained Transport
 * (VL+CT) ideal-MHD time step of Cholla-MHD (arxiv 2402.05240), written from
 * the paper (/root/reference/PAPER.md, cited below as PAPER.md:<line>) and from
 * the readings listed in SURVEY.md section 8(c) (cited as O0..O12, G1..G24) and
 * restated in DESIGN.md.  It exists only so that tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs can check and time the
 * CUDA path against it.  Nothing in the product path may import, link or call
 * anything in this directory, and this file shares no code, header, table or
 * helper with paper_2402_05240_b200/csrc.
 *
 * Style: every function follows the paper's step order and notation; there is
 * no blocking, fusion or reordering.  All intermediates of a time step (fluxes
 * on every face, edge electric fields, the half-step state) are materialised
 * in full arrays.  The only concession to run time is an OpenMP "parallel for"
 * on the outermost k loop of each stage (independent iterations, no change of
 * arithmetic), used by bench.py's cpu_baseline.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/build.py).
 * No -ffast-math.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): T1..T14 of SURVEY.md 8(c); for the
 * primitive-variable variants PLMP / PPMP: the scalar
 * limiter of Eq. 26-28 typed out per component, agreement with PLMC on a single entropy wave,
 * the scalar PPM per variable, T1, T8 (2nd-order linear-wave convergence) and T10.
 * Parity unpinned (choice among valid variants, no author code or printed
 * numbers to compare against): HLLD wave-speed estimate and degeneracy
 * tolerance (G15), eigenvector normalisation in degenerate states (G16), the
 * PPM variant (G17, O10; its constant C is bracketed by a smooth-extremum pin),
 * outflow boundary treatment (G24).  Each of these is
 * pinned to the mathematics it must satisfy (consistency, exactness on
 * polynomials, L.R = I ...) but not to the authors' code.
 *
 * Layout (O0): unit box, cell (i,j,k), i fastest, Delta_a = 1/n_a.  Conserved
 * rho, m_x, m_y, m_z, E at cell centres; B_a on the LOWER a-face of each cell
 * (Eq. 20 indexing B_{x,i-1/2}).  Arrays carry ng ghost layers
 * on every side; ng = 3 + (stencil radius of the reconstruction), so that one
 * ghost fill per step suffices.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#define NF 8 /* rho mx my mz E bx by bz */

/* ------------------------------------------------------------------ */
/* O2 / Eq. 12: fast magnetosonic speed squared along   */
/* the direction whose field component is bn.                          */
/* ------------------------------------------------------------------ */
static double fast_speed_sq(double gamma, double rho, double P, double bn,
                            double bt1, double bt2)
{
    double gp = gamma * P;
    double b2 = bn * bn + bt1 * bt1 + bt2 * bt2;
    double s = gp + b2;
    double disc = s * s - 4.0 * gp * bn * bn;
    if (disc < 0.0) disc = 0.0; /* round-off guard, reading R3 */
    return (s + sqrt(disc)) / (2.0 * rho);
}

/* ------------------------------------------------------------------ */
/* O4: HLLD (Miyoshi & Kusano 2005, cited PAPER.md:149).               */
/* W = (rho, u, v, w, P, By, Bz) in solver-local axes; bx = face-normal */
/* field.  F = (mass, mom_n, mom_t1, mom_t2, energy, By-flux, Bz-flux). */
/* ------------------------------------------------------------------ */
static void phys_flux(const double W[7], double bx, double e, double pT,
                      double F[7])
{
    double rho = W[0], u = W[1], v = W[2], w = W[3], by = W[5], bz = W[6];
    /* Eq. 8 without the zero row */
    F[0] = rho * u;
    F[1] = rho * u * u + pT - bx * bx;
    F[2] = rho * u * v - bx * by;
    F[3] = rho * u * w - bx * bz;
    F[4] = u * (e + pT) - bx * (u * bx + v * by + w * bz);
    F[5] = by * u - bx * v;
    F[6] = bz * u - bx * w;
}

static void hlld_fan(double gamma, const double WL[7], const double WR[7],
                     double bx, double F[7])
{
    const double *Wa[2] = {WL, WR};
    double rho[2], u[2], v[2], w[2], P[2], by[2], bz[2];
    double pT[2], e[2], cf[2], Fa[2][7], Ua[2][7];
    int s, c;
    for (s = 0; s < 2; s++) {
        rho[s] = Wa[s][0]; u[s] = Wa[s][1]; v[s] = Wa[s][2]; w[s] = Wa[s][3];
        P[s] = Wa[s][4]; by[s] = Wa[s][5]; bz[s] = Wa[s][6];
        double b2 = bx * bx + by[s] * by[s] + bz[s] * bz[s];
        pT[s] = P[s] + 0.5 * b2;
        e[s] = P[s] / (gamma - 1.0)
             + 0.5 * rho[s] * (u[s] * u[s] + v[s] * v[s] + w[s] * w[s])
             + 0.5 * b2;
        cf[s] = sqrt(fast_speed_sq(gamma, rho[s], P[s], bx, by[s], bz[s]));
        phys_flux(Wa[s], bx, e[s], pT[s], Fa[s]);
        Ua[s][0] = rho[s]; Ua[s][1] = rho[s] * u[s]; Ua[s][2] = rho[s] * v[s];
        Ua[s][3] = rho[s] * w[s]; Ua[s][4] = e[s]; Ua[s][5] = by[s];
        Ua[s][6] = bz[s];
    }
    /* outer wave speeds (G15: Davis-type estimate with max(cfL, cfR)) */
    double cfmax = fmax(cf[0], cf[1]);
    double S[2];
    S[0] = fmin(u[0], u[1]) - cfmax;
    S[1] = fmax(u[0], u[1]) + cfmax;

    if (S[0] > 0.0) { for (c = 0; c < 7; c++) F[c] = Fa[0][c]; return; }
    if (S[1] < 0.0) { for (c = 0; c < 7; c++) F[c] = Fa[1][c]; return; }

    /* entropy (middle) wave speed and total pressure of the Riemann fan */
    double sduL = (S[0] - u[0]) * rho[0];
    double sduR = (S[1] - u[1]) * rho[1];
    double den = sduR - sduL;
    double SM = (sduR * u[1] - sduL * u[0] - pT[1] + pT[0]) / den;
    double pTs = (sduR * pT[0] - sduL * pT[1]
                  + rho[0] * rho[1] * (S[1] - u[1]) * (S[0] - u[0]) * (u[1] - u[0])) / den;

    /* single-star states */
    double rhos[2], vs[2], ws[2], bys[2], bzs[2], es[2], Us[2][7], Sstar[2];
    for (s = 0; s < 2; s++) {
        double Su = S[s] - u[s];
        double SSm = S[s] - SM;
        rhos[s] = rho[s] * (Su / SSm);
        double D = rho[s] * Su * SSm - bx * bx;
        if (fabs(D) < 1e-8 * pTs) {
            /* degenerate 0/0 case of M&K: no jump in the tangential fields */
            vs[s] = v[s]; ws[s] = w[s]; bys[s] = by[s]; bzs[s] = bz[s];
        } else {
            double fv = bx * (SM - u[s]) / D;
            double fb = (rho[s] * Su * Su - bx * bx) / D;
            vs[s] = v[s] - by[s] * fv;
            ws[s] = w[s] - bz[s] * fv;
            bys[s] = by[s] * fb;
            bzs[s] = bz[s] * fb;
        }
        double vb = u[s] * bx + v[s] * by[s] + w[s] * bz[s];
        double vbs = SM * bx + vs[s] * bys[s] + ws[s] * bzs[s];
        es[s] = (Su * e[s] - pT[s] * u[s] + pTs * SM + bx * (vb - vbs)) / SSm;
        Us[s][0] = rhos[s]; Us[s][1] = rhos[s] * SM; Us[s][2] = rhos[s] * vs[s];
        Us[s][3] = rhos[s] * ws[s]; Us[s][4] = es[s]; Us[s][5] = bys[s];
        Us[s][6] = bzs[s];
    }
    Sstar[0] = SM - fabs(bx) / sqrt(rhos[0]);
    Sstar[1] = SM + fabs(bx) / sqrt(rhos[1]);

    /* F*_alpha = F_alpha + S_alpha (U*_alpha - U_alpha) */
    if (Sstar[0] >= 0.0) {
        for (c = 0; c < 7; c++) F[c] = Fa[0][c] + S[0] * (Us[0][c] - Ua[0][c]);
        return;
    }
    if (Sstar[1] <= 0.0) {
        for (c = 0; c < 7; c++) F[c] = Fa[1][c] + S[1] * (Us[1][c] - Ua[1][c]);
        return;
    }

    /* double-star states */
    double sgn = (bx > 0.0) ? 1.0 : ((bx < 0.0) ? -1.0 : 0.0);
    double rL = sqrt(rhos[0]), rR = sqrt(rhos[1]);
    double inv = 1.0 / (rL + rR);
    double vss = (rL * vs[0] + rR * vs[1] + (bys[1] - bys[0]) * sgn) * inv;
    double wss = (rL * ws[0] + rR * ws[1] + (bzs[1] - bzs[0]) * sgn) * inv;
    double byss = (rL * bys[1] + rR * bys[0] + rL * rR * (vs[1] - vs[0]) * sgn) * inv;
    double bzss = (rL * bzs[1] + rR * bzs[0] + rL * rR * (ws[1] - ws[0]) * sgn) * inv;
    double vbss = SM * bx + vss * byss + wss * bzss;
    s = (SM >= 0.0) ? 0 : 1;
    {
        double vbs = SM * bx + vs[s] * bys[s] + ws[s] * bzs[s];
        double r = (s == 0) ? rL : rR;
        double ess = (s == 0) ? es[s] - r * (vbs - vbss) * sgn
                              : es[s] + r * (vbs - vbss) * sgn;
        double Uss[7];
        Uss[0] = rhos[s]; Uss[1] = rhos[s] * SM; Uss[2] = rhos[s] * vss;
        Uss[3] = rhos[s] * wss; Uss[4] = ess; Uss[5] = byss; Uss[6] = bzss;
        /* F**_alpha = F*_alpha + S*_alpha (U**_alpha - U*_alpha) */
        for (c = 0; c < 7; c++)
            F[c] = Fa[s][c] + S[s] * (Us[s][c] - Ua[s][c])
                 + Sstar[s] * (Uss[c] - Us[s][c]);
    }
}

/* Pin support (tests/test_oracle_guards.py): the two round-off guards of readings R6 and R7 can be
 * switched off, so that a -m "not gpu" test can show that they act on round-off ties only (the
 * linear-wave errors, the Brio-Wu run and the Sod run do not move when they are off).  Both are ON
 * in every other use; the CUDA path has no such switch. */
static int guard_r6 = 1, guard_r7 = 1;
void oracle_set_guards(int r6, int r7) { guard_r6 = r6; guard_r7 = r7; }

/* HLLD as used by the scheme: the fan solution above, with the mass flux
 * set to exactly zero when it is zero to round-off (reading R6).
 * Eq. 16 (G6) upwinds the CT terms by the sign of the
 * interface mass flux and averages "otherwise"; between mirror-image states
 * (u_L = -u_R, equal rho, P, |B|: every symmetric test problem has such
 * faces) the contact is analytically at rest, but F_rho = F + S (U* - U)
 * leaves a residue of a few 1e-16 whose sign is noise.  A contact slower than
 * 1e-13 of the fast speed counts as at rest. */
void oracle_hlld(double gamma, const double WL[7], const double WR[7],
                 double bx, double F[7])
{
    double cfL = sqrt(fast_speed_sq(gamma, WL[0], WL[4], bx, WL[5], WL[6]));
    double cfR = sqrt(fast_speed_sq(gamma, WR[0], WR[4], bx, WR[5], WR[6]));
    hlld_fan(gamma, WL, WR, bx, F);
    if (guard_r6 && fabs(F[0]) <= 1e-13 * (WL[0] + WR[0]) * fmax(cfL, cfR)) F[0] = 0.0;
}

/* ------------------------------------------------------------------ */
/* O9: eigen-system of the primitive-variable MHD equations            */
/* (Stone et al. 2008 App. A, cited PAPER.md:249).  W as above, bx the  */
/* cell-centred normal field.  Wave order u-cf,u-ca,u-cs,u,u+cs,u+ca,   */
/* u+cf.  L[m][c]: row m = left eigenvector m;  R[c][m]: column m =     */
/* right eigenvector m; c runs over (rho,u,v,w,P,By,Bz).                */
/* ------------------------------------------------------------------ */
void oracle_eigensystem(double gamma, const double W[7], double bx,
                        double lambda[7], double L[49], double R[49])
{
    double rho = W[0], u = W[1], P = W[4], by = W[5], bz = W[6];
    double a2 = gamma * P / rho;
    double a = sqrt(a2);
    double cf2 = fast_speed_sq(gamma, rho, P, bx, by, bz);
    double ca2 = bx * bx / rho;
    double cs2 = (cf2 > 0.0) ? a2 * ca2 / cf2 : 0.0;
    double cf = sqrt(cf2), cs = sqrt(cs2), ca = sqrt(ca2);
    double bperp = sqrt(by * by + bz * bz);
    double betay, betaz, alf, als;
    if (bperp == 0.0) { betay = 1.0; betaz = 0.0; }
    else { betay = by / bperp; betaz = bz / bperp; }
    if (cf2 - cs2 == 0.0) { alf = 1.0; als = 0.0; }
    else {
        double af2 = (a2 - cs2) / (cf2 - cs2);
        double as2 = (cf2 - a2) / (cf2 - cs2);
        if (af2 < 0.0) af2 = 0.0; if (af2 > 1.0) af2 = 1.0;
        if (as2 < 0.0) as2 = 0.0; if (as2 > 1.0) as2 = 1.0;
        alf = sqrt(af2); als = sqrt(as2);
    }
    double S = (bx >= 0.0) ? 1.0 : -1.0;
    double sr = sqrt(rho);
    double Cff = cf * alf, Css = cs * als;
    double Qf = cf * alf * S, Qs = cs * als * S;
    double Af = a * alf * sr, As = a * als * sr;
    double N = 1.0 / (2.0 * a2);
    int m, c;

    lambda[0] = u - cf; lambda[1] = u - ca; lambda[2] = u - cs; lambda[3] = u;
    lambda[4] = u + cs; lambda[5] = u + ca; lambda[6] = u + cf;

    for (m = 0; m < 49; m++) { L[m] = 0.0; R[m] = 0.0; }
#define RR(c, m) R[(c) * 7 + (m)]
#define LL(m, c) L[(m) * 7 + (c)]
    /* right eigenvectors (columns) */
    RR(0,0) = rho * alf;      RR(0,2) = rho * als;      RR(0,3) = 1.0;
    RR(0,4) = rho * als;      RR(0,6) = rho * alf;
    RR(1,0) = -Cff;           RR(1,2) = -Css;           RR(1,4) = Css;   RR(1,6) = Cff;
    RR(2,0) = Qs * betay;     RR(2,1) = -betaz;         RR(2,2) = -Qf * betay;
    RR(2,4) = Qf * betay;     RR(2,5) = betaz;          RR(2,6) = -Qs * betay;
    RR(3,0) = Qs * betaz;     RR(3,1) = betay;          RR(3,2) = -Qf * betaz;
    RR(3,4) = Qf * betaz;     RR(3,5) = -betay;         RR(3,6) = -Qs * betaz;
    RR(4,0) = rho * a2 * alf; RR(4,2) = rho * a2 * als;
    RR(4,4) = rho * a2 * als; RR(4,6) = rho * a2 * alf;
    RR(5,0) = As * betay;     RR(5,1) = -betaz * S * sr; RR(5,2) = -Af * betay;
    RR(5,4) = -Af * betay;    RR(5,5) = -betaz * S * sr; RR(5,6) = As * betay;
    RR(6,0) = As * betaz;     RR(6,1) = betay * S * sr;  RR(6,2) = -Af * betaz;
    RR(6,4) = -Af * betaz;    RR(6,5) = betay * S * sr;  RR(6,6) = As * betaz;
    /* left eigenvectors (rows) */
    LL(0,1) = -N * Cff; LL(0,2) = N * Qs * betay; LL(0,3) = N * Qs * betaz;
    LL(0,4) = N * alf / rho; LL(0,5) = N * As * betay / rho; LL(0,6) = N * As * betaz / rho;
    LL(1,2) = -0.5 * betaz; LL(1,3) = 0.5 * betay;
    LL(1,5) = -0.5 * betaz * S / sr; LL(1,6) = 0.5 * betay * S / sr;
    LL(2,1) = -N * Css; LL(2,2) = -N * Qf * betay; LL(2,3) = -N * Qf * betaz;
    LL(2,4) = N * als / rho; LL(2,5) = -N * Af * betay / rho; LL(2,6) = -N * Af * betaz / rho;
    LL(3,0) = 1.0; LL(3,4) = -1.0 / a2;
    LL(4,1) = N * Css; LL(4,2) = N * Qf * betay; LL(4,3) = N * Qf * betaz;
    LL(4,4) = N * als / rho; LL(4,5) = -N * Af * betay / rho; LL(4,6) = -N * Af * betaz / rho;
    LL(5,2) = 0.5 * betaz; LL(5,3) = -0.5 * betay;
    LL(5,5) = -0.5 * betaz * S / sr; LL(5,6) = 0.5 * betay * S / sr;
    LL(6,1) = N * Cff; LL(6,2) = -N * Qs * betay; LL(6,3) = -N * Qs * betaz;
    LL(6,4) = N * alf / rho; LL(6,5) = N * As * betay / rho; LL(6,6) = N * As * betaz / rho;
#undef RR
#undef LL
    (void)c;
}

static void matvec7(const double M[49], const double x[7], double y[7])
{
    int r, c;
    for (r = 0; r < 7; r++) {
        double s = 0.0;
        for (c = 0; c < 7; c++) s += M[r * 7 + c] * x[c];
        y[r] = s;
    }
}

/* ------------------------------------------------------------------ */
/* O8: PLMC, Eq. 23-28.                             */
/* Wm, W0, Wp = W_{i-1}, W_i, W_{i+1}; bx0 = cell-centred normal field  */
/* of cell i.  Out: Wlo = W_{R,i-1/2}, Whi = W_{L,i+1/2}.               */
/* ------------------------------------------------------------------ */
void oracle_plmc(double gamma, const double Wm[7], const double W0[7],
                 const double Wp[7], double bx0, double Wlo[7], double Whi[7])
{
    double dL[7], dR[7], dC[7], dVL[7], aL[7], aR[7], aC[7], aVL[7], am[7], dWm[7];
    double lambda[7], L[49], R[49];
    int c;
    for (c = 0; c < 7; c++) {
        dL[c] = W0[c] - Wm[c];                 /* Eq. 23 */
        dR[c] = Wp[c] - W0[c];                 /* Eq. 24 */
        dC[c] = (Wp[c] - Wm[c]) / 2.0;         /* Eq. 25 */
        dVL[c] = (dL[c] * dR[c] > 0.0)         /* Eq. 26 (G10) */
               ? 2.0 * dL[c] * dR[c] / (dL[c] + dR[c]) : 0.0;
    }
    /* step 3: all four slopes projected with the eigenvectors of cell i */
    oracle_eigensystem(gamma, W0, bx0, lambda, L, R);
    matvec7(L, dL, aL); matvec7(L, dR, aR); matvec7(L, dC, aC); matvec7(L, dVL, aVL);
    /* step 4: Eq. 27 */
    for (c = 0; c < 7; c++) {
        if (aL[c] * aR[c] > 0.0) {
            double m = fmin(fmin(2.0 * fabs(aL[c]), 2.0 * fabs(aR[c])),
                            fmin(fabs(aC[c]), fabs(aVL[c])));
            double sg = (aC[c] > 0.0) ? 1.0 : ((aC[c] < 0.0) ? -1.0 : 0.0);
            am[c] = sg * m;
        } else am[c] = 0.0;
    }
    /* step 5 */
    matvec7(R, am, dWm);
    /* step 6: Eq. 28 */
    for (c = 0; c < 7; c++) {
        Whi[c] = W0[c] + dWm[c] / 2.0;
        Wlo[c] = W0[c] - dWm[c] / 2.0;
    }
}

/* ------------------------------------------------------------------ */
/* PLMP ("To limit in the primitive variables instead ...  */
/* skip steps 3 and 5"): Eq. 23-26, then the limiter of Eq. 27 applied   */
/* to the primitive differences themselves, then Eq. 28.                 */
/* ------------------------------------------------------------------ */
void oracle_plmp(const double Wm[7], const double W0[7], const double Wp[7],
                 double Wlo[7], double Whi[7])
{
    int c;
    for (c = 0; c < 7; c++) {
        double dL = W0[c] - Wm[c];                      /* Eq. 23 */
        double dR = Wp[c] - W0[c];                      /* Eq. 24 */
        double dC = (Wp[c] - Wm[c]) / 2.0;              /* Eq. 25 */
        double dVL = (dL * dR > 0.0) ? 2.0 * dL * dR / (dL + dR) : 0.0; /* Eq. 26 */
        double dm = 0.0;
        if (dL * dR > 0.0) {                            /* Eq. 27 on delta W */
            double m = fmin(fmin(2.0 * fabs(dL), 2.0 * fabs(dR)),
                            fmin(fabs(dC), fabs(dVL)));
            double sg = (dC > 0.0) ? 1.0 : ((dC < 0.0) ? -1.0 : 0.0);
            dm = sg * m;
        }
        Whi[c] = W0[c] + dm / 2.0;                      /* Eq. 28 */
        Wlo[c] = W0[c] - dm / 2.0;
    }
}

/* ------------------------------------------------------------------ */
/* O10: PPMC (reading G17 of Felker & Stone 2018, cited PAPER.md:231).  */
/* One characteristic variable: q[0..4] = q_{i-2..i+2}.                 */
/* ------------------------------------------------------------------ */
static double sgn3(double x) { return (x > 0.0) ? 1.0 : ((x < 0.0) ? -1.0 : 0.0); }

/* steps (1)+(2): limited 4th-order value on the face between cells j, j+1;
 * qa..qd = q_{j-1}, q_j, q_{j+1}, q_{j+2} */
static double ppm_face(double qa, double qb, double qc, double qd)
{
    const double C = 1.25;
    double qf = (7.0 / 12.0) * (qb + qc) - (1.0 / 12.0) * (qa + qd);
    if ((qf - qb) * (qc - qf) < 0.0) {
        double Df = 3.0 * (qb - 2.0 * qf + qc);
        double Dj = qa - 2.0 * qb + qc;
        double Dj1 = qb - 2.0 * qc + qd;
        double Dlim = 0.0;
        if (sgn3(Df) == sgn3(Dj) && sgn3(Df) == sgn3(Dj1) && sgn3(Df) != 0.0)
            Dlim = sgn3(Df) * fmin(fmin(C * fabs(Dj), C * fabs(Dj1)), fabs(Df));
        qf = 0.5 * (qb + qc) - Dlim / 6.0;
    }
    return qf;
}

void oracle_ppm_scalar(const double q[5], double *qlo, double *qhi)
{
    const double C = 1.25;
    double qm = ppm_face(q[0], q[1], q[2], q[3]); /* lower face of cell i */
    double qp = ppm_face(q[1], q[2], q[3], q[4]); /* upper face of cell i */
    double qi = q[2];
    /* step (3).  Reading O10 / R7: the four differences whose signs classify the cell as an
     * extremum are zero when they are zero to round-off (|x| <= 1e-12 max|q_{i-1..i+1}|, the
     * same guard as for D_f below).  On a plateau next to a jump, or between mirror-image
     * cells, they are analytically zero, and the two branches give different faces. */
    double tau = 1e-12 * fmax(fabs(q[1]), fmax(fabs(q[2]), fabs(q[3])));
    double dm = qi - qm, dp = qp - qi, e3 = q[3] - qi, e1 = qi - q[1];
    if (guard_r7) {
        if (fabs(dm) <= tau) dm = 0.0;
        if (fabs(dp) <= tau) dp = 0.0;
        if (fabs(e3) <= tau) e3 = 0.0;
        if (fabs(e1) <= tau) e1 = 0.0;
    }
    if (dm * dp <= 0.0 || e3 * e1 <= 0.0) {
        double Df = 6.0 * (qm - 2.0 * qi + qp);
        double Dm1 = q[0] - 2.0 * q[1] + q[2];
        double D0 = q[1] - 2.0 * q[2] + q[3];
        double Dp1 = q[2] - 2.0 * q[3] + q[4];
        double Dlim = 0.0, r = 0.0;
        double s = sgn3(Df);
        if (s != 0.0 && s == sgn3(Dm1) && s == sgn3(D0) && s == sgn3(Dp1))
            Dlim = s * fmin(fmin(C * fabs(Dm1), C * fabs(D0)),
                            fmin(C * fabs(Dp1), fabs(Df)));
        if (fabs(Df) > tau) r = Dlim / Df;
        if (r <= 1.0 - 1e-12) { qm = qi - r * dm; qp = qi + r * dp; }
    } else {
        if (fabs(dm) >= 2.0 * fabs(dp)) qm = qi - 2.0 * dp;
        if (fabs(dp) >= 2.0 * fabs(dm)) qp = qi + 2.0 * dm;
    }
    *qlo = qm; *qhi = qp;
}

/* Ws[5][7] = W_{i-2..i+2}; bx0 = cell-centred normal field of cell i */
void oracle_ppmc(double gamma, const double *Ws, double bx0,
                 double Wlo[7], double Whi[7])
{
    double lambda[7], L[49], R[49], q[5][7], qlo[7], qhi[7];
    int s, m;
    oracle_eigensystem(gamma, Ws + 2 * 7, bx0, lambda, L, R);
    for (s = 0; s < 5; s++) matvec7(L, Ws + s * 7, q[s]);
    for (m = 0; m < 7; m++) {
        double qq[5];
        for (s = 0; s < 5; s++) qq[s] = q[s][m];
        oracle_ppm_scalar(qq, &qlo[m], &qhi[m]);
    }
    matvec7(R, qlo, Wlo); /* step (4) */
    matvec7(R, qhi, Whi);
}

/* PPMP (PAPER.md:263 applied to the PPM of O10): the same limited parabola,
 * variable by variable on the primitives, no characteristic projection. */
void oracle_ppmp(const double *Ws, double Wlo[7], double Whi[7])
{
    int s, c;
    for (c = 0; c < 7; c++) {
        double qq[5];
        for (s = 0; s < 5; s++) qq[s] = Ws[s * 7 + c];
        oracle_ppm_scalar(qq, &Wlo[c], &Whi[c]);
    }
}

/* ------------------------------------------------------------------ */
/* O6: CT edge field, Eq. 15-18 (readings G5-G7).     */
/* Edge along c at (ia-1/2, ib-1/2), (a,b,c) cyclic.                    */
/*  Ea0 = E_c on a-face (ia-1/2, ib)    Ea1 = E_c on a-face (ia-1/2, ib-1) */
/*  Eb0 = E_c on b-face (ia, ib-1/2)    Eb1 = E_c on b-face (ia-1, ib-1/2) */
/*  Ma0, Ma1, Mb0, Mb1 = mass flux on those same four faces              */
/*  Er00 = E_ref cell (ia,ib), Er10 = (ia-1,ib), Er01 = (ia,ib-1),       */
/*  Er11 = (ia-1,ib-1)                                                   */
/* ------------------------------------------------------------------ */
static double upwind(double M, double from_lower, double from_upper)
{
    if (M > 0.0) return from_lower;
    if (M < 0.0) return from_upper;
    return 0.5 * (from_lower + from_upper);
}

double oracle_ct_edge(double Ea0, double Ea1, double Eb0, double Eb1,
                      double Ma0, double Ma1, double Mb0, double Mb1,
                      double Er00, double Er10, double Er01, double Er11)
{
    /* Eq. 17: each slope is 2 (face value on the edge's side - reference) / Delta,
     * taken in the direction towards the edge; Eq. 15 weights it by Delta / 8. */
    double T1 = upwind(Ma0, Eb1 - Er10, Eb0 - Er00); /* (a-1/2, b-1/4) */
    double T2 = upwind(Ma1, Eb1 - Er11, Eb0 - Er01); /* (a-1/2, b-3/4) */
    double T3 = upwind(Mb0, Ea1 - Er01, Ea0 - Er00); /* (a-1/4, b-1/2) */
    double T4 = upwind(Mb1, Ea1 - Er11, Ea0 - Er10); /* (a-3/4, b-1/2) */
    return 0.25 * (Ea0 + Ea1 + Eb0 + Eb1) + 0.25 * (T1 + T2 + T3 + T4);
}

/* ================================================================== */
/* Grid driver                                                         */
/* ================================================================== */
typedef struct {
    int inited;
    int n[3], ng, N[3];
    long s[3], ntot;
    double gamma, d[3];
    int recon;     /* 0 PCM, 1 PLMC, 2 PPMC, 3 PLMP, 4 PPMP */
    int radius;    /* stencil radius of the reconstruction: 0, 1, 2, 1, 2 */
    int bc[3];     /* 0 periodic, 1 outflow */
    double *U[NF];    /* state at t^n */
    double *Uh[NF];   /* state at t^{n+1/2} */
    double *F[3][7];  /* face fluxes per sweep direction, solver-local order */
    double *E[3];     /* edge electric fields */
} Grid;

static Grid G;

#define IDX(g, i, j, k) (((long)(i) + (g)->ng) + (g)->N[0] * (((long)(j) + (g)->ng) + (long)(g)->N[1] * ((long)(k) + (g)->ng)))

int oracle_finalize(void)
{
    int f, a, c;
    if (!G.inited) return 0;
    for (f = 0; f < NF; f++) { free(G.U[f]); free(G.Uh[f]); }
    for (a = 0; a < 3; a++) { for (c = 0; c < 7; c++) free(G.F[a][c]); free(G.E[a]); }
    memset(&G, 0, sizeof(G));
    return 0;
}

int oracle_init(int nx, int ny, int nz, double gamma, int recon)
{
    int a, c, f;
    if (nx < 1 || ny < 1 || nz < 1 || !(gamma > 1.0) || recon < 0 || recon > 4) return -1;
    oracle_finalize();
    G.n[0] = nx; G.n[1] = ny; G.n[2] = nz;
    G.recon = recon;
    G.radius = (recon == 0) ? 0 : ((recon == 1 || recon == 3) ? 1 : 2);
    G.ng = 3 + G.radius; /* stencil radius: PCM 0, PLMC/PLMP 1, PPMC/PPMP 2 */
    G.gamma = gamma;
    for (a = 0; a < 3; a++) {
        G.N[a] = G.n[a] + 2 * G.ng;
        G.d[a] = 1.0 / G.n[a];
        G.bc[a] = 0;
    }
    G.s[0] = 1; G.s[1] = G.N[0]; G.s[2] = (long)G.N[0] * G.N[1];
    G.ntot = (long)G.N[0] * G.N[1] * G.N[2];
    for (f = 0; f < NF; f++) {
        G.U[f] = calloc(G.ntot, sizeof(double));
        G.Uh[f] = calloc(G.ntot, sizeof(double));
        if (!G.U[f] || !G.Uh[f]) return -3;
    }
    for (a = 0; a < 3; a++) {
        for (c = 0; c < 7; c++) { G.F[a][c] = calloc(G.ntot, sizeof(double)); if (!G.F[a][c]) return -3; }
        G.E[a] = calloc(G.ntot, sizeof(double)); if (!G.E[a]) return -3;
    }
    G.inited = 1;
    return 0;
}

/* Domain lengths (default 1 x 1 x 1): Delta_a = L_a / n_a.  The paper's non-cubic test boxes
 * (3 x 1.5 x 1.5; 1 x 1 x 2; 1 x 1.5 x 1) keep cubic cells. */
int oracle_set_domain(double lx, double ly, double lz)
{
    double L[3] = {lx, ly, lz};
    int a;
    if (!G.inited) return -2;
    for (a = 0; a < 3; a++) if (!(L[a] > 0.0)) return -1;
    for (a = 0; a < 3; a++) G.d[a] = L[a] / G.n[a];
    return 0;
}

int oracle_set_boundary(int axis, int kind)
{
    if (!G.inited) return -2;
    if (axis < 0 || axis > 2 || kind < 0 || kind > 1) return -1;
    G.bc[axis] = kind;
    return 0;
}

/* O12: ghost fill of all 8 fields, axis by axis (x, y, z) over the full
 * extent of the other axes so that edges and corners are filled too. */
static void fill_ghosts(Grid *g, double *U[NF])
{
    int a, f;
    for (a = 0; a < 3; a++) {
        int a1 = (a + 1) % 3, a2 = (a + 2) % 3;
        int na = g->n[a], ng = g->ng;
        for (f = 0; f < NF; f++) {
            int normalB = (f == 5 + a);
            long p, q;
            int i;
            for (q = 0; q < g->N[a2]; q++)
                for (p = 0; p < g->N[a1]; p++) {
                    long base = p * g->s[a1] + q * g->s[a2];
                    for (i = -ng; i < na + ng; i++) {
                        int src;
                        if (g->bc[a] == 0) {            /* periodic wrap */
                            if (i < 0) src = i + na;
                            else if (i >= na) src = i - na;
                            else continue;
                            /* tiny grids (n < ng): wrap repeatedly */
                            while (src < 0) src += na;
                            while (src >= na) src -= na;
                        } else {                        /* zero-gradient outflow */
                            if (normalB) {              /* faces 0..na are active */
                                if (i < 0) src = 0;
                                else if (i > na) src = na;
                                else continue;
                            } else {
                                if (i < 0) src = 0;
                                else if (i >= na) src = na - 1;
                                else continue;
                            }
                        }
                        U[f][base + (long)(i + ng) * g->s[a]] =
                            U[f][base + (long)(src + ng) * g->s[a]];
                    }
                }
        }
    }
}

int oracle_set_state(const double *rho, const double *mx, const double *my,
                     const double *mz, const double *E, const double *bx,
                     const double *by, const double *bz)
{
    const double *src[NF] = {rho, mx, my, mz, E, bx, by, bz};
    int f, i, j, k;
    if (!G.inited) return -2;
    for (f = 0; f < NF; f++) {
        int ex = G.n[0] + (f == 5), ey = G.n[1] + (f == 6), ez = G.n[2] + (f == 7);
        if (!src[f]) return -1;
        for (k = 0; k < ez; k++)
            for (j = 0; j < ey; j++)
                for (i = 0; i < ex; i++)
                    G.U[f][IDX(&G, i, j, k)] = src[f][i + (long)ex * (j + (long)ey * k)];
    }
    fill_ghosts(&G, G.U);
    return 0;
}

static int get_any(double *U[NF], double *rho, double *mx, double *my, double *mz,
                   double *E, double *bx, double *by, double *bz)
{
    double *dst[NF] = {rho, mx, my, mz, E, bx, by, bz};
    int f, i, j, k;
    if (!G.inited) return -2;
    for (f = 0; f < NF; f++) {
        int ex = G.n[0] + (f == 5), ey = G.n[1] + (f == 6), ez = G.n[2] + (f == 7);
        if (!dst[f]) continue;
        for (k = 0; k < ez; k++)
            for (j = 0; j < ey; j++)
                for (i = 0; i < ex; i++)
                    dst[f][i + (long)ex * (j + (long)ey * k)] = U[f][IDX(&G, i, j, k)];
    }
    return 0;
}

int oracle_get_state(double *rho, double *mx, double *my, double *mz, double *E,
                     double *bx, double *by, double *bz)
{
    return get_any(G.U, rho, mx, my, mz, E, bx, by, bz);
}

/* debug: the predictor's U^{n+1/2} of the last step */
int oracle_get_half_state(double *rho, double *mx, double *my, double *mz, double *E,
                          double *bx, double *by, double *bz)
{
    return get_any(G.Uh, rho, mx, my, mz, E, bx, by, bz);
}

/* debug: corrector flux component comp (0 mass, 1 mom_n, 2 mom_t1, 3 mom_t2, 4 energy, 5 B_t1, 6 B_t2;
 * solver-local order of sweep `axis`) on the lower axis-face of every active cell, as left by the last
 * step (the predictor's fluxes were overwritten by the corrector's).  Accessor only. */
int oracle_get_flux(int axis, int comp, double *out)
{
    int i, j, k;
    if (!G.inited) return -2;
    if (axis < 0 || axis > 2 || comp < 0 || comp > 6 || !out) return -1;
    for (k = 0; k < G.n[2]; k++)
        for (j = 0; j < G.n[1]; j++)
            for (i = 0; i < G.n[0]; i++)
                out[i + (long)G.n[0] * (j + (long)G.n[1] * k)] = G.F[axis][comp][IDX(&G, i, j, k)];
    return 0;
}

/* O1: primitives of one cell, recomputed wherever needed.
 * B_cc from Eq. 13. */
static void cell_prim(const Grid *g, double *const U[NF], long idx,
                      double *rho, double v[3], double *P, double B[3])
{
    int a;
    double r = U[0][idx];
    for (a = 0; a < 3; a++) {
        B[a] = 0.5 * (U[5 + a][idx] + U[5 + a][idx + g->s[a]]);
        v[a] = U[1 + a][idx] / r;
    }
    *rho = r;
    *P = (g->gamma - 1.0) * (U[4][idx]
          - 0.5 * r * (v[0] * v[0] + v[1] * v[1] + v[2] * v[2])
          - 0.5 * (B[0] * B[0] + B[1] * B[1] + B[2] * B[2]));
}

/* solver-local 1-D state for sweep a: (n,t1,t2) = (a,a+1,a+2) mod 3 (O0) */
static void cell_W(const Grid *g, double *const U[NF], long idx, int a,
                   double W[7], double *bn_cc)
{
    double rho, v[3], P, B[3];
    int t1 = (a + 1) % 3, t2 = (a + 2) % 3;
    cell_prim(g, U, idx, &rho, v, &P, B);
    W[0] = rho; W[1] = v[a]; W[2] = v[t1]; W[3] = v[t2]; W[4] = P;
    W[5] = B[t1]; W[6] = B[t2];
    *bn_cc = B[a];
}

/* O2 / Eq. 11 */
int oracle_compute_dt(double cfl, double *dt)
{
    int i, j, k, a;
    double tmin = INFINITY;
    if (!G.inited) return -2;
    if (!dt) return -1;
    for (k = 0; k < G.n[2]; k++)
        for (j = 0; j < G.n[1]; j++)
            for (i = 0; i < G.n[0]; i++) {
                double rho, v[3], P, B[3];
                cell_prim(&G, G.U, IDX(&G, i, j, k), &rho, v, &P, B);
                for (a = 0; a < 3; a++) {
                    double cf = sqrt(fast_speed_sq(G.gamma, rho, P, B[a],
                                                   B[(a + 1) % 3], B[(a + 2) % 3]));
                    double t = G.d[a] / (fabs(v[a]) + cf);
                    if (t < tmin) tmin = t;
                }
            }
    *dt = cfl * tmin;
    return 0;
}

/* Steps 2-3 / 6-7: interface states and HLLD flux on every a-face whose
 * stencil is available.  Face (index i along a) lies between cells i-1, i.
 * recon: 0 PCM (Eq. 14), 1 PLMC (O8), 2 PPMC (O10), 3 PLMP, 4 PPMP. */
static void reconstruct_cell(const Grid *g, double *const U[NF], long idx, int a,
                             int recon, double Wlo[7], double Whi[7])
{
    double W[5][7], bn[5];
    int s, c;
    if (recon == 0) {
        cell_W(g, U, idx, a, W[2], &bn[2]);
        for (c = 0; c < 7; c++) { Wlo[c] = W[2][c]; Whi[c] = W[2][c]; }
    } else if (recon == 1 || recon == 3) {
        for (s = 1; s <= 3; s++) cell_W(g, U, idx + (s - 2) * g->s[a], a, W[s], &bn[s]);
        if (recon == 1) oracle_plmc(g->gamma, W[1], W[2], W[3], bn[2], Wlo, Whi);
        else oracle_plmp(W[1], W[2], W[3], Wlo, Whi);
    } else {
        for (s = 0; s <= 4; s++) cell_W(g, U, idx + (s - 2) * g->s[a], a, W[s], &bn[s]);
        if (recon == 2) oracle_ppmc(g->gamma, (const double *)W, bn[2], Wlo, Whi);
        else oracle_ppmp((const double *)W, Wlo, Whi);
    }
}

static void sweep_fluxes(Grid *g, double *const U[NF], int a, int recon,
                         const int lo[3], const int hi[3])
{
    int k;
#pragma omp parallel for schedule(static)
    for (k = lo[2]; k < hi[2]; k++) {
        int i, j, c;
        for (j = lo[1]; j < hi[1]; j++)
            for (i = lo[0]; i < hi[0]; i++) {
                long idx = IDX(g, i, j, k);
                double WL[7], WR[7], tmp[7], Fl[7];
                /* left state = upper-face state of cell i-1; right = lower-face state of cell i */
                reconstruct_cell(g, U, idx - g->s[a], a, recon, tmp, WL);
                reconstruct_cell(g, U, idx, a, recon, WR, tmp);
                /* the longitudinal field is taken directly from the face */
                oracle_hlld(g->gamma, WL, WR, U[5 + a][idx], Fl);
                for (c = 0; c < 7; c++) g->F[a][c][idx] = Fl[c];
            }
    }
}

/* Step 4 / 8: edge fields E_c on edges (ia-1/2, ib-1/2, ic) */
static void ct_fields(Grid *g, double *const U[NF], const int lo[3][3], const int hi[3][3])
{
    int c;
    for (c = 0; c < 3; c++) {
        int a = (c + 1) % 3, b = (c + 2) % 3;
        long sa = g->s[a], sb = g->s[b];
        int k;
#pragma omp parallel for schedule(static)
        for (k = lo[c][2]; k < hi[c][2]; k++) {
            int i, j;
            for (j = lo[c][1]; j < hi[c][1]; j++)
                for (i = lo[c][0]; i < hi[c][0]; i++) {
                    long idx = IDX(g, i, j, k);
                    long cells[4] = {idx, idx - sa, idx - sb, idx - sa - sb};
                    double Er[4];
                    int q;
                    for (q = 0; q < 4; q++) { /* Eq. 18 */
                        double rho, v[3], P, B[3];
                        cell_prim(g, U, cells[q], &rho, v, &P, B);
                        Er[q] = -(v[a] * B[b] - v[b] * B[a]);
                    }
                    /* O5 / Table 1: on an a-face E_c = -F_a[B_t1];
                     * on a b-face E_c = +F_b[B_t2] */
                    double Ea0 = -g->F[a][5][idx], Ea1 = -g->F[a][5][idx - sb];
                    double Eb0 = g->F[b][6][idx], Eb1 = g->F[b][6][idx - sa];
                    double Ma0 = g->F[a][0][idx], Ma1 = g->F[a][0][idx - sb];
                    double Mb0 = g->F[b][0][idx], Mb1 = g->F[b][0][idx - sa];
                    g->E[c][idx] = oracle_ct_edge(Ea0, Ea1, Eb0, Eb1, Ma0, Ma1, Mb0, Mb1,
                                                  Er[0], Er[1], Er[2], Er[3]);
                }
        }
    }
}

/* Step 5 / 9 (O7): Uout = Ubase - dt/Delta * flux differences; face B from edge E */
static void update(Grid *g, double *const Ubase[NF], double *Uout[NF], double dt,
                   const int clo[3], const int chi[3],
                   const int flo[3][3], const int fhi[3][3])
{
    int k, a;
#pragma omp parallel for schedule(static)
    for (k = clo[2]; k < chi[2]; k++) {
        int i, j, a2;
        for (j = clo[1]; j < chi[1]; j++)
            for (i = clo[0]; i < chi[0]; i++) {
                long idx = IDX(g, i, j, k);
                double rho = Ubase[0][idx], E = Ubase[4][idx], m[3];
                m[0] = Ubase[1][idx]; m[1] = Ubase[2][idx]; m[2] = Ubase[3][idx];
                for (a2 = 0; a2 < 3; a2++) { /* Eq. 19 / 29, x then y then z */
                    long up = idx + g->s[a2];
                    double dtd = dt / g->d[a2];
                    rho -= dtd * (g->F[a2][0][up] - g->F[a2][0][idx]);
                    m[a2] -= dtd * (g->F[a2][1][up] - g->F[a2][1][idx]);
                    m[(a2 + 1) % 3] -= dtd * (g->F[a2][2][up] - g->F[a2][2][idx]);
                    m[(a2 + 2) % 3] -= dtd * (g->F[a2][3][up] - g->F[a2][3][idx]);
                    E -= dtd * (g->F[a2][4][up] - g->F[a2][4][idx]);
                }
                Uout[0][idx] = rho; Uout[1][idx] = m[0]; Uout[2][idx] = m[1];
                Uout[3][idx] = m[2]; Uout[4][idx] = E;
            }
    }
    for (a = 0; a < 3; a++) { /* Eq. 20-22 / 30-32 */
        int b = (a + 1) % 3, c = (a + 2) % 3;
        long sb = g->s[b], sc = g->s[c];
#pragma omp parallel for schedule(static)
        for (k = flo[a][2]; k < fhi[a][2]; k++) {
            int i, j;
            for (j = flo[a][1]; j < fhi[a][1]; j++)
                for (i = flo[a][0]; i < fhi[a][0]; i++) {
                    long idx = IDX(g, i, j, k);
                    Uout[5 + a][idx] = Ubase[5 + a][idx]
                        + dt / g->d[c] * (g->E[b][idx + sc] - g->E[b][idx])
                        - dt / g->d[b] * (g->E[c][idx + sb] - g->E[c][idx]);
                }
        }
    }
}

int oracle_step(double dt)
{
    Grid *g = &G;
    int a, c, x, r = g->radius, ng = g->ng;
    int lo[3], hi[3], elo[3][3], ehi[3][3], clo[3], chi[3], flo[3][3], fhi[3][3];
    if (!g->inited) return -2;
    if (!(dt > 0.0)) return -1;

    fill_ghosts(g, g->U); /* one boundary update per step */

    /* Steps 2-3: PCM + HLLD on every face that has both neighbour cells and
     * their cell-centred fields */
    for (a = 0; a < 3; a++) {
        for (x = 0; x < 3; x++) { lo[x] = -ng; hi[x] = g->n[x] + ng - 1; }
        lo[a] = -ng + 1;
        sweep_fluxes(g, g->U, a, 0, lo, hi);
    }
    /* Step 4 */
    for (c = 0; c < 3; c++)
        for (x = 0; x < 3; x++) {
            elo[c][x] = (x == c) ? -ng : -ng + 1;
            ehi[c][x] = g->n[x] + ng - 1;
        }
    ct_fields(g, g->U, elo, ehi);
    /* Step 5: half update (G8: dt/2) */
    for (x = 0; x < 3; x++) { clo[x] = -ng + 1; chi[x] = g->n[x] + ng - 2; }
    for (a = 0; a < 3; a++)
        for (x = 0; x < 3; x++) {
            flo[a][x] = -ng + 1;
            fhi[a][x] = (x == a) ? g->n[x] + ng - 1 : g->n[x] + ng - 2;
        }
    update(g, g->U, g->Uh, 0.5 * dt, clo, chi, flo, fhi);

    /* Steps 6-7: high-order states from U^{n+1/2}; prims valid on cells
     * [-ng+1, n+ng-2); a cell is reconstructed if its +-r neighbours are valid */
    for (a = 0; a < 3; a++) {
        for (x = 0; x < 3; x++) { lo[x] = -ng + 1; hi[x] = g->n[x] + ng - 2; }
        lo[a] = -ng + 2 + r; hi[a] = g->n[a] + ng - 2 - r;
        sweep_fluxes(g, g->Uh, a, g->recon, lo, hi);
    }
    /* Step 8 (G12) */
    for (c = 0; c < 3; c++)
        for (x = 0; x < 3; x++) {
            elo[c][x] = (x == c) ? -ng + 1 : -ng + 2 + r;
            ehi[c][x] = (x == c) ? g->n[x] + ng - 2 : g->n[x] + ng - 2 - r;
        }
    ct_fields(g, g->Uh, elo, ehi);
    /* Step 9: full update of the active cells and of faces 0..n (G11) */
    for (x = 0; x < 3; x++) { clo[x] = 0; chi[x] = g->n[x]; }
    for (a = 0; a < 3; a++)
        for (x = 0; x < 3; x++) {
            flo[a][x] = 0;
            fhi[a][x] = (x == a) ? g->n[x] + 1 : g->n[x];
        }
    update(g, g->U, g->U, dt, clo, chi, flo, fhi);
    return 0;
}

/* max over active cells of |sum_a (B_a[upper] - B_a[lower]) / Delta_a| */
int oracle_max_divb(double *out)
{
    int i, j, k, a;
    double m = 0.0;
    if (!G.inited) return -2;
    for (k = 0; k < G.n[2]; k++)
        for (j = 0; j < G.n[1]; j++)
            for (i = 0; i < G.n[0]; i++) {
                long idx = IDX(&G, i, j, k);
                double d = 0.0;
                for (a = 0; a < 3; a++)
                    d += (G.U[5 + a][idx + G.s[a]] - G.U[5 + a][idx]) / G.d[a];
                if (fabs(d) > m) m = fabs(d);
            }
    *out = m;
    return 0;
}

/* ---- small accessors used by the pins ---- */
double oracle_fast_speed(double gamma, double rho, double P, double bn, double bt1, double bt2)
{
    return sqrt(fast_speed_sq(gamma, rho, P, bn, bt1, bt2));
}

void oracle_phys_flux(double gamma, const double W[7], double bx, double F[7])
{
    double b2 = bx * bx + W[5] * W[5] + W[6] * W[6];
    double pT = W[4] + 0.5 * b2;
    double e = W[4] / (gamma - 1.0) + 0.5 * W[0] * (W[1] * W[1] + W[2] * W[2] + W[3] * W[3]) + 0.5 * b2;
    phys_flux(W, bx, e, pT, F);
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}
