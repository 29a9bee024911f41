/* oracle/mhd_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see mhd_oracle.h).
 *
 * One loop nest per stage, full-size scratch arrays, no blocking, no fusion, no
 * reordering beyond what the paper's description states.  Citations are PAPER.md
 * line numbers; "O<n>" are the readings listed in DESIGN.md (section "Readings").
 */
#include "mhd_oracle.h"
#include <float.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>

#define HALF ((real)0.5)
#define QUART ((real)0.25)
#define ZERO ((real)0)

#if defined(ORACLE_IS_FLOAT)
#define R_EPS FLT_EPSILON
#define R_SQRT sqrtf
#define R_FABS fabsf
#else
#define R_EPS DBL_EPSILON
#define R_SQRT sqrt
#define R_FABS fabs
#endif

static real rmin(real a, real b) { return a < b ? a : b; }
static real rmax(real a, real b) { return a > b ? a : b; }

/* ------------------------------------------------------------------ geometry -- */
typedef struct {
  int n[3], g[3], m[3], act[3];
  long s[3]; /* index step for +1 in dimension d; 0 in a collapsed dimension (O0) */
  long M;    /* cells per patch, guards included */
  int np;
  real gamma, dx[3];
  int limiter, emf_solver, flux_solver;
} geom;

static void mkgeom(const orc_desc *d, geom *G) {
  for (int a = 0; a < 3; ++a) {
    G->n[a] = d->n[a];
    G->act[a] = d->n[a] > 1;
    G->g[a] = G->act[a] ? d->ng : 0;
    G->m[a] = d->n[a] + 2 * G->g[a];
    G->dx[a] = (real)d->dx[a];
  }
  G->s[0] = G->act[0] ? 1 : 0;
  G->s[1] = G->act[1] ? G->m[0] : 0;
  G->s[2] = G->act[2] ? (long)G->m[0] * G->m[1] : 0;
  G->M = (long)G->m[0] * G->m[1] * G->m[2];
  G->np = d->npatch;
  G->gamma = (real)d->gamma;
  G->limiter = d->limiter;
  G->emf_solver = d->emf_solver;
  G->flux_solver = d->flux_solver;
}

/* index of the cell with interior-relative coordinates (i,j,k) */
static long cidx(const geom *G, int i, int j, int k) {
  return ((long)(k + G->g[2]) * G->m[1] + (j + G->g[1])) * G->m[0] + (i + G->g[0]);
}

/* a box of cells: [-lo_d, n_d-1+hi_d] in an active dimension, [0,0] in a collapsed one */
typedef struct { int lo[3], hi[3]; } box;
static box mkbox(const geom *G, int ax, int bx, int ay, int by, int az, int bz) {
  int a[3] = {ax, ay, az}, b[3] = {bx, by, bz};
  box B;
  for (int d = 0; d < 3; ++d) {
    B.lo[d] = G->act[d] ? -a[d] : 0;
    B.hi[d] = G->act[d] ? G->n[d] - 1 + b[d] : 0;
  }
  return B;
}
#define BOXLOOP(B)                                   \
  for (int k = (B).lo[2]; k <= (B).hi[2]; ++k)       \
    for (int j = (B).lo[1]; j <= (B).hi[1]; ++j)     \
      for (int i = (B).lo[0]; i <= (B).hi[0]; ++i)

int orc_sizeof_real(void) { return (int)sizeof(real); }

/* threads of the OpenMP build (bench.py's all-cores timing leg); 1 in the plain build */
#ifdef _OPENMP
#include <omp.h>
int orc_threads(int want) { if (want > 0) omp_set_num_threads(want); return omp_get_max_threads(); }
#else
int orc_threads(int want) { (void)want; return 1; }
#endif
int64_t orc_patch_cells(const orc_desc *d) { geom G; mkgeom(d, &G); return G.M; }
int64_t orc_state_elems(const orc_desc *d) { geom G; mkgeom(d, &G); return 8 * (int64_t)G.np * G.M; }

/* ------------------------------------------------------------ O1 guard fill -- */
/* the framework supplies guard data from neighbours; here
 * the same-time, same-resolution copy.  Width 3 from 24^3 -> 30^3 (L212).           */
void orc_fill_guards(const orc_desc *d, const int32_t *nbr, real *U) {
  geom G; mkgeom(d, &G);
  box all = mkbox(&G, G.g[0], G.g[0], G.g[1], G.g[1], G.g[2], G.g[2]);
  /* patches only read each other's INTERIOR cells here, so they are independent: the pragma is
   * inert unless the file is built with -fopenmp (bench.py's all-cores timing leg only)        */
#pragma omp parallel for schedule(dynamic)
  for (int p = 0; p < G.np; ++p) {
    BOXLOOP(all) {
      int c[3] = {i, j, k}, o[3], src[3], clamp[3];
      int guard = 0;
      for (int a = 0; a < 3; ++a) {
        o[a] = c[a] < 0 ? -1 : (c[a] >= G.n[a] ? 1 : 0);
        if (o[a]) guard = 1;
        src[a] = c[a] - o[a] * G.n[a];
        clamp[a] = c[a] < 0 ? 0 : (c[a] >= G.n[a] ? G.n[a] - 1 : c[a]);
      }
      if (!guard) continue;
      int q = nbr[p * 27 + (o[2] + 1) * 9 + (o[1] + 1) * 3 + (o[0] + 1)];
      long dst = cidx(&G, i, j, k);
      for (int f = 0; f < 8; ++f) {
        real *Uf = U + (long)f * G.np * G.M;
        if (q >= 0) {
          Uf[(long)p * G.M + dst] = Uf[(long)q * G.M + cidx(&G, src[0], src[1], src[2])];
        } else {
          /* zero-gradient; the closing face (normal face field at index n, other two
           * indices interior) holds an evolved value (O8) and is left untouched      */
          if (f >= 5) {
            int a = f - 5, b = (a + 1) % 3, e = (a + 2) % 3;
            if (c[a] == G.n[a] && G.act[a] && o[b] == 0 && o[e] == 0) continue;
          }
          Uf[(long)p * G.M + dst] = Uf[(long)p * G.M + cidx(&G, clamp[0], clamp[1], clamp[2])];
        }
      }
    }
  }
}

/* ---------------------------------------------------------------- pointwise -- */
/* O3 limiter ("choice of slope estimate is crucial", unnamed).     */
real orc_limiter(int32_t kind, real a, real b) {
  if (a * b <= ZERO) return ZERO;
  real sa = a > ZERO ? (real)1 : (real)-1;
  real fa = R_FABS(a), fb = R_FABS(b);
  if (kind == 2) { /* monotonised central */
    real m = rmin((real)2 * fa, (real)2 * fb);
    return sa * rmin(m, HALF * R_FABS(a + b));
  }
  return sa * rmin(fa, fb); /* minmod */
}

/* fast magnetosonic speed along the normal (O6) */
real orc_fast_speed(double gamma, real rho, real p, real bn, real bt1, real bt2) {
  real gp = (real)gamma * p;
  real b2 = bn * bn + bt1 * bt1 + bt2 * bt2;
  real s = gp + b2;
  real disc = s * s - (real)4 * gp * bn * bn;
  if (disc < ZERO) disc = ZERO;
  return R_SQRT((s + R_SQRT(disc)) / ((real)2 * rho));
}

/* O6  HLLD (Miyoshi & Kusano 2005, cited PAPER.md L76; six regions, Fig. 1).
 * L, R = (rho, u, v, w, p, By, Bz) with u the normal velocity; bn the common normal
 * field.  F = fluxes of (rho, rho u, rho v, rho w, E, By, Bz); Eq. 6 (L66) is the
 * physical flux.                                                                    */
static void phys_flux(real gamma, const real q[7], real bn, real U[7], real F[7], real *pT_out) {
  real rho = q[0], u = q[1], v = q[2], w = q[3], p = q[4], by = q[5], bz = q[6];
  real b2 = bn * bn + by * by + bz * bz;
  real pT = p + HALF * b2;
  real E = p / (gamma - (real)1) + HALF * rho * (u * u + v * v + w * w) + HALF * b2;
  real ub = u * bn + v * by + w * bz;
  U[0] = rho; U[1] = rho * u; U[2] = rho * v; U[3] = rho * w; U[4] = E; U[5] = by; U[6] = bz;
  F[0] = rho * u;
  F[1] = rho * u * u + pT - bn * bn;
  F[2] = rho * v * u - by * bn;
  F[3] = rho * w * u - bz * bn;
  F[4] = u * (E + pT) - bn * ub;
  F[5] = by * u - bn * v;
  F[6] = bz * u - bn * w;
  *pT_out = pT;
}

void orc_hlld(double gamma_, const real L[7], const real R[7], real bn, real F[7]) {
  real gamma = (real)gamma_;
  real UL[7], UR[7], FL[7], FR[7], pTL, pTR;
  phys_flux(gamma, L, bn, UL, FL, &pTL);
  phys_flux(gamma, R, bn, UR, FR, &pTR);
  real rhoL = L[0], uL = L[1], vL = L[2], wL = L[3], byL = L[5], bzL = L[6];
  real rhoR = R[0], uR = R[1], vR = R[2], wR = R[3], byR = R[5], bzR = R[6];
  real cfL = orc_fast_speed(gamma_, rhoL, L[4], bn, byL, bzL);
  real cfR = orc_fast_speed(gamma_, rhoR, R[4], bn, byR, bzR);
  real cmax = rmax(cfL, cfR);
  real SL = rmin(uL, uR) - cmax;
  real SR = rmax(uL, uR) + cmax;

  real sdL = SL - uL, sdR = SR - uR;
  real SM = (sdR * rhoR * uR - sdL * rhoL * uL - pTR + pTL) / (sdR * rhoR - sdL * rhoL);
  real pTs = pTL + rhoL * sdL * (SM - uL);

  /* star states */
  real UsL[7], UsR[7];
  real vsL, wsL, bysL, bzsL, vsR, wsR, bysR, bzsR, rhosL, rhosR;
  {
    rhosL = rhoL * sdL / (SL - SM);
    real D = rhoL * sdL * (SL - SM) - bn * bn;
    real ref = rhoL * sdL * sdL;
    if (R_FABS(D) <= (real)16 * R_EPS * ref) {
      vsL = vL; wsL = wL; bysL = byL; bzsL = bzL;
    } else {
      vsL = vL - bn * byL * (SM - uL) / D;
      wsL = wL - bn * bzL * (SM - uL) / D;
      bysL = byL * (ref - bn * bn) / D;
      bzsL = bzL * (ref - bn * bn) / D;
    }
    real ubL = uL * bn + vL * byL + wL * bzL;
    real ubs = SM * bn + vsL * bysL + wsL * bzsL;
    real EsL = (sdL * UL[4] - pTL * uL + pTs * SM + bn * (ubL - ubs)) / (SL - SM);
    UsL[0] = rhosL; UsL[1] = rhosL * SM; UsL[2] = rhosL * vsL; UsL[3] = rhosL * wsL;
    UsL[4] = EsL; UsL[5] = bysL; UsL[6] = bzsL;
  }
  {
    rhosR = rhoR * sdR / (SR - SM);
    real D = rhoR * sdR * (SR - SM) - bn * bn;
    real ref = rhoR * sdR * sdR;
    if (R_FABS(D) <= (real)16 * R_EPS * ref) {
      vsR = vR; wsR = wR; bysR = byR; bzsR = bzR;
    } else {
      vsR = vR - bn * byR * (SM - uR) / D;
      wsR = wR - bn * bzR * (SM - uR) / D;
      bysR = byR * (ref - bn * bn) / D;
      bzsR = bzR * (ref - bn * bn) / D;
    }
    real ubR = uR * bn + vR * byR + wR * bzR;
    real ubs = SM * bn + vsR * bysR + wsR * bzsR;
    real EsR = (sdR * UR[4] - pTR * uR + pTs * SM + bn * (ubR - ubs)) / (SR - SM);
    UsR[0] = rhosR; UsR[1] = rhosR * SM; UsR[2] = rhosR * vsR; UsR[3] = rhosR * wsR;
    UsR[4] = EsR; UsR[5] = bysR; UsR[6] = bzsR;
  }

  /* Alfven waves and double-star states */
  real rL = R_SQRT(rhosL), rR = R_SQRT(rhosR);
  real absbn = R_FABS(bn);
  real SsL = SM - absbn / rL, SsR = SM + absbn / rR;
  real sg = bn > ZERO ? (real)1 : (bn < ZERO ? (real)-1 : ZERO);
  real rsum = rL + rR;
  real vss = (rL * vsL + rR * vsR + (bysR - bysL) * sg) / rsum;
  real wss = (rL * wsL + rR * wsR + (bzsR - bzsL) * sg) / rsum;
  real byss = (rL * bysR + rR * bysL + rL * rR * (vsR - vsL) * sg) / rsum;
  real bzss = (rL * bzsR + rR * bzsL + rL * rR * (wsR - wsL) * sg) / rsum;
  real ubss = SM * bn + vss * byss + wss * bzss;
  real ubsL = SM * bn + vsL * bysL + wsL * bzsL;
  real ubsR = SM * bn + vsR * bysR + wsR * bzsR;
  real UssL[7], UssR[7];
  UssL[0] = rhosL; UssL[1] = rhosL * SM; UssL[2] = rhosL * vss; UssL[3] = rhosL * wss;
  UssL[4] = UsL[4] - rL * (ubsL - ubss) * sg; UssL[5] = byss; UssL[6] = bzss;
  UssR[0] = rhosR; UssR[1] = rhosR * SM; UssR[2] = rhosR * vss; UssR[3] = rhosR * wss;
  UssR[4] = UsR[4] + rR * (ubsR - ubss) * sg; UssR[5] = byss; UssR[6] = bzss;

  /* flux by region, evaluated in exactly this order (O6) */
  for (int f = 0; f < 7; ++f) {
    real FsL = FL[f] + SL * (UsL[f] - UL[f]);
    real FsR = FR[f] + SR * (UsR[f] - UR[f]);
    if (SL > ZERO)        F[f] = FL[f];
    else if (SsL > ZERO)  F[f] = FsL;
    else if (SM >= ZERO)  F[f] = FsL + SsL * (UssL[f] - UsL[f]);
    else if (SsR >= ZERO) F[f] = FsR + SsR * (UssR[f] - UsR[f]);
    else if (SR >= ZERO)  F[f] = FsR;
    else                  F[f] = FR[f];
  }
}

/* HLL (section 2.1.1; Harten, Lax & van Leer 1983): three regions, the
 * star state is the integral average of the solution between the two outer waves,
 *     U* = (SR UR - SL UL - (FR - FL)) / (SR - SL),
 * and the flux through x = 0 follows from the jump condition across either outer wave,
 *     F* = FL + SL (U* - UL)   [ = FR + SR (U* - UR) ].
 * Outer speeds as in O6.  Same argument and flux layout as orc_hlld.                    */
void orc_hll(double gamma_, const real L[7], const real R[7], real bn, real F[7]) {
  real gamma = (real)gamma_;
  real UL[7], UR[7], FL[7], FR[7], pTL, pTR;
  phys_flux(gamma, L, bn, UL, FL, &pTL);
  phys_flux(gamma, R, bn, UR, FR, &pTR);
  real cfL = orc_fast_speed(gamma_, L[0], L[4], bn, L[5], L[6]);
  real cfR = orc_fast_speed(gamma_, R[0], R[4], bn, R[5], R[6]);
  real cmax = rmax(cfL, cfR);
  real SL = rmin(L[1], R[1]) - cmax;
  real SR = rmax(L[1], R[1]) + cmax;
  for (int f = 0; f < 7; ++f) {
    if (SL > ZERO) F[f] = FL[f];
    else if (SR >= ZERO) {
      real Us = (SR * UR[f] - SL * UL[f] - (FR[f] - FL[f])) / (SR - SL);
      F[f] = FL[f] + SL * (Us - UL[f]);
    } else F[f] = FR[f];
  }
}

/* O7  two-dimensional Riemann problem at a cell edge (Fig. 3
 * L148).  The paper names the solver and prints no formula: DESIGN.md reading O7.
 * Corners c: 0 SW, 1 SE, 2 NW, 3 NE; each (rho, ua, ub, ue, p, Be).  In-plane fields
 * are single-valued on the four sides: A (component a) south/north, B (component b)
 * west/east.  Returns the edge EMF  ua*B - ub*A  (sign of Eq. 7).               */
typedef struct { real SM, rsL, rsR, btsL, btsR, lo, hi; } sub1d;

/* star quantities of a 1D sub-problem with prescribed outer speeds SL, SR */
static sub1d substar(real rhoL, real unL, real pTL, real btL,
                     real rhoR, real unR, real pTR, real btR, real bn, real SL, real SR) {
  sub1d s;
  real sdL = SL - unL, sdR = SR - unR;
  s.SM = (sdR * rhoR * unR - sdL * rhoL * unL - pTR + pTL) / (sdR * rhoR - sdL * rhoL);
  s.rsL = rhoL * sdL / (SL - s.SM);
  s.rsR = rhoR * sdR / (SR - s.SM);
  real DL = rhoL * sdL * (SL - s.SM) - bn * bn, refL = rhoL * sdL * sdL;
  real DR = rhoR * sdR * (SR - s.SM) - bn * bn, refR = rhoR * sdR * sdR;
  s.btsL = (R_FABS(DL) <= (real)16 * R_EPS * refL) ? btL : btL * (refL - bn * bn) / DL;
  s.btsR = (R_FABS(DR) <= (real)16 * R_EPS * refR) ? btR : btR * (refR - bn * bn) / DR;
  s.lo = s.SM - R_FABS(bn) / R_SQRT(s.rsL);
  s.hi = s.SM + R_FABS(bn) / R_SQRT(s.rsR);
  return s;
}

real orc_emf2d(double gamma_, int32_t solver, const real c[4][6],
               real AS, real AN, real BW, real BE) {
  enum { SW = 0, SE = 1, NW = 2, NE = 3 };
  real A[4] = {AS, AS, AN, AN}, B[4] = {BW, BE, BW, BE};
  real e[4], cfa[4], cfb[4], pT[4];
  for (int q = 0; q < 4; ++q) {
    real rho = c[q][0], ua = c[q][1], ub = c[q][2], p = c[q][4], be = c[q][5];
    e[q] = ua * B[q] - ub * A[q];
    cfa[q] = orc_fast_speed(gamma_, rho, p, A[q], B[q], be);
    cfb[q] = orc_fast_speed(gamma_, rho, p, B[q], A[q], be);
    pT[q] = p + HALF * (A[q] * A[q] + B[q] * B[q] + be * be);
  }
  /* step 1: raw outer speeds from all four corners */
  real uamin = rmin(rmin(c[0][1], c[1][1]), rmin(c[2][1], c[3][1]));
  real uamax = rmax(rmax(c[0][1], c[1][1]), rmax(c[2][1], c[3][1]));
  real ubmin = rmin(rmin(c[0][2], c[1][2]), rmin(c[2][2], c[3][2]));
  real ubmax = rmax(rmax(c[0][2], c[1][2]), rmax(c[2][2], c[3][2]));
  real camax = rmax(rmax(cfa[0], cfa[1]), rmax(cfa[2], cfa[3]));
  real cbmax = rmax(rmax(cfb[0], cfb[1]), rmax(cfb[2], cfb[3]));
  real tW = uamin - camax, tE = uamax + camax, tS = ubmin - cbmax, tN = ubmax + cbmax;

  real SWs, SEs, SSs, SNs;       /* speeds used in the composition (dagger)          */
  real es[4], BsW, BsE, AsS, AsN; /* values used in the composition                   */
  if (solver == 1) {
    /* HLL-2D: corner values themselves, fast speeds clipped at zero */
    SWs = rmin(ZERO, tW); SEs = rmax(ZERO, tE); SSs = rmin(ZERO, tS); SNs = rmax(ZERO, tN);
    for (int q = 0; q < 4; ++q) es[q] = e[q];
    BsW = BW; BsE = BE; AsS = AS; AsN = AN;
  } else {
    /* step 2: four 1D sub-problems sharing the outer speeds */
    sub1d xS = substar(c[SW][0], c[SW][1], pT[SW], BW, c[SE][0], c[SE][1], pT[SE], BE, AS, tW, tE);
    sub1d xN = substar(c[NW][0], c[NW][1], pT[NW], BW, c[NE][0], c[NE][1], pT[NE], BE, AN, tW, tE);
    sub1d yW = substar(c[SW][0], c[SW][2], pT[SW], AS, c[NW][0], c[NW][2], pT[NW], AN, BW, tS, tN);
    sub1d yE = substar(c[SE][0], c[SE][2], pT[SE], AS, c[NE][0], c[NE][2], pT[NE], AN, BE, tS, tN);
    /* step 3: inner (Alfven-type) speeds; not clamped to the outer ones */
    SWs = tW >= ZERO ? ZERO : rmin(ZERO, rmin(xS.lo, xN.lo));
    SEs = tE <= ZERO ? ZERO : rmax(ZERO, rmax(xS.hi, xN.hi));
    SSs = tS >= ZERO ? ZERO : rmin(ZERO, rmin(yW.lo, yE.lo));
    SNs = tN <= ZERO ? ZERO : rmax(ZERO, rmax(yW.hi, yE.hi));
    /* step 4: corner star EMFs from the jump conditions across the outer waves */
    real Bs[4] = {xS.btsL, xS.btsR, xN.btsL, xN.btsR};
    real As[4] = {yW.btsL, yE.btsL, yW.btsR, yE.btsR};
    real SxW = rmin(tW, ZERO), SxE = rmax(tE, ZERO), SyS = rmin(tS, ZERO), SyN = rmax(tN, ZERO);
    real Sx[4] = {SxW, SxE, SxW, SxE}, Sy[4] = {SyS, SyS, SyN, SyN};
    for (int q = 0; q < 4; ++q)
      es[q] = e[q] + Sx[q] * (Bs[q] - B[q]) - Sy[q] * (As[q] - A[q]);
    /* step 5: edge-side star fields, weighted like (dagger) -- needs the weights */
    real dy = SNs - SSs, dxs = SEs - SWs;
    real bN = dy == ZERO ? HALF : SNs / dy, bS = dy == ZERO ? HALF : -SSs / dy;
    real aE = dxs == ZERO ? HALF : SEs / dxs, aW = dxs == ZERO ? HALF : -SWs / dxs;
    BsW = bN * Bs[SW] + bS * Bs[NW];
    BsE = bN * Bs[SE] + bS * Bs[NE];
    AsS = aE * As[SW] + aW * As[SE];
    AsN = aE * As[NW] + aW * As[NE];
  }
  /* step 6: the two-dimensional HLL composition (dagger) */
  real dxs = SEs - SWs, dy = SNs - SSs;
  real aE = dxs == ZERO ? HALF : SEs / dxs, aW = dxs == ZERO ? HALF : -SWs / dxs;
  real bN = dy == ZERO ? HALF : SNs / dy, bS = dy == ZERO ? HALF : -SSs / dy;
  real dissx = dxs == ZERO ? ZERO : SWs * SEs / dxs;
  real dissy = dy == ZERO ? ZERO : SSs * SNs / dy;
  return aE * bN * es[SW] + aW * bN * es[SE] + aE * bS * es[NW] + aW * bS * es[NE]
       + dissx * (BsE - BsW) - dissy * (AsN - AsS);
}

/* ------------------------------------------------------------------- stages -- */
typedef struct {
  real *q[8];       /* O2 primitives rho,u,v,w,p,Bcx,Bcy,Bcz                         */
  real *dq[3][8];   /* O3 limited undivided slopes per direction                     */
  real *dbf[6];     /* O3 face-field transverse slopes: dy bx, dz bx, dx by, dz by,
                       dx bz, dy bz                                                  */
  real *e0[3];      /* O4a edge EMFs at time n: ex, ey, ez                           */
  real *bh[3];      /* O4b half-step face fields                                     */
  real *qh[8];      /* O4c half-step primitives (Bc^h = mean of bh faces)            */
  real *flux[3][5]; /* O6 fluxes of rho, mx, my, mz, E through lower faces           */
  real *emf[3];     /* O7 edge EMFs at n+1/2: ex, ey, ez                             */
  real *base;
} scratch;

static void scratch_bind(scratch *S, real *base, long M) {
  real *p = base;
  S->base = base;
  for (int f = 0; f < 8; ++f) { S->q[f] = p; p += M; }
  for (int d = 0; d < 3; ++d) for (int f = 0; f < 8; ++f) { S->dq[d][f] = p; p += M; }
  for (int f = 0; f < 6; ++f) { S->dbf[f] = p; p += M; }
  for (int f = 0; f < 3; ++f) { S->e0[f] = p; p += M; }
  for (int f = 0; f < 3; ++f) { S->bh[f] = p; p += M; }
  for (int f = 0; f < 8; ++f) { S->qh[f] = p; p += M; }
  for (int d = 0; d < 3; ++d) for (int f = 0; f < 5; ++f) { S->flux[d][f] = p; p += M; }
  for (int f = 0; f < 3; ++f) { S->emf[f] = p; p += M; }
}

/* index into dbf: slope of face field b_a along transverse direction t */
static int dbf_index(int a, int t) {
  /* a=0: t=1->0, t=2->1; a=1: t=0->2, t=2->3; a=2: t=0->4, t=1->5 */
  static const int tab[3][3] = {{-1, 0, 1}, {2, -1, 3}, {4, 5, -1}};
  return tab[a][t];
}

/* run stages O2..O7 for patch p; Up[f] points at the patch's field f (guards filled) */
static void run_stages(const geom *G, const real *const Up[8], real dt, scratch *S) {
  const long sx = G->s[0], sy = G->s[1], sz = G->s[2];
  const long *s = G->s;
  memset(S->base, 0, sizeof(real) * ORC_NSTAGE * G->M);

  /* O2 primitives on cells [-2, n+1] (EOS L68) */
  {
    box B = mkbox(G, 2, 2, 2, 2, 2, 2);
    BOXLOOP(B) {
      long c = cidx(G, i, j, k);
      real rho = Up[0][c];
      real u = Up[1][c] / rho, v = Up[2][c] / rho, w = Up[3][c] / rho;
      real bcx = HALF * (Up[5][c] + Up[5][c + sx]);
      real bcy = HALF * (Up[6][c] + Up[6][c + sy]);
      real bcz = HALF * (Up[7][c] + Up[7][c + sz]);
      real p = (G->gamma - (real)1) *
               (Up[4][c] - HALF * rho * (u * u + v * v + w * w) - HALF * (bcx * bcx + bcy * bcy + bcz * bcz));
      S->q[0][c] = rho; S->q[1][c] = u; S->q[2][c] = v; S->q[3][c] = w; S->q[4][c] = p;
      S->q[5][c] = bcx; S->q[6][c] = bcy; S->q[7][c] = bcz;
    }
  }
  /* O3 slopes on cells [-1, n] */
  {
    box B = mkbox(G, 1, 1, 1, 1, 1, 1);
    BOXLOOP(B) {
      long c = cidx(G, i, j, k);
      for (int d = 0; d < 3; ++d) {
        if (!G->act[d]) continue;
        for (int f = 0; f < 8; ++f) {
          if (f == 5 + d) continue; /* the normal component has no limited slope */
          S->dq[d][f][c] = orc_limiter(G->limiter, S->q[f][c] - S->q[f][c - s[d]],
                                       S->q[f][c + s[d]] - S->q[f][c]);
        }
      }
      for (int a = 0; a < 3; ++a)
        for (int t = 0; t < 3; ++t) {
          if (t == a || !G->act[t]) continue;
          const real *b = Up[5 + a];
          S->dbf[dbf_index(a, t)][c] = orc_limiter(G->limiter, b[c] - b[c - s[t]], b[c + s[t]] - b[c]);
        }
    }
  }
  /* O4a edge EMFs at time n on edges [-1, n+1]: Eq. 7-11 and their
   * cyclic images */
  {
    box B = mkbox(G, 1, 2, 1, 2, 1, 2);
    const real *u = S->q[1], *v = S->q[2], *w = S->q[3];
    const real *bx = Up[5], *by = Up[6], *bz = Up[7];
    BOXLOOP(B) {
      long c = cidx(G, i, j, k);
      { /* ez at (x_{i-1/2}, y_{j-1/2}, z_k) */
        real ub = QUART * (u[c] + u[c - sy] + u[c - sx] + u[c - sx - sy]);   /* Eq. 8  */
        real vb = QUART * (v[c] + v[c - sy] + v[c - sx] + v[c - sx - sy]);   /* Eq. 9  */
        real bxb = HALF * (bx[c] + bx[c - sy]);                               /* Eq. 10 */
        real byb = HALF * (by[c] + by[c - sx]);                               /* Eq. 11 */
        S->e0[2][c] = ub * byb - vb * bxb;                                    /* Eq. 7  */
      }
      { /* ex at (x_i, y_{j-1/2}, z_{k-1/2}) */
        real vb = QUART * (v[c] + v[c - sz] + v[c - sy] + v[c - sy - sz]);
        real wb = QUART * (w[c] + w[c - sz] + w[c - sy] + w[c - sy - sz]);
        real byb = HALF * (by[c] + by[c - sz]);
        real bzb = HALF * (bz[c] + bz[c - sy]);
        S->e0[0][c] = vb * bzb - wb * byb;
      }
      { /* ey at (x_{i-1/2}, y_j, z_{k-1/2}) */
        real wb = QUART * (w[c] + w[c - sx] + w[c - sz] + w[c - sz - sx]);
        real ub = QUART * (u[c] + u[c - sx] + u[c - sz] + u[c - sz - sx]);
        real bzb = HALF * (bz[c] + bz[c - sx]);
        real bxb = HALF * (bx[c] + bx[c - sz]);
        S->e0[1][c] = wb * bxb - ub * bzb;
      }
    }
  }
  /* O4b half-step face fields: Eq. 12 with dt/2, faces [-1, n+1] in
   * the normal index, [-1, n] transversally */
  {
    const real hdt = HALF * dt;
    const real *ex = S->e0[0], *ey = S->e0[1], *ez = S->e0[2];
    box Bx = mkbox(G, 1, 2, 1, 1, 1, 1), By = mkbox(G, 1, 1, 1, 2, 1, 1), Bz = mkbox(G, 1, 1, 1, 1, 1, 2);
    BOXLOOP(Bx) {
      long c = cidx(G, i, j, k);
      S->bh[0][c] = Up[5][c] + hdt * ((ez[c + sy] - ez[c]) / G->dx[1] - (ey[c + sz] - ey[c]) / G->dx[2]);
    }
    BOXLOOP(By) {
      long c = cidx(G, i, j, k);
      S->bh[1][c] = Up[6][c] + hdt * ((ex[c + sz] - ex[c]) / G->dx[2] - (ez[c + sx] - ez[c]) / G->dx[0]);
    }
    BOXLOOP(Bz) {
      long c = cidx(G, i, j, k);
      S->bh[2][c] = Up[7][c] + hdt * ((ey[c + sx] - ey[c]) / G->dx[0] - (ex[c + sy] - ex[c]) / G->dx[1]);
    }
  }
  /* O4c hydro half step on cells [-1, n]: forward Euler in primitive variables
   * (PAPER.md L114), Eq. 1-4 in primitive form */
  {
    box B = mkbox(G, 1, 1, 1, 1, 1, 1);
    real lam[3];
    for (int d = 0; d < 3; ++d) lam[d] = G->act[d] ? HALF * dt / G->dx[d] : ZERO;
    BOXLOOP(B) {
      long c = cidx(G, i, j, k);
      real rho = S->q[0][c], vel[3] = {S->q[1][c], S->q[2][c], S->q[3][c]}, p = S->q[4][c];
      real bc[3] = {S->q[5][c], S->q[6][c], S->q[7][c]};
      real rho_h = rho, p_h = p, vel_h[3] = {vel[0], vel[1], vel[2]};
      for (int d = 0; d < 3; ++d) {
        real du_d = S->dq[d][1 + d][c]; /* slope of the velocity component along d */
        rho_h -= lam[d] * (vel[d] * S->dq[d][0][c] + rho * du_d);
        p_h -= lam[d] * (vel[d] * S->dq[d][4][c] + G->gamma * p * du_d);
        for (int a = 0; a < 3; ++a) vel_h[a] -= lam[d] * vel[d] * S->dq[d][1 + a][c];
      }
      for (int a = 0; a < 3; ++a) {
        int b = (a + 1) % 3, e = (a + 2) % 3;
        /* -(1/rho) d_a (p + Bb^2/2 + Be^2/2) + (1/rho)(Bb d_b Ba + Be d_e Ba) */
        vel_h[a] -= lam[a] * (S->dq[a][4][c] + bc[b] * S->dq[a][5 + b][c] + bc[e] * S->dq[a][5 + e][c]) / rho;
        vel_h[a] += (lam[b] * bc[b] * S->dq[b][5 + a][c] + lam[e] * bc[e] * S->dq[e][5 + a][c]) / rho;
      }
      S->qh[0][c] = rho_h; S->qh[1][c] = vel_h[0]; S->qh[2][c] = vel_h[1]; S->qh[3][c] = vel_h[2];
      S->qh[4][c] = p_h;
      for (int a = 0; a < 3; ++a) S->qh[5 + a][c] = HALF * (S->bh[a][c] + S->bh[a][c + s[a]]);
    }
  }
  /* O5 + O6: interface states and HLLD fluxes at faces [0, n] of each active direction
   * */
  for (int d = 0; d < 3; ++d) {
    if (!G->act[d]) continue;
    int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
    int ext[3] = {0, 0, 0};
    ext[d] = 1;
    box B = mkbox(G, 0, ext[0], 0, ext[1], 0, ext[2]);
    BOXLOOP(B) {
      long c = cidx(G, i, j, k), cl = c - s[d];
      int comp[7] = {0, 1 + d, 1 + t1, 1 + t2, 4, 5 + t1, 5 + t2};
      real L[7], R[7], F[7];
      for (int f = 0; f < 7; ++f) {
        L[f] = S->qh[comp[f]][cl] + HALF * S->dq[d][comp[f]][cl];
        R[f] = S->qh[comp[f]][c] - HALF * S->dq[d][comp[f]][c];
      }
      if (G->flux_solver == 1) orc_hll((double)G->gamma, L, R, S->bh[d][c], F);
      else orc_hlld((double)G->gamma, L, R, S->bh[d][c], F);
      S->flux[d][0][c] = F[0];
      S->flux[d][1 + d][c] = F[1];
      S->flux[d][1 + t1][c] = F[2];
      S->flux[d][1 + t2][c] = F[3];
      S->flux[d][4][c] = F[4];
    }
  }
  /* O5 + O7: corner states and the 2D Riemann problem at edges (PAPER.md L104-106,
   * Fig. 3).  Edge direction e, in-plane directions a=(e+1)%3, b=(e+2)%3.       */
  for (int e = 0; e < 3; ++e) {
    int a = (e + 1) % 3, b = (e + 2) % 3;
    int ext[3] = {0, 0, 0};
    ext[a] = 1; ext[b] = 1;
    box B = mkbox(G, 0, ext[0], 0, ext[1], 0, ext[2]);
    int comp[6] = {0, 1 + a, 1 + b, 1 + e, 4, 5 + e};
    const real *dba = S->dbf[dbf_index(a, b)]; /* slope of b_a along b (0 if b collapsed) */
    const real *dbb = S->dbf[dbf_index(b, a)]; /* slope of b_b along a                    */
    BOXLOOP(B) {
      long c = cidx(G, i, j, k);
      /* SW = RT of cell (a-1,b-1), SE = LT of (a,b-1), NW = RB of (a-1,b), NE = LB of (a,b) */
      long cc[4] = {c - s[a] - s[b], c - s[b], c - s[a], c};
      real sga[4] = {1, -1, 1, -1}, sgb[4] = {1, 1, -1, -1};
      real cs[4][6];
      for (int q = 0; q < 4; ++q)
        for (int f = 0; f < 6; ++f)
          cs[q][f] = S->qh[comp[f]][cc[q]] + sga[q] * HALF * S->dq[a][comp[f]][cc[q]]
                                           + sgb[q] * HALF * S->dq[b][comp[f]][cc[q]];
      real AS = S->bh[a][c - s[b]] + HALF * dba[c - s[b]];
      real AN = S->bh[a][c] - HALF * dba[c];
      real BW = S->bh[b][c - s[a]] + HALF * dbb[c - s[a]];
      real BE = S->bh[b][c] - HALF * dbb[c];
      S->emf[e][c] = orc_emf2d((double)G->gamma, G->emf_solver, (const real(*)[6])cs, AS, AN, BW, BE);
    }
  }
}

/* O8 conservative update + constrained transport (Eq. 12 L100 with the
 * metric factor of each term, L154) */
static void update_patch(const geom *G, const real *const Up[8], real *const Un[8], real dt,
                         const scratch *S) {
  const long *s = G->s;
  box I = mkbox(G, 0, 0, 0, 0, 0, 0);
  BOXLOOP(I) {
    long c = cidx(G, i, j, k);
    for (int f = 0; f < 5; ++f) {
      real v = Up[f][c];
      for (int d = 0; d < 3; ++d) {
        if (!G->act[d]) continue;
        v -= dt * (S->flux[d][f][c + s[d]] - S->flux[d][f][c]) / G->dx[d];
      }
      Un[f][c] = v;
    }
  }
  for (int a = 0; a < 3; ++a) {
    int b = (a + 1) % 3, e = (a + 2) % 3;
    int ext[3] = {0, 0, 0};
    ext[a] = 1; /* faces 0..n: the closing face n lives in the first high guard slot */
    box B = mkbox(G, 0, ext[0], 0, ext[1], 0, ext[2]);
    BOXLOOP(B) {
      long c = cidx(G, i, j, k);
      /* d b_a/dt = d_b E_e - d_e E_b */
      Un[5 + a][c] = Up[5 + a][c] + dt * ((S->emf[e][c + s[b]] - S->emf[e][c]) / G->dx[b]
                                        - (S->emf[b][c + s[e]] - S->emf[b][c]) / G->dx[e]);
    }
  }
}

void orc_step(const orc_desc *d, const real *U, real *Unew, double dt) {
  geom G; mkgeom(d, &G);
  memcpy(Unew, U, sizeof(real) * 8 * (size_t)G.np * G.M);
  /* patches are independent between guard fills; each gets its own scratch */
#pragma omp parallel for schedule(dynamic)
  for (int p = 0; p < G.np; ++p) {
    real *buf = (real *)malloc(sizeof(real) * ORC_NSTAGE * G.M);
    scratch S; scratch_bind(&S, buf, G.M);
    const real *Up[8]; real *Un[8];
    for (int f = 0; f < 8; ++f) {
      Up[f] = U + ((long)f * G.np + p) * G.M;
      Un[f] = Unew + ((long)f * G.np + p) * G.M;
    }
    run_stages(&G, Up, (real)dt, &S);
    update_patch(&G, Up, Un, (real)dt, &S);
    free(buf);
  }
}

void orc_stages(const orc_desc *d, const real *U, int32_t patch, double dt, real *out) {
  geom G; mkgeom(d, &G);
  scratch S; scratch_bind(&S, out, G.M);
  const real *Up[8];
  for (int f = 0; f < 8; ++f) Up[f] = U + ((long)f * G.np + patch) * G.M;
  run_stages(&G, Up, (real)dt, &S);
}

/* O9 CFL (each patch carries a time step; formula: DESIGN.md O9) */
double orc_cfl_dt(const orc_desc *d, const real *U, double courant, double *per_patch) {
  geom G; mkgeom(d, &G);
  box I = mkbox(&G, 0, 0, 0, 0, 0, 0);
  double dtmin = INFINITY;
  double *dts = (double *)malloc(sizeof(double) * (size_t)G.np);
#pragma omp parallel for schedule(dynamic)
  for (int p = 0; p < G.np; ++p) {
    const real *Up[8];
    for (int f = 0; f < 8; ++f) Up[f] = U + ((long)f * G.np + p) * G.M;
    real rate_max = ZERO;
    BOXLOOP(I) {
      long c = cidx(&G, i, j, k);
      real rho = Up[0][c];
      real vel[3] = {Up[1][c] / rho, Up[2][c] / rho, Up[3][c] / rho};
      real bc[3];
      for (int a = 0; a < 3; ++a) bc[a] = HALF * (Up[5 + a][c] + Up[5 + a][c + G.s[a]]);
      real p_ = (G.gamma - (real)1) * (Up[4][c] - HALF * rho * (vel[0] * vel[0] + vel[1] * vel[1] + vel[2] * vel[2])
                                       - HALF * (bc[0] * bc[0] + bc[1] * bc[1] + bc[2] * bc[2]));
      real rate = ZERO;
      for (int a = 0; a < 3; ++a) {
        if (!G.act[a]) continue;
        real cf = orc_fast_speed(d->gamma, rho, p_, bc[a], bc[(a + 1) % 3], bc[(a + 2) % 3]);
        rate += (R_FABS(vel[a]) + cf) / G.dx[a];
      }
      if (!(rate <= rate_max)) rate_max = rate; /* NaN propagates into the maximum */
    }
    dts[p] = courant / (double)rate_max;
  }
  for (int p = 0; p < G.np; ++p) {
    if (per_patch) per_patch[p] = dts[p];
    if (!(dts[p] >= dtmin)) dtmin = dts[p];
  }
  free(dts);
  return dtmin;
}


/* ------------------------------------------------- O10 local time steps -- */
/* PAPER.md L122 (section 2.2): a patch holds several time slices and its own time and time
 * step; L188, L200 (section 3.1): neighbouring patches sit at different times and ghost-zone
 * values are interpolated.  Reading O10: two slices per patch, S[cur[p]] the newer
 * one at time t_new[p], the other the older one at t_old[p]; guard values of a patch p are
 * its neighbours' slices interpolated LINEARLY IN TIME to t_new[p].                          */
static int times_equal(double a, double b) {
  double s = fabs(a) > fabs(b) ? fabs(a) : fabs(b);
  return fabs(a - b) <= 1e-12 * (s > 1.0 ? s : 1.0);
}

int orc_local_ready(const orc_desc *d, const int32_t *nbr, const double *t_old, const double *t_new,
                    const int32_t *list, int32_t n) {
  for (int i = 0; i < n; ++i) {
    int p = list[i];
    if (p < 0 || p >= d->npatch) return 0;
    for (int c = 0; c < 27; ++c) {
      int q = nbr[p * 27 + c];
      if (q < 0 || q == p) continue;
      int lo_ok = t_old[q] <= t_new[p] || times_equal(t_old[q], t_new[p]);
      int hi_ok = t_new[p] <= t_new[q] || times_equal(t_new[p], t_new[q]);
      if (!(lo_ok && hi_ok)) return 0;
    }
  }
  return 1;
}

/* guard fill of the newer slice of patch p from its neighbours' two slices */
void orc_fill_guards_local(const orc_desc *d, const int32_t *nbr, real *S0, real *S1, const int32_t *cur,
                           const double *t_old, const double *t_new, int32_t p) {
  geom G; mkgeom(d, &G);
  real *S[2] = {S0, S1};
  real *Up = S[cur[p]];
  box all = mkbox(&G, G.g[0], G.g[0], G.g[1], G.g[1], G.g[2], G.g[2]);
  BOXLOOP(all) {
    int c[3] = {i, j, k}, o[3], src[3], clamp[3];
    int guard = 0;
    for (int a = 0; a < 3; ++a) {
      o[a] = c[a] < 0 ? -1 : (c[a] >= G.n[a] ? 1 : 0);
      if (o[a]) guard = 1;
      src[a] = c[a] - o[a] * G.n[a];
      clamp[a] = c[a] < 0 ? 0 : (c[a] >= G.n[a] ? G.n[a] - 1 : c[a]);
    }
    if (!guard) continue;
    int q = nbr[p * 27 + (o[2] + 1) * 9 + (o[1] + 1) * 3 + (o[0] + 1)];
    long dst = cidx(&G, i, j, k);
    for (int f = 0; f < 8; ++f) {
      long fo = (long)f * G.np * G.M;
      if (q >= 0) {
        long from = fo + (long)q * G.M + cidx(&G, src[0], src[1], src[2]);
        real vnew = S[cur[q]][from];
        real v = vnew;
        if (!times_equal(t_new[p], t_new[q]) && !times_equal(t_new[q], t_old[q])) {
          real vold = S[1 - cur[q]][from];
          real w = (real)((t_new[p] - t_old[q]) / (t_new[q] - t_old[q]));
          v = vold + w * (vnew - vold);
        }
        Up[fo + (long)p * G.M + dst] = v;
      } else {
        if (f >= 5) { /* the closing face keeps its evolved value (O8) */
          int a = f - 5, b = (a + 1) % 3, e = (a + 2) % 3;
          if (c[a] == G.n[a] && G.act[a] && o[b] == 0 && o[e] == 0) continue;
        }
        Up[fo + (long)p * G.M + dst] = Up[fo + (long)p * G.M + cidx(&G, clamp[0], clamp[1], clamp[2])];
      }
    }
  }
}

/* One call advances the patches list[0..n) by their own dt[i]: (1) time-interpolated guard fill
 * of the newer slice of every listed patch; (2) O2-O8 from the newer slice into the older one,
 * which becomes the newer one (cur flips, t_old <- t_new, t_new += dt).  Readiness (the rule
 * under which DISPATCH updates a task): t_old[q] <= t_new[p] <= t_new[q] for every neighbour q of
 * a listed p, so that guard values are interpolated, never extrapolated; two listed neighbours
 * are then at the same time and read only each other's newer slices, which this call does not
 * write.  Returns 0, or -1 (nothing done) if a listed patch is not ready.                      */
int orc_step_local(const orc_desc *d, const int32_t *nbr, real *S0, real *S1, int32_t *cur, double *t_old,
                   double *t_new, const int32_t *list, int32_t n, const double *dt) {
  if (!orc_local_ready(d, nbr, t_old, t_new, list, n)) return -1;
  geom G; mkgeom(d, &G);
  real *S[2] = {S0, S1};
  for (int i = 0; i < n; ++i) orc_fill_guards_local(d, nbr, S0, S1, cur, t_old, t_new, list[i]);
  real *buf = (real *)malloc(sizeof(real) * ORC_NSTAGE * G.M);
  scratch Sc; scratch_bind(&Sc, buf, G.M);
  for (int i = 0; i < n; ++i) {
    int p = list[i];
    const real *Up[8]; real *Un[8];
    for (int f = 0; f < 8; ++f) {
      Up[f] = S[cur[p]] + ((long)f * G.np + p) * G.M;
      Un[f] = S[1 - cur[p]] + ((long)f * G.np + p) * G.M;
    }
    run_stages(&G, Up, (real)dt[i], &Sc);
    update_patch(&G, Up, Un, (real)dt[i], &Sc);
  }
  free(buf);
  for (int i = 0; i < n; ++i) {
    int p = list[i];
    cur[p] = 1 - cur[p];
    t_old[p] = t_new[p];
    t_new[p] += dt[i];
  }
  return 0;
}
