// mhd_math.cuh -- pointwise device arithmetic of the bunch MHD update (sm_100a).
//
// Limiter, fast speed, HLLD flux (Miyoshi & Kusano 2005)
// and the two-dimensional Riemann problem for the edge EMF (
// DESIGN.md reading O7).  Everything is branch-light: wave-pattern choices are selects,
// so a warp never serialises over the six HLLD regions.
#pragma once
#include <cuda_runtime.h>
#include <float.h>

namespace mhd {

template <typename T> struct num;
// fp32: one MUFU per reciprocal / square root (rcp.approx, sqrt.approx: <= 2 ulp) instead of
// the IEEE sequences with their slow-path branches; the parity budget (2e-5 per cell and
// step against ~1e-7 observed) leaves two orders of magnitude for this.
template <> struct num<float> {
  static __device__ __forceinline__ float eps() { return FLT_EPSILON; }
  static __device__ __forceinline__ float sqrt(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
  static __device__ __forceinline__ float abs(float x) { return fabsf(x); }
  static __device__ __forceinline__ float min(float a, float b) { return fminf(a, b); }
  static __device__ __forceinline__ float max(float a, float b) { return fmaxf(a, b); }
  static __device__ __forceinline__ float rcp(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
  static __device__ __forceinline__ float rsqrt(float x) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
  static __device__ __forceinline__ float div(float a, float b) { return a * rcp(b); }
  // single correctly rounded operations the compiler never fuses or reorders
  static __device__ __forceinline__ float xmul(float a, float b) { return __fmul_rn(a, b); }
  static __device__ __forceinline__ float xadd(float a, float b) { return __fadd_rn(a, b); }
  static __device__ __forceinline__ float xfma(float a, float b, float c) { return __fmaf_rn(a, b, c); }
};
template <> struct num<double> {
  static __device__ __forceinline__ double eps() { return DBL_EPSILON; }
  // fp64: MUFU seed (rcp/rsqrt.approx.ftz.f64, relative error below 2^-20) refined by ONE
  // third-order step in DFMA -- the residual e of the seed leaves e^3 < 2^-60, i.e. the result
  // is good to a few units of 1e-16 without the IEEE sequences' slow-path calls and branches
  // and with fewer DFMA than two Newton steps (tolerance of the path: 1e-12 per cell and
  // step).  Arguments here are normal, non-zero numbers; sqrt(0) is handled explicitly.
  static __device__ __forceinline__ double rsqrt(double a) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    const double e = fma(-(a * y), y, 1.0);            // 1 - a y^2
    return fma(y, fma(0.375, e, 0.5) * e, y);          // y (1 + e/2 + 3 e^2/8)
  }
  static __device__ __forceinline__ double sqrt(double a) {
    const double s = a * rsqrt(a);
    return a > 0.0 ? s : 0.0;
  }
  static __device__ __forceinline__ double abs(double x) { return fabs(x); }
  static __device__ __forceinline__ double min(double a, double b) { return fmin(a, b); }
  static __device__ __forceinline__ double max(double a, double b) { return fmax(a, b); }
  static __device__ __forceinline__ double rcp(double a) {
    double x;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(x) : "d"(a));
    const double e = fma(-a, x, 1.0);                  // 1 - a x
    return fma(x, fma(e, e, e), x);                    // x (1 + e + e^2)
  }
  static __device__ __forceinline__ double div(double a, double b) { return a * rcp(b); }
  static __device__ __forceinline__ double xmul(double a, double b) { return __dmul_rn(a, b); }
  static __device__ __forceinline__ double xadd(double a, double b) { return __dadd_rn(a, b); }
  static __device__ __forceinline__ double xfma(double a, double b, double c) { return __fma_rn(a, b, c); }
};

// ---- slope limiter: 0 at extrema; minmod (1) or monotonised central (2) -------------
template <typename T>
__device__ __forceinline__ T limited_slope(int kind, T a, T b) {
  using N = num<T>;
  const T fa = N::abs(a), fb = N::abs(b);
  T m = N::min(fa, fb);
  if (kind == 2) m = N::min(T(2) * m, T(0.5) * N::abs(a + b));
  m = (a * b > T(0)) ? m : T(0);
  return a < T(0) ? -m : m;
}
// the same with the kind fixed at compile time.  minmod(a,b) is the median of (a, b, 0):
// four min/max instructions and no product, sign test or select (and no underflow of a*b)
template <int KIND, typename T>
__device__ __forceinline__ T limited_slope_k(T a, T b) {
  using N = num<T>;
  if (KIND == 1) return N::max(N::min(a, b), N::min(N::max(a, b), T(0)));
  return limited_slope(2, a, b);
}

// ---- fast magnetosonic speed along a direction with normal field bn ---------------
// gp = gamma*p, b2 = |B|^2, bn2 = bn^2, irho = 1/rho
template <typename T>
__device__ __forceinline__ T fast_speed2(T gp, T b2, T bn2, T irho) {   // c_f^2
  using N = num<T>;
  const T s = gp + b2;
  const T disc = N::max(s * s - T(4) * gp * bn2, T(0));
  return T(0.5) * (s + N::sqrt(disc)) * irho;
}
template <typename T>
__device__ __forceinline__ T fast_speed(T gp, T b2, T bn2, T irho) {
  return num<T>::sqrt(fast_speed2(gp, b2, bn2, irho));
}

// ---- CFL rate of a cell (O9): sum over active d of (|u_d| + c_f,d)/dx_d ----
// From the conserved values and the six face fields of the cell.  Written with explicitly rounded
// operations in a fixed order, so that every kernel that evaluates it (the stand-alone k_cfl and the
// epilogue of the one-pass step) gets the same bits from the same inputs.  NaN -> +inf (dt = 0).
template <typename T>
__device__ __forceinline__ T cfl_rate(T gamma, T idx0, T idx1, T idx2, bool a0, bool a1, bool a2, T rho, T mx, T my, T mz,
                                      T en, T bxl, T bxu, T byl, T byu, T bzl, T bzu) {
  using N = num<T>;
  const T h = T(0.5);
  const T ir = N::rcp(rho);
  const T u = N::xmul(mx, ir), v = N::xmul(my, ir), w = N::xmul(mz, ir);
  const T bx = N::xmul(h, N::xadd(bxl, bxu)), by = N::xmul(h, N::xadd(byl, byu)), bz = N::xmul(h, N::xadd(bzl, bzu));
  const T bx2 = N::xmul(bx, bx), by2 = N::xmul(by, by), bz2 = N::xmul(bz, bz);
  const T b2 = N::xadd(N::xadd(bx2, by2), bz2);
  const T v2 = N::xfma(w, w, N::xfma(v, v, N::xmul(u, u)));
  const T pr = N::xmul(gamma - T(1), N::xadd(N::xfma(-N::xmul(h, rho), v2, en), -N::xmul(h, b2)));
  const T gp = N::xmul(gamma, pr);
  const T s = N::xadd(gp, b2), s2 = N::xmul(s, s), g4 = N::xmul(T(4), gp);
  auto cf = [&](T bn2) {
    const T disc = N::max(N::xfma(-g4, bn2, s2), T(0));
    return N::sqrt(N::xmul(N::xmul(h, N::xadd(s, N::sqrt(disc))), ir));
  };
  T rate = T(0);
  if (a0) rate = N::xfma(N::xadd(N::abs(u), cf(bx2)), idx0, rate);
  if (a1) rate = N::xfma(N::xadd(N::abs(v), cf(by2)), idx1, rate);
  if (a2) rate = N::xfma(N::xadd(N::abs(w), cf(bz2)), idx2, rate);
  return rate == rate ? rate : T(INFINITY);
}

// primitive state seen by a 1D Riemann problem: normal velocity u, transverse (v,w),
// transverse field (by,bz)
template <typename T> struct State1D { T rho, u, v, w, p, by, bz; };
template <typename T> struct Flux5 { T d, mu, mv, mw, e; };

// ---- HLLD flux of (rho, rho u, rho v, rho w, E) ------------------------------------
// The side that contains the interface (left if S_L>0 or S*_L>0 or S_M>=0) is selected
// first; only that side's star and double-star states are formed.
template <typename T>
__device__ __forceinline__ Flux5<T> hlld_flux(T gamma, const State1D<T>& L, const State1D<T>& R, T bn) {
  using N = num<T>;
  const T half = T(0.5);
  const T bn2 = bn * bn;
  const T igm1 = N::rcp(gamma - T(1));

  const T b2L = bn2 + L.by * L.by + L.bz * L.bz, b2R = bn2 + R.by * R.by + R.bz * R.bz;
  const T pTL = L.p + half * b2L, pTR = R.p + half * b2R;
  // the square root is monotonic: one sqrt of the larger c_f^2
  const T cmax = N::sqrt(N::max(fast_speed2(gamma * L.p, b2L, bn2, N::rcp(L.rho)),
                                fast_speed2(gamma * R.p, b2R, bn2, N::rcp(R.rho))));
  const T SL = N::min(L.u, R.u) - cmax, SR = N::max(L.u, R.u) + cmax;

  const T sdL = SL - L.u, sdR = SR - R.u;
  const T mL = L.rho * sdL, mR = R.rho * sdR;
  const T SM = N::div(mR * R.u - mL * L.u - pTR + pTL, mR - mL);
  const T pTs = pTL + mL * (SM - L.u);

  // star densities and transverse star values of BOTH sides (the double-star state mixes them)
  const T rsL = N::div(mL, SL - SM), rsR = N::div(mR, SR - SM);
  const T DL = mL * (SL - SM) - bn2, DR = mR * (SR - SM) - bn2;
  const T refL = mL * sdL, refR = mR * sdR;
  const bool degL = N::abs(DL) <= T(16) * N::eps() * refL;
  const bool degR = N::abs(DR) <= T(16) * N::eps() * refR;
  const T iDL = degL ? T(0) : N::rcp(DL), iDR = degR ? T(0) : N::rcp(DR);
  const T kvL = bn * (SM - L.u) * iDL, kvR = bn * (SM - R.u) * iDR;       // v* = v - kv*by
  const T kbL = degL ? T(1) : (refL - bn2) * iDL, kbR = degR ? T(1) : (refR - bn2) * iDR;
  const T vsL = L.v - kvL * L.by, wsL = L.w - kvL * L.bz, bysL = L.by * kbL, bzsL = L.bz * kbL;
  const T vsR = R.v - kvR * R.by, wsR = R.w - kvR * R.bz, bysR = R.by * kbR, bzsR = R.bz * kbR;

  const T irL = N::rsqrt(rsL), irR = N::rsqrt(rsR);
  const T rL = rsL * irL, rR = rsR * irR;             // sqrt(rho*) from the same MUFU result
  const T abn = N::abs(bn);
  const T SsL = SM - abn * irL, SsR = SM + abn * irR;
  const T sg = bn > T(0) ? T(1) : (bn < T(0) ? T(-1) : T(0));

  // which side holds the interface, and how deep into the fan it sits
  const bool left = (SL > T(0)) || (SsL > T(0)) || (SM >= T(0));
  const bool star = left ? !(SL > T(0)) : (SsR >= T(0) || SR >= T(0));
  const bool dstar = left ? !(SL > T(0) || SsL > T(0)) : (SsR >= T(0));

  // own side = the selected one
  const T rho = left ? L.rho : R.rho, u = left ? L.u : R.u, v = left ? L.v : R.v, w = left ? L.w : R.w;
  const T p = left ? L.p : R.p, by = left ? L.by : R.by, bz = left ? L.bz : R.bz;
  const T b2 = left ? b2L : b2R, pT = left ? pTL : pTR;
  const T S = left ? SL : SR, sd = left ? sdL : sdR, Ss = left ? SsL : SsR;
  const T rs = left ? rsL : rsR, ro = left ? rL : rR, rx = left ? rR : rL;
  const T vs = left ? vsL : vsR, ws = left ? wsL : wsR, bys = left ? bysL : bysR, bzs = left ? bzsL : bzsR;
  const T vx = left ? vsR : vsL, wx = left ? wsR : wsL, byx = left ? bysR : bysL, bzx = left ? bzsR : bzsL;
  const T tau = left ? sg : -sg;          // sign(bn) seen from the own side

  const T E = p * igm1 + half * rho * (u * u + v * v + w * w) + half * b2;
  const T ub = u * bn + v * by + w * bz;
  // physical flux, Eq. 6
  Flux5<T> F;
  F.d = rho * u;
  F.mu = rho * u * u + pT - bn2;
  F.mv = rho * v * u - by * bn;
  F.mw = rho * w * u - bz * bn;
  F.e = u * (E + pT) - bn * ub;

  // star state
  const T ubs = SM * bn + vs * bys + ws * bzs;
  const T Es = N::div(sd * E - pT * u + pTs * SM + bn * (ub - ubs), S - SM);
  // double-star state
  const T irs = N::rcp(ro + rx);
  const T vss = (ro * vs + rx * vx + tau * (byx - bys)) * irs;
  const T wss = (ro * ws + rx * wx + tau * (bzx - bzs)) * irs;
  const T byss = (ro * byx + rx * bys + ro * rx * tau * (vx - vs)) * irs;
  const T bzss = (ro * bzx + rx * bzs + ro * rx * tau * (wx - ws)) * irs;
  const T ubss = SM * bn + vss * byss + wss * bzss;
  const T Ess = Es - tau * ro * (ubs - ubss);

  const T c1 = star ? S : T(0), c2 = dstar ? Ss : T(0);
  F.d += c1 * (rs - rho);
  F.mu += c1 * (rs * SM - rho * u);
  F.mv += c1 * (rs * vs - rho * v) + c2 * rs * (vss - vs);
  F.mw += c1 * (rs * ws - rho * w) + c2 * rs * (wss - ws);
  F.e += c1 * (Es - E) + c2 * (Ess - Es);
  return F;
}

// ---- HLL flux (section 2.1.1) --------------------------------------
// Three regions; the star state is the integral average between the outer waves, so the
// flux through the interface is (SR FL - SL FR + SL SR (UR - UL)) / (SR - SL) inside the fan.
// With SL clipped to <= 0 and SR to >= 0 the same expression returns FL / FR outside it.
template <typename T>
__device__ __forceinline__ Flux5<T> hll_flux(T gamma, const State1D<T>& L, const State1D<T>& R, T bn) {
  using N = num<T>;
  const T half = T(0.5), bn2 = bn * bn;
  const T igm1 = N::rcp(gamma - T(1));
  const T b2L = bn2 + L.by * L.by + L.bz * L.bz, b2R = bn2 + R.by * R.by + R.bz * R.bz;
  const T pTL = L.p + half * b2L, pTR = R.p + half * b2R;
  const T cmax = N::sqrt(N::max(fast_speed2(gamma * L.p, b2L, bn2, N::rcp(L.rho)),
                                fast_speed2(gamma * R.p, b2R, bn2, N::rcp(R.rho))));
  const T SL = N::min(N::min(L.u, R.u) - cmax, T(0)), SR = N::max(N::max(L.u, R.u) + cmax, T(0));
  const T EL = L.p * igm1 + half * L.rho * (L.u * L.u + L.v * L.v + L.w * L.w) + half * b2L;
  const T ER = R.p * igm1 + half * R.rho * (R.u * R.u + R.v * R.v + R.w * R.w) + half * b2R;
  const T ubL = L.u * bn + L.v * L.by + L.w * L.bz, ubR = R.u * bn + R.v * R.by + R.w * R.bz;
  const T mL = L.rho * L.u, mR = R.rho * R.u;
  const T inv = N::rcp(SR - SL), ss = SL * SR;
  Flux5<T> F;
  F.d = (SR * mL - SL * mR + ss * (R.rho - L.rho)) * inv;
  F.mu = (SR * (mL * L.u + pTL - bn2) - SL * (mR * R.u + pTR - bn2) + ss * (mR - mL)) * inv;
  F.mv = (SR * (mL * L.v - L.by * bn) - SL * (mR * R.v - R.by * bn) + ss * (R.rho * R.v - L.rho * L.v)) * inv;
  F.mw = (SR * (mL * L.w - L.bz * bn) - SL * (mR * R.w - R.bz * bn) + ss * (R.rho * R.w - L.rho * L.w)) * inv;
  F.e = (SR * (L.u * (EL + pTL) - bn * ubL) - SL * (R.u * (ER + pTR) - bn * ubR) + ss * (ER - EL)) * inv;
  return F;
}

// flux solver of the faces: 0 = HLLD, 1 = HLL (mhd_bunch_desc.flux_solver)
template <typename T>
__device__ __forceinline__ Flux5<T> riemann_flux(int flux_solver, T gamma, const State1D<T>& L, const State1D<T>& R, T bn) {
  return flux_solver == 1 ? hll_flux(gamma, L, R, bn) : hlld_flux(gamma, L, R, bn);
}
template <int FS, typename T>
__device__ __forceinline__ Flux5<T> riemann_flux_k(T gamma, const State1D<T>& L, const State1D<T>& R, T bn) {
  if (FS == 1) return hll_flux(gamma, L, R, bn);
  return hlld_flux(gamma, L, R, bn);
}

// ---- two-dimensional Riemann problem at an edge -------------------------------------
// Corner states (rho, ua, ub, p, be) with be the out-of-plane field; in-plane fields are
// single-valued per side: A (component a) south/north, B (component b) west/east.
template <typename T> struct Corner { T rho, ua, ub, p, be; };

template <typename T> struct Sub1D { T bsL, bsR, lo, hi; };

// star transverse field and Alfven-type bounds of a 1D sub-problem with given outer speeds
template <typename T>
__device__ __forceinline__ Sub1D<T> sub_star(T rhoL, T unL, T pTL, T btL, T rhoR, T unR, T pTR, T btR,
                                             T bn, T SL, T SR) {
  using N = num<T>;
  const T bn2 = bn * bn;
  const T sdL = SL - unL, sdR = SR - unR;
  const T mL = rhoL * sdL, mR = rhoR * sdR;
  const T SM = N::div(mR * unR - mL * unL - pTR + pTL, mR - mL);
  const T dL = SL - SM, dR = SR - SM;
  const T DL = mL * dL - bn2, DR = mR * dR - bn2;
  const T refL = mL * sdL, refR = mR * sdR;
  Sub1D<T> s;
  s.bsL = (N::abs(DL) <= T(16) * N::eps() * refL) ? btL : btL * N::div(refL - bn2, DL);
  s.bsR = (N::abs(DR) <= T(16) * N::eps() * refR) ? btR : btR * N::div(refR - bn2, DR);
  const T abn = N::abs(bn);
  // rho*_K = m_K / d_K  =>  |bn| / sqrt(rho*_K) = |bn| * sqrt(d_K / m_K)
  s.lo = SM - abn * N::sqrt(N::div(dL, mL));
  s.hi = SM + abn * N::sqrt(N::div(dR, mR));
  return s;
}

template <typename T>
__device__ __forceinline__ T emf_2d(T gamma, int solver, const Corner<T>& sw, const Corner<T>& se,
                                    const Corner<T>& nw, const Corner<T>& ne, T AS, T AN, T BW, T BE) {
  using N = num<T>;
  const T half = T(0.5), zero = T(0);
  const T eSW = sw.ua * BW - sw.ub * AS, eSE = se.ua * BE - se.ub * AS;
  const T eNW = nw.ua * BW - nw.ub * AN, eNE = ne.ua * BE - ne.ub * AN;
  const T AS2 = AS * AS, AN2 = AN * AN, BW2 = BW * BW, BE2 = BE * BE;
  const T b2SW = AS2 + BW2 + sw.be * sw.be, b2SE = AS2 + BE2 + se.be * se.be;
  const T b2NW = AN2 + BW2 + nw.be * nw.be, b2NE = AN2 + BE2 + ne.be * ne.be;
  const T iSW = N::rcp(sw.rho), iSE = N::rcp(se.rho), iNW = N::rcp(nw.rho), iNE = N::rcp(ne.rho);
  const T gSW = gamma * sw.p, gSE = gamma * se.p, gNW = gamma * nw.p, gNE = gamma * ne.p;
  const T ca = N::sqrt(N::max(N::max(fast_speed2(gSW, b2SW, AS2, iSW), fast_speed2(gSE, b2SE, AS2, iSE)),
                              N::max(fast_speed2(gNW, b2NW, AN2, iNW), fast_speed2(gNE, b2NE, AN2, iNE))));
  const T cb = N::sqrt(N::max(N::max(fast_speed2(gSW, b2SW, BW2, iSW), fast_speed2(gSE, b2SE, BE2, iSE)),
                              N::max(fast_speed2(gNW, b2NW, BW2, iNW), fast_speed2(gNE, b2NE, BE2, iNE))));
  const T tW = N::min(N::min(sw.ua, se.ua), N::min(nw.ua, ne.ua)) - ca;
  const T tE = N::max(N::max(sw.ua, se.ua), N::max(nw.ua, ne.ua)) + ca;
  const T tS = N::min(N::min(sw.ub, se.ub), N::min(nw.ub, ne.ub)) - cb;
  const T tN = N::max(N::max(sw.ub, se.ub), N::max(nw.ub, ne.ub)) + cb;

  T SW_, SE_, SS_, SN_, e0 = eSW, e1 = eSE, e2 = eNW, e3 = eNE;
  T BsSW = BW, BsSE = BE, BsNW = BW, BsNE = BE, AsSW = AS, AsSE = AS, AsNW = AN, AsNE = AN;
  if (solver == 1) {
    SW_ = N::min(zero, tW); SE_ = N::max(zero, tE); SS_ = N::min(zero, tS); SN_ = N::max(zero, tN);
  } else {
    const T pSW = sw.p + half * b2SW, pSE = se.p + half * b2SE, pNW = nw.p + half * b2NW, pNE = ne.p + half * b2NE;
    const Sub1D<T> xS = sub_star(sw.rho, sw.ua, pSW, BW, se.rho, se.ua, pSE, BE, AS, tW, tE);
    const Sub1D<T> xN = sub_star(nw.rho, nw.ua, pNW, BW, ne.rho, ne.ua, pNE, BE, AN, tW, tE);
    const Sub1D<T> yW = sub_star(sw.rho, sw.ub, pSW, AS, nw.rho, nw.ub, pNW, AN, BW, tS, tN);
    const Sub1D<T> yE = sub_star(se.rho, se.ub, pSE, AS, ne.rho, ne.ub, pNE, AN, BE, tS, tN);
    SW_ = tW >= zero ? zero : N::min(zero, N::min(xS.lo, xN.lo));
    SE_ = tE <= zero ? zero : N::max(zero, N::max(xS.hi, xN.hi));
    SS_ = tS >= zero ? zero : N::min(zero, N::min(yW.lo, yE.lo));
    SN_ = tN <= zero ? zero : N::max(zero, N::max(yW.hi, yE.hi));
    BsSW = xS.bsL; BsSE = xS.bsR; BsNW = xN.bsL; BsNE = xN.bsR;
    AsSW = yW.bsL; AsNW = yW.bsR; AsSE = yE.bsL; AsNE = yE.bsR;
    const T SxW = N::min(tW, zero), SxE = N::max(tE, zero), SyS = N::min(tS, zero), SyN = N::max(tN, zero);
    e0 += SxW * (BsSW - BW) - SyS * (AsSW - AS);
    e1 += SxE * (BsSE - BE) - SyS * (AsSE - AS);
    e2 += SxW * (BsNW - BW) - SyN * (AsNW - AN);
    e3 += SxE * (BsNE - BE) - SyN * (AsNE - AN);
  }
  const T dxs = SE_ - SW_, dys = SN_ - SS_;
  const bool zx = dxs == zero, zy = dys == zero;
  const T idx = zx ? zero : N::rcp(dxs), idy = zy ? zero : N::rcp(dys);
  const T aE = zx ? half : SE_ * idx, aW = zx ? half : -SW_ * idx;
  const T bN = zy ? half : SN_ * idy, bS = zy ? half : -SS_ * idy;
  const T BsW = bN * BsSW + bS * BsNW, BsE = bN * BsSE + bS * BsNE;
  const T AsS = aE * AsSW + aW * AsSE, AsN = aE * AsNW + aW * AsNE;
  return aE * (bN * e0 + bS * e2) + aW * (bN * e1 + bS * e3)
       + (SW_ * SE_ * idx) * (BsE - BsW) - (SS_ * SN_ * idy) * (AsN - AsS);
}

}  // namespace mhd
