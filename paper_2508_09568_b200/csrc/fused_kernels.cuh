// fused_kernels.cuh -- the fast 3D path of the step (all three dimensions active).
//
// k_riemann_update: interface states + HLLD at the three lower faces + the 2D Riemann
// problem at the three lower edges + conservative/constrained-transport update
// (Eq. 12) in ONE kernel.  A CTA owns an (x,y) tile of one patch
// and marches along z.  Per plane the predictor data of the tile and its one-cell halo
// ("D-data": half-step primitives, half-step fields, limited slopes) are staged in
// shared memory with compile-time strides; fluxes and EMFs never touch HBM: a thread
// keeps its own lower-face values in registers and reads the upper-face values of its
// +x / +y neighbours through a small shared exchange buffer.
#pragma once
#include "bunch_types.cuh"
#include "mhd_math.cuh"
#include "tma_utils.cuh"

namespace mhd {

// order of the D-data arrays, in the shared-memory planes AND in the scratch block W_D
enum : int {
  D_QH = 0,    // 5  rho,u,v,w,p at n+1/2
  D_BCH = 5,   // 3  cell-centred half-step field (mean of the two half-step faces)
  D_BH = 8,    // 3  half-step lower-face fields
  D_DQ = 11,   // 21 limited slopes [dir][rho,u,v,w,p, B_(dir+1), B_(dir+2)]
  D_DBF = 32,  // 6  transverse slopes of the face fields
  D_COUNT = 38
};
static_assert((int)D_COUNT == (int)W_DCOUNT, "the D block must hold the D arrays");

// slot of the slope of primitive f (0..7, f != 5+d) along d
__host__ __device__ constexpr int dq_slot(int d, int f) {
  return D_DQ + d * 7 + (f < 5 ? f : 5 + ((f - 5 - d + 3) % 3 - 1));
}
// staged-path scratch array that corresponds to D slot a (a not in the D_BCH group)
__host__ __device__ constexpr int d_source(int a) {
  if (a < D_BCH) return W_QH + a;
  if (a < D_BH) return -1;
  if (a < D_DQ) return W_BH + (a - D_BH);
  if (a < D_DBF) {
    const int d = (a - D_DQ) / 7, r = (a - D_DQ) % 7;
    const int f = r < 5 ? r : 5 + (d + 1 + (r - 5)) % 3;
    return W_DQ + d * 8 + f;
  }
  return W_DBF + (a - D_DBF);
}

// Tile geometry of k_riemann_update.  The shared tile is DW x DH cells: columns
// x0-1 .. x0+DW-2 (at least up to x0+TXM; DW*sizeof(T) is a multiple of 16 bytes for TMA),
// rows y0-1 .. y0+TYM.  Threads form FW x FH faces/edges.
template <typename T, int TXM, int TYM> struct FusedCfg {
  static constexpr int VE = 16 / (int)sizeof(T);                           // elements per 16 bytes
  static constexpr int DW = ((TXM + 2 + VE - 1) / VE) * VE, DH = TYM + 2, DC = DW * DH;
  static constexpr int FW = TXM + 1, FH = TYM + 1;
  // Thread layout: threads [0, TXM*FH) own face columns 0..TXM-1 row by row (a warp never
  // straddles tile rows unevenly, so shared-memory accesses are conflict-free); one more warp
  // starting at CB owns the closing column fi = TXM, one lane per row.
  static constexpr int CB = ((TXM * FH + 31) / 32) * 32;
  static constexpr int NTH = CB + 32;
  static_assert(FH <= 32 && 32 % TXM == 0, "tile shape");
  static constexpr int XV = sizeof(T) == 8 ? 3 : 4;                 // values per y-exchange pass (7 in all)
  static constexpr int XC = 7;                                      // values the closing column hands to column TXM-1
  static constexpr int XR = FH <= 16 ? 16 : 32;                     // rows of that hand-over buffer
  static constexpr uint32_t slot_bytes = (uint32_t)(sizeof(T) * D_COUNT * DC);
  static constexpr uint32_t slot_stride = (slot_bytes + 127u) / 128u * 128u;   // TMA destinations: 128-byte aligned
  static constexpr size_t smem = 2 * (size_t)slot_stride + sizeof(T) * (size_t)(XV * NTH + XC * XR) + 16;
};

// HLLD flux through the face between cell `cl` and cell `cr` along D; pointers address
// array 0 of the respective cells, arrays are DC elements apart
template <typename T, int DC, int D>
__device__ __forceinline__ Flux5<T> face_flux(const T* __restrict__ cl, const T* __restrict__ cr, T gamma, int flux_solver) {
  constexpr int T1 = (D + 1) % 3, T2 = (D + 2) % 3;
  const T h = T(0.5);
  State1D<T> L, R;
  L.rho = cl[(D_QH + 0) * DC] + h * cl[dq_slot(D, 0) * DC];
  L.u = cl[(D_QH + 1 + D) * DC] + h * cl[dq_slot(D, 1 + D) * DC];
  L.v = cl[(D_QH + 1 + T1) * DC] + h * cl[dq_slot(D, 1 + T1) * DC];
  L.w = cl[(D_QH + 1 + T2) * DC] + h * cl[dq_slot(D, 1 + T2) * DC];
  L.p = cl[(D_QH + 4) * DC] + h * cl[dq_slot(D, 4) * DC];
  L.by = cl[(D_BCH + T1) * DC] + h * cl[dq_slot(D, 5 + T1) * DC];
  L.bz = cl[(D_BCH + T2) * DC] + h * cl[dq_slot(D, 5 + T2) * DC];
  R.rho = cr[(D_QH + 0) * DC] - h * cr[dq_slot(D, 0) * DC];
  R.u = cr[(D_QH + 1 + D) * DC] - h * cr[dq_slot(D, 1 + D) * DC];
  R.v = cr[(D_QH + 1 + T1) * DC] - h * cr[dq_slot(D, 1 + T1) * DC];
  R.w = cr[(D_QH + 1 + T2) * DC] - h * cr[dq_slot(D, 1 + T2) * DC];
  R.p = cr[(D_QH + 4) * DC] - h * cr[dq_slot(D, 4) * DC];
  R.by = cr[(D_BCH + T1) * DC] - h * cr[dq_slot(D, 5 + T1) * DC];
  R.bz = cr[(D_BCH + T2) * DC] - h * cr[dq_slot(D, 5 + T2) * DC];
  return riemann_flux(flux_solver, gamma, L, R, cr[(D_BH + D) * DC]);
}

// EMF at the edge along E shared by cells sw=(a-1,b-1), se=(a,b-1), nw=(a-1,b), ne=(a,b)
template <typename T, int DC, int E>
__device__ __forceinline__ T edge_emf(const T* __restrict__ csw, const T* __restrict__ cse, const T* __restrict__ cnw,
                                      const T* __restrict__ cne, T gamma, int solver) {
  constexpr int A = (E + 1) % 3, B = (E + 2) % 3;
  const T h = T(0.5);
  auto corner = [&](const T* c, T sa, T sb) {
    Corner<T> q;
    q.rho = c[(D_QH + 0) * DC] + sa * c[dq_slot(A, 0) * DC] + sb * c[dq_slot(B, 0) * DC];
    q.ua = c[(D_QH + 1 + A) * DC] + sa * c[dq_slot(A, 1 + A) * DC] + sb * c[dq_slot(B, 1 + A) * DC];
    q.ub = c[(D_QH + 1 + B) * DC] + sa * c[dq_slot(A, 1 + B) * DC] + sb * c[dq_slot(B, 1 + B) * DC];
    q.p = c[(D_QH + 4) * DC] + sa * c[dq_slot(A, 4) * DC] + sb * c[dq_slot(B, 4) * DC];
    q.be = c[(D_BCH + E) * DC] + sa * c[dq_slot(A, 5 + E) * DC] + sb * c[dq_slot(B, 5 + E) * DC];
    return q;
  };
  const Corner<T> sw = corner(csw, h, h), se = corner(cse, -h, h), nw = corner(cnw, h, -h), ne = corner(cne, -h, -h);
  constexpr int SA = D_DBF + (A == 0 ? (B == 1 ? 0 : 1) : (A == 1 ? (B == 0 ? 2 : 3) : (B == 0 ? 4 : 5)));
  constexpr int SB = D_DBF + (B == 0 ? (A == 1 ? 0 : 1) : (B == 1 ? (A == 0 ? 2 : 3) : (A == 0 ? 4 : 5)));
  const T AS = cse[(D_BH + A) * DC] + h * cse[SA * DC], AN = cne[(D_BH + A) * DC] - h * cne[SA * DC];
  const T BW = cnw[(D_BH + B) * DC] + h * cnw[SB * DC], BE = cne[(D_BH + B) * DC] - h * cne[SB * DC];
  return emf_2d(gamma, solver, sw, se, nw, ne, AS, AN, BW, BE);
}

// ---------------------------------------------------------------------------------------
// k_predict_fused: primitives (O2), edge EMFs at time n (O4a, Eq. 7-11), limited slopes (O3),
// half-step face fields (O4b, Eq. 12 with dt/2), primitive half step (O4c) and the
// cell-centred half-step field, written straight into the D block -- one kernel instead of
// prim + emf0 + predict + pack.  A CTA owns a y-tile of one patch over
// the full x extent and marches along z; a thread owns one (x,y) position.  Rings in shared
// memory hold what neighbours need: primitives of 3 planes, raw face fields of 3 planes,
// edge EMFs of 2 planes; the state itself is read exactly once per position and plane
// (register prefetch of the next plane).
// Position (pc,pr) <-> cell i = pc-2, j = y0-2+pr; PW = nx+5 columns, PH = TY+5 rows.
__host__ __device__ constexpr int predict_max_threads(int ty) { return ty == 8 ? 512 : 832; }

template <typename T, int TY>
__global__ void __launch_bounds__(predict_max_threads(TY), (TY == 8 && sizeof(T) == 4) ? 2 : 1)
k_predict_fused(Params<T> P, const double* __restrict__ dtp, unsigned long long* __restrict__ bad,
                const int* __restrict__ nbr, int gather) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const Geom& G = P.G;
  const int nx = G.n[0], ny = G.n[1], nz = G.n[2];
  const int PW = nx + 5, PH = TY + 5, PA = PW * PH;
  T* Q = reinterpret_cast<T*>(smem_raw);   // [3][8][PA] primitives
  T* QB = Q + 3 * 8 * PA;                  // [3][3][PA] raw face fields
  T* E = QB + 3 * 3 * PA;                  // [2][3][PA] edge EMFs at time n (ex, ey, ez)

  const int pl = blockIdx.y, y0 = blockIdx.x * TY;
  const int rows = min(TY, ny - y0);
  const bool lasty = (y0 + rows == ny);
  const int ya = (y0 == 0) ? -1 : y0, yb = lasty ? ny : y0 + rows - 1;   // D rows written by this tile
  const int t = threadIdx.x;
  const int pr = t / PW, pc = t - pr * PW;
  const bool inpos = t < PA;
  const int i = pc - 2, j = y0 - 2 + pr;
  const int o = pr * PW + pc;
  const bool rowok = inpos && (j + G.g[1] >= 0) && (j + G.g[1] < G.m[1]);
  const long long pitch = G.pitch, plane = (long long)G.pitch * G.m[1], fs = G.fs;
  const long long cbase = (long long)P.patch(pl) * G.ps + G.lead + (i + G.g[0]) + (long long)(j + G.g[1]) * pitch +
                          (long long)G.g[2] * plane;
  // GATHER mode (guard fill O1 folded into the loads, as in the one-pass kernel): a position
  // outside the patch reads the image cell of the neighbour of class (ox,oy,oz) through the
  // neighbour table, so the guard shell in HBM is neither written nor read.  The column of a
  // thread crosses at most three patches along z: one base each.
  long long cb0 = cbase, cbm = cbase, cbp = cbase;
  if (gather && rowok) {
    const int ox = i < 0 ? -1 : (i >= nx ? 1 : 0), oy = j < 0 ? -1 : (j >= ny ? 1 : 0);
    const long long inner = G.lead + (i - ox * nx + G.g[0]) + (long long)(j - oy * ny + G.g[1]) * pitch + (long long)G.g[2] * plane;
    const int* tb = nbr + (long long)P.patch(pl) * 27 + (oy + 1) * 3 + (ox + 1);
    cbm = (long long)tb[0] * G.ps + inner + (long long)nz * plane;
    cb0 = (long long)tb[9] * G.ps + inner;
    cbp = (long long)tb[18] * G.ps + inner - (long long)nz * plane;
  }
  auto at = [&](int rr) { return (rr < 0 ? cbm : (rr >= nz ? cbp : cb0)) + (long long)rr * plane; };
  const T h = T(0.5), q4 = T(0.25);
  const T dt = P.dt_of(pl, dtp), hdt = h * dt;
  const T lx = hdt * P.idx[0], ly = hdt * P.idx[1], lz = hdt * P.idx[2];
  const int lim = G.limiter;

  const bool qpos = rowok && (pc <= PW - 2) && (pr <= PH - 2) && (j + 1 + G.g[1] < G.m[1]);
  const bool epos = qpos && (pc >= 1) && (pr >= 1);
  const bool dpos = inpos && (pc >= 1) && (pc <= nx + 2) && (j >= ya) && (j <= yb);
  const bool countpos = inpos && (i >= 0) && (i < nx) && (j >= y0) && (j < y0 + rows);

  auto Qs = [&](int plane_, int f) { return Q + (((plane_ + 3) % 3) * 8 + f) * PA; };
  auto Bs = [&](int plane_, int a) { return QB + (((plane_ + 3) % 3) * 3 + a) * PA; };
  auto Es = [&](int plane_, int a) { return E + (((plane_ + 2) & 1) * 3 + a) * PA; };

  // Own-column registers.  The state of plane r is loaded at the top of iteration r but its
  // hydro part is first used in iteration r+1 and its bx, by after the first barrier, so the
  // loads overlap a whole iteration; only bz is needed at once and runs one plane ahead.
  // Every global load is issued at least one full iteration before its first use: the
  // hydro part of plane r is used in iteration r+1 (as Uprev); bx, by of plane r are used in
  // iteration r (shared-memory write), so they are loaded in iteration r-1; bz of plane r is
  // used at the top of iteration r, so it runs two planes ahead.
  T Ucur[8], Uprev[8];
  T bxm[3] = {T(0), T(0), T(0)}, bym[3] = {T(0), T(0), T(0)};   // own raw bx, by at planes r-1, r-2, r-3
  T bxn = T(0), byn = T(0), bzn1 = T(0), bzn2 = T(0);
#pragma unroll
  for (int f = 0; f < 8; ++f) { Ucur[f] = T(0); Uprev[f] = T(0); }
  const int rlo = -2, rhi = nz + 2;
  if (rowok) {
    bxn = P.U[5 * fs + at(rlo)];
    byn = P.U[6 * fs + at(rlo)];
    bzn1 = P.U[7 * fs + at(rlo)];
    bzn2 = P.U[7 * fs + at(rlo + 1)];
  }
  unsigned int nbad = 0;

  for (int r = rlo; r <= rhi; ++r) {
    Ucur[5] = bxn; Ucur[6] = byn; Ucur[7] = bzn1; bzn1 = bzn2;
    if (rowok) {
      const long long cr = at(r);
#pragma unroll
      for (int f = 0; f < 5; ++f) Ucur[f] = P.U[f * fs + cr];
      if (r + 1 <= rhi) {
        const long long c1 = at(r + 1);
        bxn = P.U[5 * fs + c1];
        byn = P.U[6 * fs + c1];
      }
      if (r + 2 <= rhi) bzn2 = P.U[7 * fs + at(r + 2)];
    }

    // ---- primitives of plane r-1 (O2): needs bx(i+1), by(j+1) of plane r-1 and bz of plane r
    if (r - 1 >= rlo && qpos) {
      const T rho = Uprev[0], ir = num<T>::rcp(rho);
      const T u = Uprev[1] * ir, v = Uprev[2] * ir, w = Uprev[3] * ir;
      const T bcx = h * (Uprev[5] + Bs(r - 1, 0)[o + 1]);
      const T bcy = h * (Uprev[6] + Bs(r - 1, 1)[o + PW]);
      const T bcz = h * (Uprev[7] + Ucur[7]);
      const T pr_ = (P.gamma - T(1)) * (Uprev[4] - h * rho * (u * u + v * v + w * w) - h * (bcx * bcx + bcy * bcy + bcz * bcz));
      T* q = Qs(r - 1, 0) + o;
      q[0] = rho; q[PA] = u; q[2 * PA] = v; q[3 * PA] = w; q[4 * PA] = pr_; q[5 * PA] = bcx; q[6 * PA] = bcy; q[7 * PA] = bcz;
      if (countpos && r - 1 >= 0 && r - 1 < nz && !(rho > T(0) && pr_ > T(0) && rho < T(INFINITY) && pr_ < T(INFINITY))) ++nbad;
    }
    __syncthreads();

    // ---- edge EMFs of plane r-1 (O4a: Eq. 7-11 and cyclic images); raw fields of plane r
    if (r - 2 >= rlo && epos) {
      const T *u1 = Qs(r - 1, 1) + o, *v1 = Qs(r - 1, 2) + o, *w1 = Qs(r - 1, 3) + o;
      const T *u2 = Qs(r - 2, 1) + o, *v2 = Qs(r - 2, 2) + o, *w2 = Qs(r - 2, 3) + o;
      const T *bx1 = Bs(r - 1, 0) + o, *by1 = Bs(r - 1, 1) + o, *bz1 = Bs(r - 1, 2) + o;
      {  // ez over cells (i-1..i, j-1..j)
        const T ub = q4 * (u1[0] + u1[-PW] + u1[-1] + u1[-PW - 1]);
        const T vb = q4 * (v1[0] + v1[-PW] + v1[-1] + v1[-PW - 1]);
        Es(r - 1, 2)[o] = ub * (h * (by1[0] + by1[-1])) - vb * (h * (bx1[0] + bx1[-PW]));
      }
      {  // ex over (j-1..j, k-1..k)
        const T vb = q4 * (v1[0] + v2[0] + v1[-PW] + v2[-PW]);
        const T wb = q4 * (w1[0] + w2[0] + w1[-PW] + w2[-PW]);
        Es(r - 1, 0)[o] = vb * (h * (bz1[0] + bz1[-PW])) - wb * (h * (by1[0] + bym[1]));
      }
      {  // ey over (k-1..k, i-1..i)
        const T wb = q4 * (w1[0] + w1[-1] + w2[0] + w2[-1]);
        const T ub = q4 * (u1[0] + u1[-1] + u2[0] + u2[-1]);
        Es(r - 1, 1)[o] = wb * (h * (bx1[0] + bxm[1])) - ub * (h * (bz1[0] + bz1[-1]));
      }
    }
    if (inpos) { Bs(r, 0)[o] = Ucur[5]; Bs(r, 1)[o] = Ucur[6]; Bs(r, 2)[o] = Ucur[7]; }
    __syncthreads();

    // ---- D data of plane kd = r-2
    const int kd = r - 2;
    if (kd >= -1 && dpos) {
      const T* qc = Qs(kd, 0) + o;
      const T* qm = Qs(kd - 1, 0) + o;
      const T* qp = Qs(kd + 1, 0) + o;
      T* D = P.D + (long long)pl * P.DG.ps + (i + 1) + (long long)(j + 1) * P.DG.pitch +
             (long long)(kd + 1) * P.DG.pitch * P.DG.ny;
      const long long dfs = P.DG.fs;
      T c[8];
#pragma unroll
      for (int f = 0; f < 8; ++f) c[f] = qc[f * PA];
      // slopes (O3) and the primitive half step (O4c), one direction at a time: every term of
      // the predictor that involves direction d needs only the slopes along d
      const T rho = c[0], p_ = c[4], ir = num<T>::rcp(rho);
      const T lam[3] = {lx, ly, lz};
      T rho_h = rho, p_h = p_, vh[3] = {c[1], c[2], c[3]};
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        T dq[8];
#pragma unroll
        for (int f = 0; f < 8; ++f) {
          if (f == 5 + d) { dq[f] = T(0); continue; }
          const T lo = d == 0 ? qc[f * PA - 1] : (d == 1 ? qc[f * PA - PW] : qm[f * PA]);
          const T hi = d == 0 ? qc[f * PA + 1] : (d == 1 ? qc[f * PA + PW] : qp[f * PA]);
          dq[f] = limited_slope(lim, c[f] - lo, hi - c[f]);
          D[(long long)dq_slot(d, f) * dfs] = dq[f];
        }
        const int b = (d + 1) % 3, e = (d + 2) % 3;
        const T ud = c[1 + d], dud = dq[1 + d];
        rho_h -= lam[d] * (ud * dq[0] + rho * dud);
        p_h -= lam[d] * (ud * dq[4] + P.gamma * p_ * dud);
#pragma unroll
        for (int a = 0; a < 3; ++a) vh[a] -= lam[d] * ud * dq[1 + a];
        // -(1/rho) d_d (p + B_b^2/2 + B_e^2/2) acts on u_d;  +(B_d/rho) d_d B_a acts on u_a, a != d
        vh[d] -= lam[d] * (dq[4] + c[5 + b] * dq[5 + b] + c[5 + e] * dq[5 + e]) * ir;
        vh[b] += lam[d] * c[5 + d] * dq[5 + b] * ir;
        vh[e] += lam[d] * c[5 + d] * dq[5 + e] * ir;
      }
      const T *bx = Bs(kd, 0) + o, *by = Bs(kd, 1) + o, *bz = Bs(kd, 2) + o;
      const T bxc = bx[0], byc = by[0], bzc = bz[0];
      const T bxu = Bs(kd + 1, 0)[o], byu = Bs(kd + 1, 1)[o];   // own raw fields one plane up
      // face-field transverse slopes: dy bx, dz bx, dx by, dz by, dx bz, dy bz
      T db[6];
      db[0] = limited_slope(lim, bxc - bx[-PW], bx[PW] - bxc);
      db[1] = limited_slope(lim, bxc - bxm[2], bxu - bxc);
      db[2] = limited_slope(lim, byc - by[-1], by[1] - byc);
      db[3] = limited_slope(lim, byc - bym[2], byu - byc);
      db[4] = limited_slope(lim, bzc - bz[-1], bz[1] - bzc);
      db[5] = limited_slope(lim, bzc - bz[-PW], bz[PW] - bzc);
      // half-step faces (Eq. 12 with dt/2) of this cell and of its +x, +y, +z neighbours
      const T *ex0 = Es(kd, 0) + o, *ey0 = Es(kd, 1) + o, *ez0 = Es(kd, 2) + o;
      const T *ex1 = Es(kd + 1, 0) + o, *ey1 = Es(kd + 1, 1) + o;
      auto bxh_at = [&](int d) { return bx[d] + (ly * (ez0[d + PW] - ez0[d]) - lz * (ey1[d] - ey0[d])); };
      auto byh_at = [&](int d) { return by[d] + (lz * (ex1[d] - ex0[d]) - lx * (ez0[d + 1] - ez0[d])); };
      const T bxh = bxh_at(0), byh = byh_at(0);
      const T bzh = bzc + (lx * (ey0[1] - ey0[0]) - ly * (ex0[PW] - ex0[0]));
      const T bzu = Bs(kd + 1, 2)[o];
      const T bzh_up = bzu + (lx * (ey1[1] - ey1[0]) - ly * (ex1[PW] - ex1[0]));
      const T bchx = h * (bxh + bxh_at(1)), bchy = h * (byh + byh_at(PW)), bchz = h * (bzh + bzh_up);
      D[(D_QH + 0) * dfs] = rho_h; D[(D_QH + 1) * dfs] = vh[0]; D[(D_QH + 2) * dfs] = vh[1]; D[(D_QH + 3) * dfs] = vh[2];
      D[(D_QH + 4) * dfs] = p_h;
      D[(D_BCH + 0) * dfs] = bchx; D[(D_BCH + 1) * dfs] = bchy; D[(D_BCH + 2) * dfs] = bchz;
      D[(D_BH + 0) * dfs] = bxh; D[(D_BH + 1) * dfs] = byh; D[(D_BH + 2) * dfs] = bzh;
#pragma unroll
      for (int a = 0; a < 6; ++a) D[(D_DBF + a) * dfs] = db[a];
    }
    // shift the own-column history
    bxm[2] = bxm[1]; bxm[1] = bxm[0]; bxm[0] = Ucur[5];
    bym[2] = bym[1]; bym[1] = bym[0]; bym[0] = Ucur[6];
#pragma unroll
    for (int f = 0; f < 8; ++f) Uprev[f] = Ucur[f];
  }
  if (nbad) atomicAdd(bad, (unsigned long long)nbad);
}

// interim producer of the D block from the staged predictor's arrays (until the fused
// predictor writes W_D directly): D[a] = W[d_source(a)], D_BCH = mean of the two half-step faces
template <typename T>
__global__ void __launch_bounds__(256) k_pack_d(Params<T> P, Box B) {
  const Geom& G = P.G;
  int pl, i, j, k; long long c;
  if (!decode(G, B, P.npl, (long long)blockIdx.x * blockDim.x + threadIdx.x, pl, i, j, k, c)) return;
  const long long cw = (long long)pl * G.ps + c, wfs = P.wfs;
  T* D = P.D + (long long)pl * P.DG.ps + (i + 1) + (long long)(j + 1) * P.DG.pitch + (long long)(k + 1) * P.DG.pitch * P.DG.ny;
#pragma unroll
  for (int a = 0; a < D_COUNT; ++a) {
    if (a >= D_BCH && a < D_BH) {
      const T* bh = P.W + (W_BH + (a - D_BCH)) * wfs + cw;
      D[a * P.DG.fs] = T(0.5) * (bh[0] + bh[G.s[a - D_BCH]]);
    } else {
      D[a * P.DG.fs] = P.W[(long long)d_source(a) * wfs + cw];
    }
  }
}

// two CTAs per SM where two tiles' planes fit in shared memory (fp32 32x8), one otherwise (fp64 16x16)
template <typename T, int TXM, int TYM>
__global__ void __launch_bounds__(FusedCfg<T, TXM, TYM>::NTH, (FusedCfg<T, TXM, TYM>::smem > 116 * 1024) ? 1 : 2)
k_riemann_update(Params<T> P, const __grid_constant__ CUtensorMap tmap, const double* __restrict__ dtp, int xtiles) {
  using C = FusedCfg<T, TXM, TYM>;
  constexpr int DC = C::DC, DW = C::DW, NTH = C::NTH;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  T* X = reinterpret_cast<T*>(smem_raw + 2 * C::slot_stride);                 // [XV][NTH]  +y exchange
  T* XCs = X + C::XV * NTH;                                                   // [XC][XR]   closing column
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + 2 * C::slot_stride + sizeof(T) * (C::XV * NTH + C::XC * C::XR));

  const Geom& G = P.G;
  const int nx = G.n[0], ny = G.n[1], nz = G.n[2];
  const int pl = blockIdx.y;
  const int xt = blockIdx.x % xtiles, yt = blockIdx.x / xtiles;
  const int x0 = xt * TXM, y0 = yt * TYM;
  const int tw = min(TXM, nx - x0), th = min(TYM, ny - y0);
  const int t = threadIdx.x;
  const bool colthr = t >= C::CB;                       // closing-column warp
  const int fj = colthr ? t - C::CB : t / TXM;
  const int fi = colthr ? TXM : t - fj * TXM;
  const bool active = (fi <= tw) && (fj <= th) && (colthr ? fj < C::FH : t < TXM * C::FH);
  const int ty = colthr ? t + 1 : t + TXM;              // thread that owns (fi, fj+1)
  const long long pitch = G.pitch, plane = (long long)G.pitch * G.m[1];
  const T dt = P.dt_of(pl, dtp);
  const T cx = dt * P.idx[0], cy = dt * P.idx[1], cz = dt * P.idx[2];
  const T gamma = P.gamma;
  const int solver = G.emf_solver, fsolver = G.flux_solver;

  // D-block coordinates of the tile's first cell (i = x0-1, j = y0-1): cell -1 sits at 0, so
  // the start column x0 is a multiple of TXM and the box start is 16-byte aligned (TMA)
  const int tc0 = x0, tc1 = y0;
  auto slot = [&](int s) { return reinterpret_cast<T*>(smem_raw + (size_t)s * C::slot_stride); };
  auto issue = [&](int k, int s) {   // one thread: plane k of the D block -> slot s
    mbar_arrive_expect_tx(&bar[s], C::slot_bytes);
    tma_load_5d(slot(s), &tmap, &bar[s], tc0, tc1, k + 1, pl, 0);
  };

  if (t == 0) {
    mbar_init(&bar[0], 1);
    mbar_init(&bar[1], 1);
    fence_mbar_init();
  }
  __syncthreads();
  if (t == 0) {
    issue(-1, 0);
    issue(0, 1);
  }
  uint32_t phase[2] = {0u, 0u};

  // own cell inside the tile: row fj+1, column fi+1
  const int own = (fj + 1) * DW + (fi + 1);
  // state offset of cell (x0+fi, y0+fj, k=0)
  const long long ubase = (long long)P.patch(pl) * G.ps + G.lead + (x0 + fi + G.g[0]) +
                          (long long)(y0 + fj + G.g[1]) * pitch + (long long)G.g[2] * plane;
  const bool cell = (fi < tw) && (fj < th);
  const bool lastx = (x0 + tw == nx), lasty = (y0 + th == ny);

  Flux5<T> pFx = {}, pFy = {}, pFz = {};
  T pez = T(0), pex = T(0), pey = T(0);

  for (int k = 0; k <= nz + 1; ++k) {
    const int cur = (k + 1) & 1, prv = cur ^ 1;
    if (k <= nz) {
      if (k == 0) { mbar_wait(&bar[prv], phase[prv]); phase[prv] ^= 1u; }
      mbar_wait(&bar[cur], phase[cur]);
      phase[cur] ^= 1u;
    }
    const T* dc_ = slot(cur) + own;   // this cell, plane k
    const T* dp_ = slot(prv) + own;   // this cell, plane k-1
    if (k >= 1 && active) {
      // pull the U^n lines of plane k-1 towards L2 now: they are read after phase [A], and no
      // registers can be spared to hold them across it
      const T* up = P.U + ubase + (long long)(k - 1) * plane;
#pragma unroll
      for (int f = 0; f < 8; ++f) asm volatile("prefetch.global.L2 [%0];" ::"l"(up + f * G.fs));
    }

    // [A] values that couple planes k-1 and k: z-face flux and the x- and y-directed edges
    Flux5<T> cFz = {};
    T cex = T(0), cey = T(0);
    if (k <= nz && active) {
      cFz = face_flux<T, DC, 2>(dp_, dc_, gamma, fsolver);
      // ex: in-plane (y,z): sw=(j-1,k-1) se=(j,k-1) nw=(j-1,k) ne=(j,k)
      cex = edge_emf<T, DC, 0>(dp_ - DW, dp_, dc_ - DW, dc_, gamma, solver);
      // ey: in-plane (z,x): sw=(k-1,i-1) se=(k,i-1) nw=(k-1,i) ne=(k,i)
      cey = edge_emf<T, DC, 1>(dp_ - 1, dc_ - 1, dp_, dc_, gamma, solver);
    }

    // [B] exchange of the previous plane's in-plane values: the +x neighbour is the next lane
    // (warp shuffle; the closing column hands its values over through XCs), the +y neighbour
    // goes through X in two passes.  Barrier 1 also marks the point where every thread is
    // done with slot prv (plane k-1), so the next plane can be prefetched into it.
    Flux5<T> xF = {}, yF = {};
    T xez = T(0), xey = T(0), yez = T(0), yex = T(0);
    T un[8];
#pragma unroll
    for (int f = 0; f < 8; ++f) un[f] = T(0);
    if (k >= 1) {
      // U^n of the cell this thread updates: issued here so the loads fly during the exchange
      const long long cu = ubase + (long long)(k - 1) * plane;
      const long long fs = G.fs;
      if (k - 1 < nz) {
        if (cell) {
#pragma unroll
          for (int f = 0; f < 5; ++f) un[f] = P.U[f * fs + cu];
        }
        if (fj < th && (fi < tw || (fi == tw && lastx))) un[5] = P.U[5 * fs + cu];
        if (fi < tw && (fj < th || (fj == th && lasty))) un[6] = P.U[6 * fs + cu];
      }
      if (cell) un[7] = P.U[7 * fs + cu];
      if (colthr && fj < C::XR) {
        XCs[0 * C::XR + fj] = pFx.d; XCs[1 * C::XR + fj] = pFx.mu; XCs[2 * C::XR + fj] = pFx.mv; XCs[3 * C::XR + fj] = pFx.mw;
        XCs[4 * C::XR + fj] = pFx.e; XCs[5 * C::XR + fj] = pez;    XCs[6 * C::XR + fj] = pey;
      }
    }
    // +y exchange: 7 values in passes of XV through X; pass 0 is written before barrier 1
    const T sendv[7] = {pFy.d, pFy.mu, pFy.mv, pFy.mw, pFy.e, pez, pex};
    T recv[7] = {T(0), T(0), T(0), T(0), T(0), T(0), T(0)};
    constexpr int NPASS = (7 + C::XV - 1) / C::XV;
    if (k >= 1) {
#pragma unroll
      for (int v = 0; v < C::XV; ++v) X[v * NTH + t] = sendv[v];
    }
    __syncthreads();                                                   // barrier 1
    if (t == 0 && k + 1 <= nz) issue(k + 1, prv);   // prefetch plane k+1 while [B] and [C] run
    if (k >= 1) {
      xF.d = __shfl_down_sync(0xffffffffu, pFx.d, 1);   xF.mu = __shfl_down_sync(0xffffffffu, pFx.mu, 1);
      xF.mv = __shfl_down_sync(0xffffffffu, pFx.mv, 1); xF.mw = __shfl_down_sync(0xffffffffu, pFx.mw, 1);
      xF.e = __shfl_down_sync(0xffffffffu, pFx.e, 1);
      xez = __shfl_down_sync(0xffffffffu, pez, 1);      xey = __shfl_down_sync(0xffffffffu, pey, 1);
      if (!colthr && fi == TXM - 1 && fj < C::XR) {       // the +x neighbour is the closing column
        xF.d = XCs[0 * C::XR + fj]; xF.mu = XCs[1 * C::XR + fj]; xF.mv = XCs[2 * C::XR + fj]; xF.mw = XCs[3 * C::XR + fj];
        xF.e = XCs[4 * C::XR + fj]; xez = XCs[5 * C::XR + fj];   xey = XCs[6 * C::XR + fj];
      }
      const bool ynb = (fj < th) && active;
#pragma unroll
      for (int ps = 0; ps < NPASS; ++ps) {
        if (ps > 0) {
#pragma unroll
          for (int v = 0; v < C::XV; ++v)
            if (ps * C::XV + v < 7) X[v * NTH + t] = sendv[ps * C::XV + v];
          __syncthreads();
        }
        if (ynb) {
#pragma unroll
          for (int v = 0; v < C::XV; ++v)
            if (ps * C::XV + v < 7) recv[ps * C::XV + v] = X[v * NTH + ty];
        }
        __syncthreads();
      }
      yF.d = recv[0]; yF.mu = recv[1]; yF.mv = recv[2]; yF.mw = recv[3]; yF.e = recv[4]; yez = recv[5]; yex = recv[6];

      // update of plane k-1
      const long long cu = ubase + (long long)(k - 1) * plane;
      const long long fs = G.fs;
      if (k - 1 < nz) {
        if (cell) {
          // O8: U - dt * sum_d (F_d(c+e_d) - F_d(c)) / dx_d
          P.Un[cu] = un[0] - cx * (xF.d - pFx.d) - cy * (yF.d - pFy.d) - cz * (cFz.d - pFz.d);
          // momentum components are stored by solver frame: x-face (mu,mv,mw)=(mx,my,mz);
          // y-face (mu,mv,mw)=(my,mz,mx); z-face (mu,mv,mw)=(mz,mx,my)
          P.Un[fs + cu] = un[1] - cx * (xF.mu - pFx.mu) - cy * (yF.mw - pFy.mw) - cz * (cFz.mv - pFz.mv);
          P.Un[2 * fs + cu] = un[2] - cx * (xF.mv - pFx.mv) - cy * (yF.mu - pFy.mu) - cz * (cFz.mw - pFz.mw);
          P.Un[3 * fs + cu] = un[3] - cx * (xF.mw - pFx.mw) - cy * (yF.mv - pFy.mv) - cz * (cFz.mu - pFz.mu);
          P.Un[4 * fs + cu] = un[4] - cx * (xF.e - pFx.e) - cy * (yF.e - pFy.e) - cz * (cFz.e - pFz.e);
        }
        // Eq. 12 with the metric factor of each term (L154)
        if (fj < th && (fi < tw || (fi == tw && lastx)))       // bx on faces x0..x0+tw (closing face at the patch end)
          P.Un[5 * fs + cu] = un[5] + (cy * (yez - pez) - cz * (cey - pey));
        if (fi < tw && (fj < th || (fj == th && lasty)))
          P.Un[6 * fs + cu] = un[6] + (cz * (cex - pex) - cx * (xez - pez));
      }
      if (cell)                                                 // bz on faces 0..nz (k-1 == nz: closing face)
        P.Un[7 * fs + cu] = un[7] + (cx * (xey - pey) - cy * (yex - pex));
    }

    // [C] in-plane values of plane k become the "previous" set of the next iteration
    if (k <= nz && active) {
      pFx = face_flux<T, DC, 0>(dc_ - 1, dc_, gamma, fsolver);
      pFy = face_flux<T, DC, 1>(dc_ - DW, dc_, gamma, fsolver);
      // ez: in-plane (x,y): sw=(i-1,j-1) se=(i,j-1) nw=(i-1,j) ne=(i,j)
      pez = edge_emf<T, DC, 2>(dc_ - DW - 1, dc_ - DW, dc_ - 1, dc_, gamma, solver);
    }
    pFz = cFz; pex = cex; pey = cey;
  }
}

}  // namespace mhd
