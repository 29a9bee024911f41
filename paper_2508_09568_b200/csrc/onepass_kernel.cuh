// onepass_kernel.cuh -- the whole step of a 3D bunch in ONE kernel (section 2.1.4,
// L108-116): primitives, limited slopes, time-n edge EMFs (Eq. 7-11), half-step predictor
// (Eq. 12 with dt/2), face and corner states, HLLD at faces, the 2D Riemann problem at
// edges, conservative + constrained-transport update (Eq. 12).  HBM traffic is
// the compulsory one: U^n is read once per tile (with its halo), U^{n+1} written once;
// nothing intermediate ever leaves the SM.
//
// A CTA owns an (x,y) tile of one patch and marches along z.  Its warps are specialised
// into three roles that run concurrently and hand data over through shared memory with
// named barriers (bar.sync / bar.arrive), so that the issue slots of the SM stay busy:
//
//   P  predictor   U^n planes arrive by 16-byte asynchronous copies (cp.async) into a ring of
//                  raw planes.  In GATHER mode the halo of a plane is read straight from
//                  the interiors of the neighbouring patches through the neighbour table
//                  (guard fill O1 folded into the load: PAPER.md L124, L188, L241), so the
//                  guard shell in HBM is neither written nor read; otherwise the patch's
//                  own (already filled) guard cells are read.  P forms primitives, edge
//                  EMFs, slopes and the half step and writes the "D data" of one plane
//                  (38 arrays, see fused_kernels.cuh) into one of two shared-memory slots.
//   A  z-coupled   reads D planes k-1 and k: HLLD at the z-face, 2D Riemann problems at the
//                  x- and y-directed edges; finishes the update of plane k-1 and of b_z.
//   C  in-plane    reads D plane k: HLLD at the x- and y-faces, 2D Riemann problem at the
//                  z-directed edge; hands the partial update (U^n - dt*(dFx/dx + dFy/dy)) to A.
//
// A releases the older D slot as soon as it has pulled the 29 state values it needs from
// it into registers, so the predictor of plane k+1 overlaps the solves of plane k.
#pragma once
#include "bunch_types.cuh"
#include "mhd_math.cuh"
#include "tma_utils.cuh"
#include "fused_kernels.cuh"

namespace mhd {

__device__ __forceinline__ void nb_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void nb_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }
// 16-byte asynchronous copy global -> shared (L2 only), and the wait for all of a thread's copies
__device__ __forceinline__ void cp_async16(void* dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

template <typename T, int TX, int TY, int NPW> struct OneCfg {
  static constexpr int PW = TX + 5, PH = TY + 5, PA = PW * PH;     // predictor positions: cells x0-2.., y0-2..
  static constexpr int BWX = TX + 8, RA = BWX * PH;                // raw box: columns x0-4.. (16-byte aligned start)
  static constexpr int DW = TX + 2, DH = TY + 2, DC = DW * DH;     // D cells: x0-1.., y0-1..
  static constexpr int FW = TX + 1, FH = TY + 1, FA = FW * FH;     // faces / edges
  static constexpr int CB = ((TX * FH + 31) / 32) * 32;            // first thread of the closing-column warp
  static constexpr int NR = CB + 32;                               // threads of role A and of role C
  static constexpr int NP = NPW * 32;                              // threads of role P
  static constexpr int NTH = 2 * NR + NP;
  static constexpr int NALL = NTH;
  // compact index spaces of the predictor passes: primitives on columns 0..PW-2 and rows
  // 0..PH-2, edge EMFs on columns 1..PW-2 and rows 1..PH-2, D cells
  static constexpr int W1 = PW - 1, N1 = W1 * (PH - 1), W2 = PW - 2, N2 = W2 * (PH - 2);
  static constexpr int PASS1 = (N1 + NP - 1) / NP, PASS2 = (N2 + NP - 1) / NP, PASS3 = (DC + NP - 1) / NP;
  static_assert(FH <= 32 && 32 % TX == 0, "tile shape");
  static constexpr size_t al(size_t x) { return (x + 127) / 128 * 128; }
  // shared-memory map (bytes)
  static constexpr size_t rawh_slot = al(sizeof(T) * 5 * RA), rawb_slot = al(sizeof(T) * 3 * RA);
  static constexpr size_t o_rawh = 0;                                  // [2] hydro planes (TMA destinations)
  static constexpr size_t o_rawb = o_rawh + 2 * rawh_slot;             // [4] field planes (TMA destinations)
  static constexpr size_t o_d = o_rawb + 4 * rawb_slot;                // [2][38][DC]
  static constexpr size_t o_q = o_d + al(sizeof(T) * 2 * D_COUNT * DC);   // [3][8][PA]
  static constexpr size_t o_e = o_q + al(sizeof(T) * 3 * 8 * PA);      // [2][3][PA]
  static constexpr size_t o_pu = o_e + al(sizeof(T) * 2 * 3 * PA);     // [7][FA]   C -> A partial update
  static constexpr size_t o_xe = o_pu + al(sizeof(T) * 7 * FA);        // [2][NR]   A: ex, ey of the neighbours
  static constexpr size_t o_xy = o_xe + al(sizeof(T) * 2 * NR);        // [6][NR]   C: +y exchange
  static constexpr size_t o_xc = o_xy + al(sizeof(T) * 6 * NR);        // [6][32]   C: closing column -> column TX-1
  static constexpr size_t o_nb = o_xc + al(sizeof(T) * 6 * 32);        // [27] source patch per neighbour class
  static constexpr size_t smem = o_nb + 128;
  static constexpr int VEC = 16 / sizeof(T), CPR = BWX / VEC;          // elements per 16-byte copy, copies per row
  static_assert(BWX % VEC == 0, "raw rows are whole 16-byte chunks");
};

// named barrier ids (0 is __syncthreads)
enum : int { NB_FULL = 1, NB_EMPTY = 3, NB_PUF = 5, NB_PUE = 6, NB_P = 7, NB_A = 8, NB_C = 9 };

// face state of cell c along D: q^h + s*dq  (s = +1/2: upper face, left state of the next
// face; s = -1/2: lower face, right state) -- O5
template <typename T, int DC, int D>
__device__ __forceinline__ State1D<T> face_state(const T* __restrict__ c, T s) {
  constexpr int T1 = (D + 1) % 3, T2 = (D + 2) % 3;
  State1D<T> q;
  q.rho = c[(D_QH + 0) * DC] + s * c[dq_slot(D, 0) * DC];
  q.u = c[(D_QH + 1 + D) * DC] + s * c[dq_slot(D, 1 + D) * DC];
  q.v = c[(D_QH + 1 + T1) * DC] + s * c[dq_slot(D, 1 + T1) * DC];
  q.w = c[(D_QH + 1 + T2) * DC] + s * c[dq_slot(D, 1 + T2) * DC];
  q.p = c[(D_QH + 4) * DC] + s * c[dq_slot(D, 4) * DC];
  q.by = c[(D_BCH + T1) * DC] + s * c[dq_slot(D, 5 + T1) * DC];
  q.bz = c[(D_BCH + T2) * DC] + s * c[dq_slot(D, 5 + T2) * DC];
  return q;
}
// corner state of cell c seen from the edge along E: q^h + sa*d_A q + sb*d_B q
template <typename T, int DC, int E>
__device__ __forceinline__ Corner<T> corner_state(const T* __restrict__ c, T sa, T sb) {
  constexpr int A = (E + 1) % 3, B = (E + 2) % 3;
  Corner<T> q;
  q.rho = c[(D_QH + 0) * DC] + sa * c[dq_slot(A, 0) * DC] + sb * c[dq_slot(B, 0) * DC];
  q.ua = c[(D_QH + 1 + A) * DC] + sa * c[dq_slot(A, 1 + A) * DC] + sb * c[dq_slot(B, 1 + A) * DC];
  q.ub = c[(D_QH + 1 + B) * DC] + sa * c[dq_slot(A, 1 + B) * DC] + sb * c[dq_slot(B, 1 + B) * DC];
  q.p = c[(D_QH + 4) * DC] + sa * c[dq_slot(A, 4) * DC] + sb * c[dq_slot(B, 4) * DC];
  q.be = c[(D_BCH + E) * DC] + sa * c[dq_slot(A, 5 + E) * DC] + sb * c[dq_slot(B, 5 + E) * DC];
  return q;
}
// D slot of the slope of face field b_a along t (a != t)
__host__ __device__ constexpr int dbf_slot(int a, int t) {
  return D_DBF + (a == 0 ? (t == 1 ? 0 : 1) : (a == 1 ? (t == 0 ? 2 : 3) : (t == 0 ? 4 : 5)));
}
// in-plane field of the edge along E on the side of cell c: component X (A or B of the edge),
// extrapolated along the other in-plane direction with sign s
template <typename T, int DC, int X, int ALONG>
__device__ __forceinline__ T edge_field(const T* __restrict__ c, T s) {
  return c[(D_BH + X) * DC] + s * c[dbf_slot(X, ALONG) * DC];
}

template <typename T, int TX, int TY, int NPW, int LIM, int FS>
__global__ void __launch_bounds__(OneCfg<T, TX, TY, NPW>::NTH, 1)
k_step_onepass(Params<T> P, const int* __restrict__ nbr, int gather, const double* __restrict__ dtp,
               unsigned long long* __restrict__ bad, int xtiles, int zseg) {
  using C = OneCfg<T, TX, TY, NPW>;
  constexpr int PW = C::PW, PH = C::PH, PA = C::PA, BWX = C::BWX, RA = C::RA, DW = C::DW, DC = C::DC;
  constexpr int FW = C::FW, FA = C::FA, NR = C::NR, NP = C::NP, NALL = C::NALL;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  T* const Dm = reinterpret_cast<T*>(smem_raw + C::o_d);
  T* const Q = reinterpret_cast<T*>(smem_raw + C::o_q);
  T* const Em = reinterpret_cast<T*>(smem_raw + C::o_e);
  T* const PU = reinterpret_cast<T*>(smem_raw + C::o_pu);
  T* const XE = reinterpret_cast<T*>(smem_raw + C::o_xe);
  T* const XY = reinterpret_cast<T*>(smem_raw + C::o_xy);
  T* const XC = reinterpret_cast<T*>(smem_raw + C::o_xc);
  int* const NBS = reinterpret_cast<int*>(smem_raw + C::o_nb);

  const Geom& G = P.G;
  const int nx = G.n[0], ny = G.n[1], nz = G.n[2];
  // Small bunches have fewer tiles than the GPU has SMs; their columns are then cut into zseg
  // segments along z (blockIdx.z), each a CTA of its own that marches planes [za, zb) after a
  // five-plane run-in through its lower neighbour's planes.  zseg == 1: za = 0, zb = nz.
  const int zlen = (nz + zseg - 1) / zseg;
  const int za = (int)blockIdx.z * zlen, zb = min(nz, za + zlen);
  const int pl = blockIdx.y;
  const int xt = blockIdx.x % xtiles, yt = blockIdx.x / xtiles;
  const int x0 = xt * TX, y0 = yt * TY;
  const int tw = min(TX, nx - x0), th = min(TY, ny - y0);
  const bool lastx = (x0 + tw == nx), lasty = (y0 + th == ny);
  const int t = threadIdx.x;
  const T h = T(0.5);
  const T dt = (T)(*dtp);
  const T gamma = P.gamma;

  // source patch of each of the 27 neighbour classes: the neighbour table in gather mode,
  // the patch itself (whose guard cells are then read) otherwise
  if (t < 27) NBS[t] = gather ? nbr[(long long)(P.p0 + pl) * 27 + t] : P.p0 + pl;
  __syncthreads();

  auto dslot = [&](int plane) { return Dm + (size_t)((plane + 2) & 1) * (D_COUNT * DC); };

  if (t >= 2 * NR) {
    // =============================================================== role P ==========
    const int tp = t - 2 * NR;
    const T q4 = T(0.25), hdt = h * dt;
    const T lx = hdt * P.idx[0], ly = hdt * P.idx[1], lz = hdt * P.idx[2];
    auto Qs = [&](int plane, int f) { return Q + (((plane + 3) % 3) * 8 + f) * PA; };
    auto Es = [&](int plane, int a) { return Em + (((plane + 2) & 1) * 3 + a) * PA; };
    auto RH = [&](int plane) { return reinterpret_cast<const T*>(smem_raw + C::o_rawh + (size_t)((plane + 2) & 1) * C::rawh_slot); };
    auto RB = [&](int plane) { return reinterpret_cast<const T*>(smem_raw + C::o_rawb + (size_t)((plane + 4) & 3) * C::rawb_slot); };
    const int rlo = za - 2, rhi = zb + 2;
    // U^n plane -> raw ring, one 16-byte chunk of a row per copy, all 8 fields.  A chunk lies
    // in one patch (x0 and, in gather mode, n_x are multiples of the chunk); its source is
    // the image cell in the neighbour of class (ox,oy,oz) -- O1 -- or, without gather, the
    // same cell of the own patch.  Chunks past the data a tile needs are skipped.
    auto issue = [&](int plane) {
      const long long zplane = (long long)G.pitch * G.m[1];
      const int oz = gather ? (plane < 0 ? -1 : (plane >= nz ? 1 : 0)) : 0;
      const long long zoff = (long long)(plane - oz * nz + G.g[2]) * zplane;
      T* const dh = const_cast<T*>(RH(plane));
      T* const db = const_cast<T*>(RB(plane));
      for (int it = tp; it < PH * C::CPR; it += NP) {
        const int row = it / C::CPR, ch = it - row * C::CPR;
        const int x = x0 - 4 + ch * C::VEC, y = y0 - 2 + row;   // first cell of the chunk (raw column 0 is cell x0-4)
        int ox = 0, oy = 0;
        if (gather) { ox = x < 0 ? -1 : (x >= nx ? 1 : 0); oy = y < 0 ? -1 : (y >= ny ? 1 : 0); }
        const int xs = x - ox * nx, ys = y - oy * ny;
        const bool ok = gather ? (xs + C::VEC <= nx && ys < ny && xs >= 0 && ys >= 0)
                               : (G.lead + G.g[0] + xs + C::VEC <= G.pitch && ys + G.g[1] < G.m[1]);
        if (!ok) continue;
        const int q = NBS[(oz + 1) * 9 + (oy + 1) * 3 + (ox + 1)];
        const T* src = P.U + (long long)q * G.ps + zoff + (long long)(ys + G.g[1]) * G.pitch + (G.lead + G.g[0] + xs);
        const int o = row * BWX + ch * C::VEC;
#pragma unroll
        for (int f = 0; f < 5; ++f) cp_async16(dh + f * RA + o, src + f * G.fs);
#pragma unroll
        for (int f = 0; f < 3; ++f) cp_async16(db + f * RA + o, src + (5 + f) * G.fs);
      }
    };
    issue(rlo);
    cp_async_wait_all();
    nb_sync(NB_P, NP);
    T cbx[C::PASS3], cby[C::PASS3];   // backward z-differences of the raw bx, by of the own D cells
#pragma unroll
    for (int s = 0; s < C::PASS3; ++s) { cbx[s] = T(0); cby[s] = T(0); }
    unsigned int nbad = 0;

    for (int r = rlo; r <= rhi; ++r) {
      // ---- primitives of plane r-1 (O2): needs bx(i+1), by(j+1) of plane r-1 and bz of plane r
      if (r - 1 >= rlo) {
        const T* hy = RH(r - 1);
        const T* bb = RB(r - 1);
        const T* bzu = RB(r) + 2 * RA;
#pragma unroll
        for (int s = 0; s < C::PASS1; ++s) {
          const int pos = tp + s * NP;
          const int pr = pos / C::W1, pc = pos - pr * C::W1;
          if (pos < C::N1) {
            const int o = pr * PW + pc, ob = pr * BWX + pc + 2;
            const T rho = hy[ob], ir = num<T>::rcp(rho);
            const T u = hy[RA + ob] * ir, v = hy[2 * RA + ob] * ir, w = hy[3 * RA + ob] * ir;
            const T bz0 = bb[2 * RA + ob];
            const T bcx = h * (bb[ob] + bb[ob + 1]);
            const T bcy = h * (bb[RA + ob] + bb[RA + ob + BWX]);
            const T bcz = h * (bz0 + bzu[ob]);
            const T pr_ = (gamma - T(1)) * (hy[4 * RA + ob] - h * rho * (u * u + v * v + w * w) - h * (bcx * bcx + bcy * bcy + bcz * bcz));
            T* q = Qs(r - 1, 0) + o;
            q[0] = rho; q[PA] = u; q[2 * PA] = v; q[3 * PA] = w; q[4 * PA] = pr_; q[5 * PA] = bcx; q[6 * PA] = bcy; q[7 * PA] = bcz;
            const int ci = pc - 2, cj = pr - 2;   // tile-relative cell
            if (ci >= 0 && ci < tw && cj >= 0 && cj < th && r - 1 >= za && r - 1 < zb &&
                !(rho > T(0) && pr_ > T(0) && rho < T(INFINITY) && pr_ < T(INFINITY)))
              ++nbad;
          }
        }
      }
      nb_sync(NB_P, NP);
      // every P thread is past iteration r-1: the slots of hydro plane r-1 and field plane r-3 are free
      if (r + 1 <= rhi) issue(r + 1);

      // ---- edge EMFs of plane r-1 (O4a: Eq. 7-11 and cyclic images)
      if (r - 2 >= rlo) {
        const T* b1 = RB(r - 1);
        const T* b2 = RB(r - 2);
#pragma unroll
        for (int s = 0; s < C::PASS2; ++s) {
          const int pos = tp + s * NP;
          const int pr = pos / C::W2 + 1, pc = pos - (pr - 1) * C::W2 + 1;
          if (pos < C::N2) {
            const int o = pr * PW + pc, ob = pr * BWX + pc + 2;
            const T *u1 = Qs(r - 1, 1) + o, *v1 = Qs(r - 1, 2) + o, *w1 = Qs(r - 1, 3) + o;
            const T *u2 = Qs(r - 2, 1) + o, *v2 = Qs(r - 2, 2) + o, *w2 = Qs(r - 2, 3) + o;
            const T *bx1 = b1 + ob, *by1 = b1 + RA + ob, *bz1 = b1 + 2 * RA + ob;
            {  // ez over cells (i-1..i, j-1..j)
              const T ub = q4 * (u1[0] + u1[-PW] + u1[-1] + u1[-PW - 1]);
              const T vb = q4 * (v1[0] + v1[-PW] + v1[-1] + v1[-PW - 1]);
              Es(r - 1, 2)[o] = ub * (h * (by1[0] + by1[-1])) - vb * (h * (bx1[0] + bx1[-BWX]));
            }
            {  // ex over (j-1..j, k-1..k)
              const T vb = q4 * (v1[0] + v2[0] + v1[-PW] + v2[-PW]);
              const T wb = q4 * (w1[0] + w2[0] + w1[-PW] + w2[-PW]);
              Es(r - 1, 0)[o] = vb * (h * (bz1[0] + bz1[-BWX])) - wb * (h * (by1[0] + b2[RA + ob]));
            }
            {  // ey over (k-1..k, i-1..i)
              const T wb = q4 * (w1[0] + w1[-1] + w2[0] + w2[-1]);
              const T ub = q4 * (u1[0] + u1[-1] + u2[0] + u2[-1]);
              Es(r - 1, 1)[o] = wb * (h * (bx1[0] + b2[ob])) - ub * (h * (bz1[0] + bz1[-1]));
            }
          }
        }
      }
      nb_sync(NB_P, NP);

      // ---- D data of plane kd = r-2 -> shared slot
      const int kd = r - 2;
      if (kd >= rlo) {
        T* const Dw = dslot(kd);
        if (kd >= za + 1) nb_sync(NB_EMPTY + ((kd + 2) & 1), NALL);   // A and C are done with plane kd-2
        const T* b0 = RB(kd);
        const T* b1 = RB(kd + 1);
#pragma unroll
        for (int s = 0; s < C::PASS3; ++s) {
          const int dcell = tp + s * NP;
          if (dcell < DC) {
            const int dr = dcell / DW, dcl = dcell - dr * DW;
            const int o = (dr + 1) * PW + dcl + 1, ob = (dr + 1) * BWX + dcl + 3;
            const T *bx = b0 + ob, *by = b0 + RA + ob, *bz = b0 + 2 * RA + ob;
            const T bxc = bx[0], byc = by[0], bzc = bz[0];
            const T bxu = b1[ob], byu = b1[RA + ob], bzu = b1[2 * RA + ob];   // raw fields one plane up
            const T fwx = bxu - bxc, fwy = byu - byc;
            if (kd >= za - 1) {
              const T* qc = Qs(kd, 0) + o;
              const T* qm = Qs(kd - 1, 0) + o;
              const T* qp = Qs(kd + 1, 0) + o;
              T* D = Dw + dcell;
              T c[8];
#pragma unroll
              for (int f = 0; f < 8; ++f) c[f] = qc[f * PA];
              // slopes (O3) and the primitive half step (O4c), one direction at a time
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
                  dq[f] = limited_slope_k<LIM>(c[f] - lo, hi - c[f]);
                  D[dq_slot(d, f) * DC] = dq[f];
                }
                const int b = (d + 1) % 3, e = (d + 2) % 3;
                const T ud = c[1 + d], dud = dq[1 + d];
                rho_h -= lam[d] * (ud * dq[0] + rho * dud);
                p_h -= lam[d] * (ud * dq[4] + gamma * p_ * dud);
#pragma unroll
                for (int a = 0; a < 3; ++a) vh[a] -= lam[d] * ud * dq[1 + a];
                // -(1/rho) d_d (p + B_b^2/2 + B_e^2/2) acts on u_d;  +(B_d/rho) d_d B_a acts on u_a, a != d
                vh[d] -= lam[d] * (dq[4] + c[5 + b] * dq[5 + b] + c[5 + e] * dq[5 + e]) * ir;
                vh[b] += lam[d] * c[5 + d] * dq[5 + b] * ir;
                vh[e] += lam[d] * c[5 + d] * dq[5 + e] * ir;
              }
              // face-field transverse slopes: dy bx, dz bx, dx by, dz by, dx bz, dy bz
              D[(D_DBF + 0) * DC] = limited_slope_k<LIM>(bxc - bx[-BWX], bx[BWX] - bxc);
              D[(D_DBF + 1) * DC] = limited_slope_k<LIM>(cbx[s], fwx);
              D[(D_DBF + 2) * DC] = limited_slope_k<LIM>(byc - by[-1], by[1] - byc);
              D[(D_DBF + 3) * DC] = limited_slope_k<LIM>(cby[s], fwy);
              D[(D_DBF + 4) * DC] = limited_slope_k<LIM>(bzc - bz[-1], bz[1] - bzc);
              D[(D_DBF + 5) * DC] = limited_slope_k<LIM>(bzc - bz[-BWX], bz[BWX] - bzc);
              // half-step faces (Eq. 12 with dt/2) of this cell and of its +x, +y, +z neighbours
              const T *ex0 = Es(kd, 0) + o, *ey0 = Es(kd, 1) + o, *ez0 = Es(kd, 2) + o;
              const T *ex1 = Es(kd + 1, 0) + o, *ey1 = Es(kd + 1, 1) + o;
              const T bxh = bxc + (ly * (ez0[PW] - ez0[0]) - lz * (ey1[0] - ey0[0]));
              const T bxh1 = bx[1] + (ly * (ez0[1 + PW] - ez0[1]) - lz * (ey1[1] - ey0[1]));
              const T byh = byc + (lz * (ex1[0] - ex0[0]) - lx * (ez0[1] - ez0[0]));
              const T byh1 = by[BWX] + (lz * (ex1[PW] - ex0[PW]) - lx * (ez0[PW + 1] - ez0[PW]));
              const T bzh = bzc + (lx * (ey0[1] - ey0[0]) - ly * (ex0[PW] - ex0[0]));
              const T bzh_up = bzu + (lx * (ey1[1] - ey1[0]) - ly * (ex1[PW] - ex1[0]));
              D[(D_QH + 0) * DC] = rho_h; D[(D_QH + 1) * DC] = vh[0]; D[(D_QH + 2) * DC] = vh[1]; D[(D_QH + 3) * DC] = vh[2];
              D[(D_QH + 4) * DC] = p_h;
              D[(D_BCH + 0) * DC] = h * (bxh + bxh1); D[(D_BCH + 1) * DC] = h * (byh + byh1); D[(D_BCH + 2) * DC] = h * (bzh + bzh_up);
              D[(D_BH + 0) * DC] = bxh; D[(D_BH + 1) * DC] = byh; D[(D_BH + 2) * DC] = bzh;
            }
            cbx[s] = fwx; cby[s] = fwy;
          }
        }
        if (kd >= za - 1) {
          __threadfence_block();
          nb_arrive(NB_FULL + ((kd + 2) & 1), NALL);
        }
      }
      cp_async_wait_all();   // own chunks of plane r+1 have landed ...
      nb_sync(NB_P, NP);     // ... and everybody's; the rings are rewritten by the next iteration
    }
    if (nbad) atomicAdd(bad, (unsigned long long)nbad);
    return;
  }

  // =========================================================== roles A and C ==========
  const bool roleA = t < NR;
  const int tr = roleA ? t : t - NR;
  const bool colthr = tr >= C::CB;                        // closing-column warp
  const int fj = colthr ? tr - C::CB : tr / TX;
  const int fi = colthr ? TX : tr - fj * TX;
  const bool valid = colthr ? (fj < C::FH) : (tr < TX * C::FH);
  const bool active = valid && (fi <= tw) && (fj <= th);
  const bool cell = active && (fi < tw) && (fj < th);
  const bool xface = active && (fj < th) && (fi < tw || lastx);   // bx faces of the tile (closing face at the patch end)
  const bool yface = active && (fi < tw) && (fj < th || lasty);
  const int own = (fj + 1) * DW + (fi + 1);
  const int fidx = min(fj, C::FH - 1) * FW + fi;
  const int tyn = colthr ? tr + 1 : tr + TX;              // thread that owns (fi, fj+1)
  const int txn = colthr ? tr : ((fi == TX - 1) ? C::CB + fj : tr + 1);   // thread that owns (fi+1, fj)
  const long long plane = (long long)G.pitch * G.m[1], fs = G.fs;
  const long long ubase = (long long)(P.p0 + pl) * G.ps + G.lead + (x0 + fi + G.g[0]) +
                          (long long)(y0 + fj + G.g[1]) * G.pitch + (long long)G.g[2] * plane;
  const T cx = dt * P.idx[0], cy = dt * P.idx[1], cz = dt * P.idx[2];
  const int solver = G.emf_solver;

  if (roleA) {
    // ------------------------------------------------------------- role A -----------
    const bool doFz = cell;
    const bool doEx = active && (fi < tw);      // ex(i, j..j+1): by faces and b_z
    const bool doEy = active && (fj < th);      // ey(i..i+1, j): bx faces and b_z
    Flux5<T> pFz = {};
    T pex = T(0), pey = T(0);
    nb_sync(NB_FULL + ((za + 1) & 1), NALL);    // plane za-1
    for (int k = za; k <= zb; ++k) {
      nb_sync(NB_FULL + ((k + 2) & 1), NALL);   // plane k
      const T* dp_ = dslot(k - 1) + own;
      const T* dc_ = dslot(k) + own;
      T u7 = T(0);
      if (cell) u7 = P.U[7 * fs + ubase + (long long)k * plane];
      // everything this thread needs from plane k-1, then the slot goes back to the predictor
      State1D<T> Lz = {};
      Corner<T> xsw = {}, xse = {}, ysw = {}, ynw = {};
      T xAS = T(0), yBW = T(0);
      if (doFz) Lz = face_state<T, DC, 2>(dp_, h);
      if (doEx) {   // ex, in-plane (y,z): sw=(j-1,k-1) se=(j,k-1) nw=(j-1,k) ne=(j,k)
        xsw = corner_state<T, DC, 0>(dp_ - DW, h, h);
        xse = corner_state<T, DC, 0>(dp_, -h, h);
        xAS = edge_field<T, DC, 1, 2>(dp_, h);
      }
      if (doEy) {   // ey, in-plane (z,x): sw=(k-1,i-1) se=(k,i-1) nw=(k-1,i) ne=(k,i)
        ysw = corner_state<T, DC, 1>(dp_ - 1, h, h);
        ynw = corner_state<T, DC, 1>(dp_, h, -h);
        yBW = edge_field<T, DC, 0, 2>(dp_, h);
      }
      if (k + 1 <= zb) nb_arrive(NB_EMPTY + ((k + 1) & 1), NALL);   // slot of plane k-1

      Flux5<T> cFz = {};
      T cex = T(0), cey = T(0);
      if (doFz) cFz = riemann_flux_k<FS>(gamma, Lz, face_state<T, DC, 2>(dc_, -h), dc_[(D_BH + 2) * DC]);
      // The hydro part of plane k-1 only waits for this flux: finish it now (C is ahead, its
      // partial update is normally there already), so that the previous plane's flux is dead
      // while the two edge problems are solved.
      const long long cu = ubase + (long long)(k - 1) * plane;
      const T* pu = PU + fidx;
      if (k >= za + 1) {
        nb_sync(NB_PUF, 2 * NR);
        if (cell) {
          // O8: (U - dt*dFx/dx - dt*dFy/dy) - dt*dFz/dz; z-face frame (mu,mv,mw) = (mz,mx,my)
          P.Un[cu] = pu[0] - cz * (cFz.d - pFz.d);
          P.Un[fs + cu] = pu[FA] - cz * (cFz.mv - pFz.mv);
          P.Un[2 * fs + cu] = pu[2 * FA] - cz * (cFz.mw - pFz.mw);
          P.Un[3 * fs + cu] = pu[3 * FA] - cz * (cFz.mu - pFz.mu);
          P.Un[4 * fs + cu] = pu[4 * FA] - cz * (cFz.e - pFz.e);
        }
      }
      pFz = cFz;
      if (doEx)
        cex = emf_2d(gamma, solver, xsw, xse, corner_state<T, DC, 0>(dc_ - DW, h, -h), corner_state<T, DC, 0>(dc_, -h, -h),
                     xAS, edge_field<T, DC, 1, 2>(dc_, -h), edge_field<T, DC, 2, 1>(dc_ - DW, h), edge_field<T, DC, 2, 1>(dc_, -h));
      if (doEy)
        cey = emf_2d(gamma, solver, ysw, corner_state<T, DC, 1>(dc_ - 1, -h, h), ynw, corner_state<T, DC, 1>(dc_, -h, -h),
                     edge_field<T, DC, 2, 0>(dc_ - 1, h), edge_field<T, DC, 2, 0>(dc_, -h), yBW, edge_field<T, DC, 0, 2>(dc_, -h));

      XE[tr] = cex;
      XE[NR + tr] = cey;
      nb_sync(NB_A, NR);
      const T yex = XE[tyn], xey = XE[NR + txn];
      // b_z on the lower z-face of plane k (k = nz: closing face) -- Eq. 12
      // (face zb belongs to the next segment unless it is the patch's closing face)
      if (cell && (k < zb || zb == nz)) P.Un[7 * fs + ubase + (long long)k * plane] = u7 + (cx * (xey - cey) - cy * (yex - cex));
      if (k >= za + 1) {
        if (xface) P.Un[5 * fs + cu] = pu[5 * FA] - cz * (cey - pey);
        if (yface) P.Un[6 * fs + cu] = pu[6 * FA] + cz * (cex - pex);
        if (k <= zb - 1) nb_arrive(NB_PUE, 2 * NR);
      }
      pex = cex; pey = cey;
    }
    return;
  }

  // --------------------------------------------------------------- role C -----------
  {
    const bool doFx = active && (fj < th);
    const bool doFy = active && (fi < tw);
    for (int kd = za - 1; kd <= zb; ++kd) {
      nb_sync(NB_FULL + ((kd + 2) & 1), NALL);
      const bool work = (kd >= za) && (kd <= zb - 1);
      Flux5<T> Fx = {}, Fy = {};
      T ez = T(0);
      T un[7];
#pragma unroll
      for (int f = 0; f < 7; ++f) un[f] = T(0);
      if (work) {
        const long long cu = ubase + (long long)kd * plane;
        if (cell) {
#pragma unroll
          for (int f = 0; f < 5; ++f) un[f] = P.U[f * fs + cu];
        }
        if (xface) un[5] = P.U[5 * fs + cu];
        if (yface) un[6] = P.U[6 * fs + cu];
        const T* dc_ = dslot(kd) + own;
        if (doFx) Fx = riemann_flux_k<FS>(gamma, face_state<T, DC, 0>(dc_ - 1, h), face_state<T, DC, 0>(dc_, -h), dc_[(D_BH + 0) * DC]);
        if (doFy) Fy = riemann_flux_k<FS>(gamma, face_state<T, DC, 1>(dc_ - DW, h), face_state<T, DC, 1>(dc_, -h), dc_[(D_BH + 1) * DC]);
        if (active)   // ez, in-plane (x,y): sw=(i-1,j-1) se=(i,j-1) nw=(i-1,j) ne=(i,j)
          ez = emf_2d(gamma, solver, corner_state<T, DC, 2>(dc_ - DW - 1, h, h), corner_state<T, DC, 2>(dc_ - DW, -h, h),
                      corner_state<T, DC, 2>(dc_ - 1, h, -h), corner_state<T, DC, 2>(dc_, -h, -h),
                      edge_field<T, DC, 0, 1>(dc_ - DW, h), edge_field<T, DC, 0, 1>(dc_, -h),
                      edge_field<T, DC, 1, 0>(dc_ - 1, h), edge_field<T, DC, 1, 0>(dc_, -h));
      }
      if (kd + 2 <= zb) nb_arrive(NB_EMPTY + ((kd + 2) & 1), NALL);   // done with plane kd
      if (!work) continue;

      // neighbours: +x by warp shuffle (the closing column hands its values over through XC),
      // +y through XY
      XY[tr] = Fy.d; XY[NR + tr] = Fy.mu; XY[2 * NR + tr] = Fy.mv; XY[3 * NR + tr] = Fy.mw; XY[4 * NR + tr] = Fy.e;
      XY[5 * NR + tr] = ez;
      if (colthr) {
        XC[fj] = Fx.d; XC[32 + fj] = Fx.mu; XC[2 * 32 + fj] = Fx.mv; XC[3 * 32 + fj] = Fx.mw; XC[4 * 32 + fj] = Fx.e;
        XC[5 * 32 + fj] = ez;
      }
      nb_sync(NB_C, NR);
      Flux5<T> xF, yF;
      xF.d = __shfl_down_sync(0xffffffffu, Fx.d, 1);   xF.mu = __shfl_down_sync(0xffffffffu, Fx.mu, 1);
      xF.mv = __shfl_down_sync(0xffffffffu, Fx.mv, 1); xF.mw = __shfl_down_sync(0xffffffffu, Fx.mw, 1);
      xF.e = __shfl_down_sync(0xffffffffu, Fx.e, 1);
      T xez = __shfl_down_sync(0xffffffffu, ez, 1);
      if (!colthr && fi == TX - 1) {
        const int cj = min(fj, 31);
        xF.d = XC[cj]; xF.mu = XC[32 + cj]; xF.mv = XC[2 * 32 + cj]; xF.mw = XC[3 * 32 + cj]; xF.e = XC[4 * 32 + cj];
        xez = XC[5 * 32 + cj];
      }
      const int ty_ = min(tyn, NR - 1);
      yF.d = XY[ty_]; yF.mu = XY[NR + ty_]; yF.mv = XY[2 * NR + ty_]; yF.mw = XY[3 * NR + ty_]; yF.e = XY[4 * NR + ty_];
      const T yez = XY[5 * NR + ty_];

      if (kd >= za + 1) nb_sync(NB_PUE, 2 * NR);   // A has consumed the previous plane
      T* pu = PU + fidx;
      if (cell) {
        // momentum components by solver frame: x-face (mu,mv,mw)=(mx,my,mz); y-face (mu,mv,mw)=(my,mz,mx)
        pu[0] = un[0] - cx * (xF.d - Fx.d) - cy * (yF.d - Fy.d);
        pu[FA] = un[1] - cx * (xF.mu - Fx.mu) - cy * (yF.mw - Fy.mw);
        pu[2 * FA] = un[2] - cx * (xF.mv - Fx.mv) - cy * (yF.mu - Fy.mu);
        pu[3 * FA] = un[3] - cx * (xF.mw - Fx.mw) - cy * (yF.mv - Fy.mv);
        pu[4 * FA] = un[4] - cx * (xF.e - Fx.e) - cy * (yF.e - Fy.e);
      }
      if (xface) pu[5 * FA] = un[5] + cy * (yez - ez);
      if (yface) pu[6 * FA] = un[6] - cx * (xez - ez);
      __threadfence_block();
      nb_arrive(NB_PUF, 2 * NR);
    }
  }
}

}  // namespace mhd
