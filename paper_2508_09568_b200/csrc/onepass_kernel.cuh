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

// Named barriers.  bar.sync / bar.arrive are the .aligned forms: they ASSERT that the whole warp
// executes them together, and ptxas uses that assertion -- seen in SASS: it merged the convergence
// region of a lane-divergent `if` with the enclosing one whose end lay after a bar.arrive, and
// dropped the __syncwarp() in front of it as redundant; the warp then arrived twice, the barrier
// count drifted and the CTA hung.  (The non-aligned barrier.sync / barrier.arrive are safe but make
// the kernel 5 % slower.)  The rules that keep the aligned forms sound here:
//   * a barrier is never nested in an `if`: conditional ones are PREDICATED instructions
//     (nb_sync_if / nb_arrive_if) at the top level of the role's plane loop, so no convergence
//     region can span them;
//   * the predictor passes keep the lanes of a warp together (tasks are clamped, not skipped);
//   * tests/test_abi_cpu.py disassembles the library and fails if a named barrier lies inside any
//     convergence region (BSSY ... BSYNC).
__device__ __forceinline__ void nb_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void nb_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void nb_sync_if(bool c, int id, int n) {
  asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.s32 p, %0, 0;\n\t@p bar.sync %1, %2;\n\t}" ::"r"((int)c), "r"(id), "r"(n) : "memory");
}
__device__ __forceinline__ void nb_arrive_if(bool c, int id, int n) {
  asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.s32 p, %0, 0;\n\t@p bar.arrive %1, %2;\n\t}" ::"r"((int)c), "r"(id), "r"(n) : "memory");
}
// 16-byte asynchronous copy global -> shared (L2 only), and the wait for all of a thread's copies
__device__ __forceinline__ void cp_async16(void* dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// two consecutive elements moved by one 8-byte (float) or 16-byte (double) shared-memory access
template <typename T> struct Pair;
template <> struct Pair<float> { using V = float2; };
template <> struct Pair<double> { using V = double2; };
template <typename T> struct V2 { T a, b; };
template <typename T> __device__ __forceinline__ V2<T> ld2(const T* p) {
  const typename Pair<T>::V v = *reinterpret_cast<const typename Pair<T>::V*>(p);
  return V2<T>{v.x, v.y};
}
template <typename T> __device__ __forceinline__ void st2(T* p, T a, T b) {
  typename Pair<T>::V v;
  v.x = a; v.y = b;
  *reinterpret_cast<typename Pair<T>::V*>(p) = v;
}

// Geometry of a tile.  Every plane array of the predictor (raw U^n, primitives, time-n EMFs) has
// PH rows of BWX columns; column rc holds cell x0-4+rc (so that 16-byte chunks of a state row land
// on 16-byte boundaries), row pr holds y0-2+pr.  Predictor threads work on STRIPS of two
// consecutive columns (rc = 2s, 2s+1; 8/16-byte shared accesses, x-differences shared between the
// two cells).  The D arrays handed to the solver roles hold cells rc = 3..TX+4 (x0-1..x0+TX),
// rows dr = pr-1 = 0..TY+1, at index dr*DP + rc with DP = TX+4: columns 0..2 of a row are unused,
// and the strip stores that overhang the row on either side (rc = 2, rc = TX+5) fall into those
// unused slots of this row and the next one.
template <typename T, int TX, int TY, int NPW> struct OneCfg {
  static constexpr int PH = TY + 5;
  static constexpr int BWX = TX + 8, RA = BWX * PH;
  static constexpr int DP = TX + 4, DH = TY + 2, DCS = DH * DP + 4;   // D arrays: row pitch, rows, elements per array
  static constexpr int FW = TX + 1, FH = TY + 1, FA = FW * FH;     // faces / edges
  static constexpr int CB = ((TX * FH + 31) / 32) * 32;            // first thread of the closing-column warp
  static constexpr int NR = CB + 32;                               // threads of role A and of role C
  static constexpr int NP = NPW * 32;                              // threads of role P
  static constexpr int NTH = 2 * NR + NP;
  static constexpr int NALL = NTH;
  // strips s = 1..NS cover rc = 2..TX+5; tasks of the three predictor passes: primitives on rows
  // 0..PH-2, edge EMFs on rows 1..PH-2, D cells on rows 1..PH-3
  static constexpr int NS = (TX + 4) / 2;
  static constexpr int NT1 = NS * (PH - 1), NT2 = NS * (PH - 2), NT3 = NS * (PH - 3);
  static constexpr int PASS1 = (NT1 + NP - 1) / NP, PASS2 = (NT2 + NP - 1) / NP, PASS3 = (NT3 + NP - 1) / NP;
  static_assert(FH <= 32 && 32 % TX == 0 && TX % 4 == 0, "tile shape");
  static constexpr size_t al(size_t x) { return (x + 127) / 128 * 128; }
  // shared-memory map (bytes)
  static constexpr size_t rawh_slot = al(sizeof(T) * 5 * RA), rawb_slot = al(sizeof(T) * 3 * RA);
  static constexpr size_t o_rawh = 0;                                  // [1] hydro plane (cp.async destination)
  static constexpr size_t o_rawb = o_rawh + rawh_slot;                 // [4] field planes (cp.async destinations)
  static constexpr size_t o_d = o_rawb + 4 * rawb_slot;                // [2][38][DCS]
  static constexpr size_t o_q = o_d + al(sizeof(T) * 2 * D_COUNT * DCS);  // [3][8][RA]
  static constexpr size_t o_e = o_q + al(sizeof(T) * 3 * 8 * RA);      // [2][3][RA]
  static constexpr size_t o_pu = o_e + al(sizeof(T) * 2 * 3 * RA);     // [8][FA]   C -> A partial update; A -> C new values (CFL)
  static constexpr size_t o_xe = o_pu + al(sizeof(T) * 8 * FA);        // [2][NR]   A: ex, ey of the neighbours
  static constexpr size_t o_xy = o_xe + al(sizeof(T) * 2 * NR);        // [6][NR]   C: +y exchange
  static constexpr size_t o_xc = o_xy + al(sizeof(T) * 6 * NR);        // [6][32]   C: closing column -> column TX-1
  static constexpr size_t o_nb = o_xc + al(sizeof(T) * 6 * 32);        // [27] source patch per neighbour class
  static constexpr size_t smem = o_nb + 128;
  static_assert(smem <= 227 * 1024, "shared memory of one CTA");
  static constexpr int VEC = 16 / sizeof(T), CPR = BWX / VEC;          // elements per 16-byte copy, copies per row
  static_assert(BWX % VEC == 0, "raw rows are whole 16-byte chunks");
};

// named barrier ids (0 is __syncthreads)
enum : int { NB_FULL = 1, NB_EMPTY = 3, NB_PUF = 5, NB_PUE = 6, NB_P = 7, NB_A = 8, NB_C = 9 };

// face state of cell c along D: q^h + s*dq  (s = +1/2: upper face, left state of the next
// face; s = -1/2: lower face, right state) -- O5
template <typename T, int DCS, int D>
__device__ __forceinline__ State1D<T> face_state(const T* __restrict__ c, T s) {
  constexpr int T1 = (D + 1) % 3, T2 = (D + 2) % 3;
  State1D<T> q;
  q.rho = c[(D_QH + 0) * DCS] + s * c[dq_slot(D, 0) * DCS];
  q.u = c[(D_QH + 1 + D) * DCS] + s * c[dq_slot(D, 1 + D) * DCS];
  q.v = c[(D_QH + 1 + T1) * DCS] + s * c[dq_slot(D, 1 + T1) * DCS];
  q.w = c[(D_QH + 1 + T2) * DCS] + s * c[dq_slot(D, 1 + T2) * DCS];
  q.p = c[(D_QH + 4) * DCS] + s * c[dq_slot(D, 4) * DCS];
  q.by = c[(D_BCH + T1) * DCS] + s * c[dq_slot(D, 5 + T1) * DCS];
  q.bz = c[(D_BCH + T2) * DCS] + s * c[dq_slot(D, 5 + T2) * DCS];
  return q;
}
// corner state of cell c seen from the edge along E: q^h + sa*d_A q + sb*d_B q
template <typename T, int DCS, int E>
__device__ __forceinline__ Corner<T> corner_state(const T* __restrict__ c, T sa, T sb) {
  constexpr int A = (E + 1) % 3, B = (E + 2) % 3;
  Corner<T> q;
  q.rho = c[(D_QH + 0) * DCS] + sa * c[dq_slot(A, 0) * DCS] + sb * c[dq_slot(B, 0) * DCS];
  q.ua = c[(D_QH + 1 + A) * DCS] + sa * c[dq_slot(A, 1 + A) * DCS] + sb * c[dq_slot(B, 1 + A) * DCS];
  q.ub = c[(D_QH + 1 + B) * DCS] + sa * c[dq_slot(A, 1 + B) * DCS] + sb * c[dq_slot(B, 1 + B) * DCS];
  q.p = c[(D_QH + 4) * DCS] + sa * c[dq_slot(A, 4) * DCS] + sb * c[dq_slot(B, 4) * DCS];
  q.be = c[(D_BCH + E) * DCS] + sa * c[dq_slot(A, 5 + E) * DCS] + sb * c[dq_slot(B, 5 + E) * DCS];
  return q;
}
// D slot of the slope of face field b_a along t (a != t)
__host__ __device__ constexpr int dbf_slot(int a, int t) {
  return D_DBF + (a == 0 ? (t == 1 ? 0 : 1) : (a == 1 ? (t == 0 ? 2 : 3) : (t == 0 ? 4 : 5)));
}
// in-plane field of the edge along E on the side of cell c: component X (A or B of the edge),
// extrapolated along the other in-plane direction with sign s
template <typename T, int DCS, int X, int ALONG>
__device__ __forceinline__ T edge_field(const T* __restrict__ c, T s) {
  return c[(D_BH + X) * DCS] + s * c[dbf_slot(X, ALONG) * DCS];
}

// LIM: limiter (1 minmod, 2 monotonised central), fixed at compile time; CFLE: reduce the CFL rates
// of the new level in the epilogue (role C), so that mhd_bunch_cfl_dt has nothing left to read
// DEFS: the default solvers (HLLD at faces, HLLD-2D at edges) fixed at compile time instead of read from the
// descriptor (2 % faster; instantiated for the default limiter without the CFL epilogue only)
template <typename T, int TX, int TY, int NPW, int LIM, bool CFLE, bool DEFS = false>
__global__ void __launch_bounds__(OneCfg<T, TX, TY, NPW>::NTH, 1)
k_step_onepass(Params<T> P, const int* __restrict__ nbr, int gather, const double* __restrict__ dtp,
               unsigned long long* __restrict__ bad, unsigned long long* __restrict__ rate_next, int xtiles, int zseg,
               int zlo, int zhi) {
  using C = OneCfg<T, TX, TY, NPW>;
  constexpr int PH = C::PH, BWX = C::BWX, RA = C::RA, DP = C::DP, DCS = C::DCS;
  constexpr int FW = C::FW, FA = C::FA, NR = C::NR, NP = C::NP, NALL = C::NALL, NS = C::NS;
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
  // five-plane run-in through its lower neighbour's planes.  The launch covers planes [zlo, zhi) of
  // its patches (the whole column unless the host-streaming path steps a chunk band by band).
  const int zlen = (zhi - zlo + zseg - 1) / zseg;
  const int za = zlo + (int)blockIdx.z * zlen, zb = min(zhi, za + zlen);
  if (za >= zb) return;   // an empty segment (the host asks for none): the whole CTA leaves before any barrier
  const int pl = blockIdx.y;
  const int xt = blockIdx.x % xtiles, yt = blockIdx.x / xtiles;
  const int x0 = xt * TX, y0 = yt * TY;
  const int tw = min(TX, nx - x0), th = min(TY, ny - y0);
  const bool lastx = (x0 + tw == nx), lasty = (y0 + th == ny);
  const int t = threadIdx.x;
  const T h = T(0.5);
  const T dt = P.dt_of(pl, dtp);
  const T gamma = P.gamma;

  // source patch of each of the 27 neighbour classes: the neighbour table in gather mode,
  // the patch itself (whose guard cells are then read) otherwise
  if (t < 27) NBS[t] = gather ? nbr[(long long)P.patch(pl) * 27 + t] : P.patch(pl);
  __syncthreads();

  auto dslot = [&](int plane) { return Dm + (size_t)((plane + 2) & 1) * (D_COUNT * DCS); };

  // Warp ids decide issue priority on an SM sub-partition (the higher id wins a tie), so the order of
  // the roles in the thread index is a tuning knob: ROLE_ORDER 0 = A, C, P (P highest), 1 = P, C, A,
  // 2 = C, P, A, 3 = P, A, C, 4 = C, A, P, 5 = A, P, C
#ifndef ONEPASS_ROLE_ORDER
#define ONEPASS_ROLE_ORDER 0
#endif
  constexpr int RO = ONEPASS_ROLE_ORDER;
  constexpr int P0 = (RO == 0 || RO == 4) ? 2 * NR : ((RO == 1 || RO == 3) ? 0 : NR);
  constexpr int A0 = (RO == 0 || RO == 5) ? 0 : ((RO == 1 || RO == 2) ? NP + NR : ((RO == 3) ? NP : NR));
  constexpr int C0 = (RO == 2 || RO == 4) ? 0 : ((RO == 0) ? NR : ((RO == 1) ? NP : ((RO == 3) ? NP + NR : NR + NP)));
  if (t >= P0 && t < P0 + NP) {
    // =============================================================== role P ==========
    const int tp = t - P0;
    const T q4 = T(0.25), hdt = h * dt;
    const T lx = hdt * P.idx[0], ly = hdt * P.idx[1], lz = hdt * P.idx[2];
    const T gm1 = gamma - T(1);
    auto Qs = [&](int plane) { return Q + ((plane + 3) % 3) * (8 * RA); };              // [8][RA]
    auto Es = [&](int plane) { return Em + ((plane + 2) & 1) * (3 * RA); };             // [3][RA]
    T* const RHs = reinterpret_cast<T*>(smem_raw + C::o_rawh);                           // [5][RA], one plane
    auto RB = [&](int plane) { return reinterpret_cast<T*>(smem_raw + C::o_rawb + (size_t)((plane + 4) & 3) * C::rawb_slot); };
    const int rlo = za - 2, rhi = zb + 2;
    // U^n -> raw planes, one 16-byte chunk of a row per copy: the hydro fields of plane ph into the
    // single hydro slot, the face fields of plane pb into the field ring.  A chunk lies in one patch
    // (x0 and, in gather mode, n_x are multiples of the chunk); its source is the image cell in the
    // neighbour of class (ox,oy,oz) -- O1 -- or, without gather, the same cell of the own patch.
    // Chunks past the data a tile needs are skipped.
    auto issue = [&](int ph, int pb, bool with_h) {
      const long long zplane = (long long)G.pitch * G.m[1];
      const int ozh = gather ? (ph < 0 ? -1 : (ph >= nz ? 1 : 0)) : 0;
      const int ozb = gather ? (pb < 0 ? -1 : (pb >= nz ? 1 : 0)) : 0;
      const long long zoffh = (long long)(ph - ozh * nz + G.g[2]) * zplane;
      const long long zoffb = (long long)(pb - ozb * nz + G.g[2]) * zplane;
      T* const db = RB(pb);
      for (int it = tp; it < PH * C::CPR; it += NP) {
        const int row = it / C::CPR, ch = it - row * C::CPR;
        const int x = x0 - 4 + ch * C::VEC, y = y0 - 2 + row;   // first cell of the chunk (raw column 0 is cell x0-4)
        int ox = 0, oy = 0;
        if (gather) { ox = x < 0 ? -1 : (x >= nx ? 1 : 0); oy = y < 0 ? -1 : (y >= ny ? 1 : 0); }
        const int xs = x - ox * nx, ys = y - oy * ny;
        const bool ok = gather ? (xs + C::VEC <= nx && ys < ny && xs >= 0 && ys >= 0)
                               : (G.lead + G.g[0] + xs + C::VEC <= G.pitch && ys + G.g[1] < G.m[1]);
        if (!ok) continue;
        const int cls = (oy + 1) * 3 + (ox + 1);
        const long long inp = (long long)(ys + G.g[1]) * G.pitch + (G.lead + G.g[0] + xs);
        const int o = row * BWX + ch * C::VEC;
        const T* sb = P.U + (long long)NBS[(ozb + 1) * 9 + cls] * G.ps + zoffb + inp;
#pragma unroll
        for (int f = 0; f < 3; ++f) cp_async16(db + f * RA + o, sb + (5 + f) * G.fs);
        if (with_h) {
          const T* sh = P.U + (long long)NBS[(ozh + 1) * 9 + cls] * G.ps + zoffh + inp;
#pragma unroll
          for (int f = 0; f < 5; ++f) cp_async16(RHs + f * RA + o, sh + f * G.fs);
        }
      }
    };
    issue(rlo, rlo, false);
    cp_async_wait_all();
    nb_sync(NB_P, NP);
    // backward z-differences of the raw bx, by of the own D cells (carried from plane to plane)
    T cbx[C::PASS3][2], cby[C::PASS3][2];
#pragma unroll
    for (int s_ = 0; s_ < C::PASS3; ++s_) { cbx[s_][0] = cbx[s_][1] = T(0); cby[s_][0] = cby[s_][1] = T(0); }
    unsigned int nbad = 0;

    for (int r = rlo; r <= rhi; ++r) {
      // ---- primitives of plane r-1 (O2): needs bx(i+1), by(j+1) of plane r-1 and bz of plane r
      if (r - 1 >= rlo) {
        const T* bb = RB(r - 1);
        const T* bzu = RB(r) + 2 * RA;
        T* const qw = Qs(r - 1);
#pragma unroll
        for (int s_ = 0; s_ < C::PASS1; ++s_) {
          // a warp runs the body whole or not at all: lanes past the last task repeat it (same
          // values to the same addresses), so no lane leaves its warp before the next barrier
          if ((tp & ~31) + s_ * NP < C::NT1) {
            const bool mine = tp + s_ * NP < C::NT1;
            const int task = mine ? tp + s_ * NP : C::NT1 - 1;
            const int pr = task / NS, st = task - pr * NS + 1;
            const int o = pr * BWX + 2 * st;
            const V2<T> rho = ld2(RHs + o), mx = ld2(RHs + RA + o), my = ld2(RHs + 2 * RA + o), mz = ld2(RHs + 3 * RA + o);
            const V2<T> en = ld2(RHs + 4 * RA + o);
            const V2<T> bx = ld2(bb + o);
            const T bx2 = bb[o + 2];
            const V2<T> by = ld2(bb + RA + o), byn = ld2(bb + RA + o + BWX);
            const V2<T> bz = ld2(bb + 2 * RA + o), bzn = ld2(bzu + o);
            T pv[2][8];
            auto prim = [&](int e, T rh, T m0, T m1, T m2, T E, T bxa, T bxb, T bya, T byb, T bza, T bzb) {
              const T ir = num<T>::rcp(rh);
              const T u = m0 * ir, v = m1 * ir, w = m2 * ir;
              const T bcx = h * (bxa + bxb), bcy = h * (bya + byb), bcz = h * (bza + bzb);
              const T pr_ = gm1 * (E - h * rh * (u * u + v * v + w * w) - h * (bcx * bcx + bcy * bcy + bcz * bcz));
              pv[e][0] = rh; pv[e][1] = u; pv[e][2] = v; pv[e][3] = w; pv[e][4] = pr_; pv[e][5] = bcx; pv[e][6] = bcy; pv[e][7] = bcz;
              const int ci = 2 * st + e - 4, cj = pr - 2;   // tile-relative cell
              if (mine && ci >= 0 && ci < tw && cj >= 0 && cj < th && r - 1 >= za && r - 1 < zb &&
                  !(rh > T(0) && pr_ > T(0) && rh < T(INFINITY) && pr_ < T(INFINITY)))
                ++nbad;
            };
            prim(0, rho.a, mx.a, my.a, mz.a, en.a, bx.a, bx.b, by.a, byn.a, bz.a, bzn.a);
            prim(1, rho.b, mx.b, my.b, mz.b, en.b, bx.b, bx2, by.b, byn.b, bz.b, bzn.b);
#pragma unroll
            for (int f = 0; f < 8; ++f) st2(qw + f * RA + o, pv[0][f], pv[1][f]);
          }
        }
      }
      nb_sync(NB_P, NP);
      // every P thread is past the primitives of plane r-1: the hydro slot and the field slot of plane r-3 are free
      if (r + 1 <= rhi) issue(r, r + 1, true);

      // ---- edge EMFs of plane r-1 (O4a: Eq. 7-11 and cyclic images)
      if (r - 2 >= rlo) {
        const T* b1 = RB(r - 1);
        const T* b2 = RB(r - 2);
        const T *q1 = Qs(r - 1), *q2 = Qs(r - 2);
        T* const ew = Es(r - 1);
#pragma unroll
        for (int s_ = 0; s_ < C::PASS2; ++s_) {
          if ((tp & ~31) + s_ * NP < C::NT2) {
            const int task = min(tp + s_ * NP, C::NT2 - 1);
            const int pr = task / NS + 1, st = task - (pr - 1) * NS + 1;
            const int o = pr * BWX + 2 * st;
            // columns -1, 0, 1 relative to the strip's first cell; rows 0 and -1; planes 1 (r-1) and 2 (r-2)
            const T *u1 = q1 + RA + o, *v1 = q1 + 2 * RA + o, *w1 = q1 + 3 * RA + o;
            const T *u2 = q2 + RA + o, *v2 = q2 + 2 * RA + o, *w2 = q2 + 3 * RA + o;
            const T u1m = u1[-1], u1dm = u1[-BWX - 1];
            const V2<T> u1c = ld2(u1), u1d = ld2(u1 - BWX);
            const T v1m = v1[-1], v1dm = v1[-BWX - 1];
            const V2<T> v1c = ld2(v1), v1d = ld2(v1 - BWX);
            const T w1m = w1[-1];
            const V2<T> w1c = ld2(w1), w1d = ld2(w1 - BWX);
            const T u2m = u2[-1];
            const V2<T> u2c = ld2(u2);
            const V2<T> v2c = ld2(v2), v2d = ld2(v2 - BWX);
            const T w2m = w2[-1];
            const V2<T> w2c = ld2(w2), w2d = ld2(w2 - BWX);
            const V2<T> bx1c = ld2(b1 + o), bx1d = ld2(b1 + o - BWX), bx2c = ld2(b2 + o);
            const T by1m = b1[RA + o - 1];
            const V2<T> by1c = ld2(b1 + RA + o), by2c = ld2(b2 + RA + o);
            const T bz1m = b1[2 * RA + o - 1];
            const V2<T> bz1c = ld2(b1 + 2 * RA + o), bz1d = ld2(b1 + 2 * RA + o - BWX);
            // one position: own cell values X, west neighbour Xw (same row), row below Xd, its west Xdw
            auto emfs = [&](T u, T uw, T ud, T udw, T v, T vw, T vd, T vdw, T w, T ww, T wd, T uu2, T uu2w, T vv2, T vv2d,
                            T ww2, T ww2w, T ww2d, T bx, T bxd, T bxp, T by, T byw, T byp, T bz, T bzw, T bzd, T& ex, T& ey,
                            T& ez) {
              {  // ez over cells (i-1..i, j-1..j)
                const T ub = q4 * (u + ud + uw + udw);
                const T vb = q4 * (v + vd + vw + vdw);
                ez = ub * (h * (by + byw)) - vb * (h * (bx + bxd));
              }
              {  // ex over (j-1..j, k-1..k)
                const T vb = q4 * (v + vv2 + vd + vv2d);
                const T wb = q4 * (w + ww2 + wd + ww2d);
                ex = vb * (h * (bz + bzd)) - wb * (h * (by + byp));
              }
              {  // ey over (k-1..k, i-1..i)
                const T wb = q4 * (w + ww + ww2 + ww2w);
                const T ub = q4 * (u + uw + uu2 + uu2w);
                ey = wb * (h * (bx + bxp)) - ub * (h * (bz + bzw));
              }
            };
            T ex0, ey0, ez0, ex1, ey1, ez1;
            emfs(u1c.a, u1m, u1d.a, u1dm, v1c.a, v1m, v1d.a, v1dm, w1c.a, w1m, w1d.a, u2c.a, u2m, v2c.a, v2d.a, w2c.a, w2m, w2d.a,
                 bx1c.a, bx1d.a, bx2c.a, by1c.a, by1m, by2c.a, bz1c.a, bz1m, bz1d.a, ex0, ey0, ez0);
            emfs(u1c.b, u1c.a, u1d.b, u1d.a, v1c.b, v1c.a, v1d.b, v1d.a, w1c.b, w1c.a, w1d.b, u2c.b, u2c.a, v2c.b, v2d.b, w2c.b, w2c.a,
                 w2d.b, bx1c.b, bx1d.b, bx2c.b, by1c.b, by1c.a, by2c.b, bz1c.b, bz1c.a, bz1d.b, ex1, ey1, ez1);
            st2(ew + o, ex0, ex1);
            st2(ew + RA + o, ey0, ey1);
            st2(ew + 2 * RA + o, ez0, ez1);
          }
        }
      }
      nb_sync(NB_P, NP);

      // ---- D data of plane kd = r-2 -> shared slot
      const int kd = r - 2;
      nb_sync_if(kd >= rlo && kd >= za + 1, NB_EMPTY + ((kd + 2) & 1), NALL);   // A and C are done with plane kd-2
      if (kd >= rlo) {
        T* const Dw = dslot(kd);
        const T* b0 = RB(kd);
        const T* b1 = RB(kd + 1);
        const T *qc = Qs(kd), *qm = Qs(kd - 1), *qp = Qs(kd + 1);
        const T *e0 = Es(kd), *e1 = Es(kd + 1);
#pragma unroll
        for (int s_ = 0; s_ < C::PASS3; ++s_) {
          if ((tp & ~31) + s_ * NP < C::NT3) {
            const int task = min(tp + s_ * NP, C::NT3 - 1);
            const int dr = task / NS, st = task - dr * NS + 1;
            const int o = (dr + 1) * BWX + 2 * st;
            const V2<T> bxc = ld2(b0 + o), byc = ld2(b0 + RA + o), bzc = ld2(b0 + 2 * RA + o);
            const V2<T> bxu = ld2(b1 + o), byu = ld2(b1 + RA + o), bzu = ld2(b1 + 2 * RA + o);   // raw fields one plane up
            const T fwx[2] = {bxu.a - bxc.a, bxu.b - bxc.b}, fwy[2] = {byu.a - byc.a, byu.b - byc.b};
            if (kd >= za - 1) {
              T* D = Dw + dr * DP + 2 * st;
              T c[8][2];
#pragma unroll
              for (int f = 0; f < 8; ++f) { const V2<T> v = ld2(qc + f * RA + o); c[f][0] = v.a; c[f][1] = v.b; }
              // slopes (O3) and the primitive half step (O4c), one direction at a time
              const T lam[3] = {lx, ly, lz};
              T ir[2], rho_h[2], p_h[2], vh[3][2];
#pragma unroll
              for (int e = 0; e < 2; ++e) {
                ir[e] = num<T>::rcp(c[0][e]); rho_h[e] = c[0][e]; p_h[e] = c[4][e];
                vh[0][e] = c[1][e]; vh[1][e] = c[2][e]; vh[2][e] = c[3][e];
              }
#pragma unroll
              for (int d = 0; d < 3; ++d) {
                T dq[8][2];
#pragma unroll
                for (int f = 0; f < 8; ++f) {
                  if (f == 5 + d) { dq[f][0] = dq[f][1] = T(0); continue; }
                  const T* qf = qc + f * RA + o;
                  if (d == 0) {
                    const T lo = qf[-1], hi = qf[2];
                    const T d0 = c[f][0] - lo, d1 = c[f][1] - c[f][0], d2 = hi - c[f][1];
                    dq[f][0] = limited_slope_k<LIM>(d0, d1);
                    dq[f][1] = limited_slope_k<LIM>(d1, d2);
                  } else {
                    const V2<T> lo = d == 1 ? ld2(qf - BWX) : ld2(qm + f * RA + o);
                    const V2<T> hi = d == 1 ? ld2(qf + BWX) : ld2(qp + f * RA + o);
                    dq[f][0] = limited_slope_k<LIM>(c[f][0] - lo.a, hi.a - c[f][0]);
                    dq[f][1] = limited_slope_k<LIM>(c[f][1] - lo.b, hi.b - c[f][1]);
                  }
                  st2(D + dq_slot(d, f) * DCS, dq[f][0], dq[f][1]);
                }
                const int b = (d + 1) % 3, eb = (d + 2) % 3;
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                  const T ud = c[1 + d][e], dud = dq[1 + d][e];
                  rho_h[e] -= lam[d] * (ud * dq[0][e] + c[0][e] * dud);
                  p_h[e] -= lam[d] * (ud * dq[4][e] + gamma * c[4][e] * dud);
#pragma unroll
                  for (int a = 0; a < 3; ++a) vh[a][e] -= lam[d] * ud * dq[1 + a][e];
                  // -(1/rho) d_d (p + B_b^2/2 + B_e^2/2) acts on u_d;  +(B_d/rho) d_d B_a acts on u_a, a != d
                  vh[d][e] -= lam[d] * (dq[4][e] + c[5 + b][e] * dq[5 + b][e] + c[5 + eb][e] * dq[5 + eb][e]) * ir[e];
                  vh[b][e] += lam[d] * c[5 + d][e] * dq[5 + b][e] * ir[e];
                  vh[eb][e] += lam[d] * c[5 + d][e] * dq[5 + eb][e] * ir[e];
                }
              }
              // face-field transverse slopes: dy bx, dz bx, dx by, dz by, dx bz, dy bz
              const T* bx = b0 + o;
              const T* by = b0 + RA + o;
              const T* bz = b0 + 2 * RA + o;
              const V2<T> bxd = ld2(bx - BWX), bxn = ld2(bx + BWX);
              const V2<T> byn = ld2(by + BWX);
              const V2<T> bzd = ld2(bz - BWX), bzn = ld2(bz + BWX);
              const T bx2 = bx[2], bym = by[-1], by2 = by[2], bzm = bz[-1], bz2 = bz[2];
              st2(D + (D_DBF + 0) * DCS, limited_slope_k<LIM>(bxc.a - bxd.a, bxn.a - bxc.a), limited_slope_k<LIM>(bxc.b - bxd.b, bxn.b - bxc.b));
              st2(D + (D_DBF + 1) * DCS, limited_slope_k<LIM>(cbx[s_][0], fwx[0]), limited_slope_k<LIM>(cbx[s_][1], fwx[1]));
              {
                const T d0 = byc.a - bym, d1 = byc.b - byc.a, d2 = by2 - byc.b;
                st2(D + (D_DBF + 2) * DCS, limited_slope_k<LIM>(d0, d1), limited_slope_k<LIM>(d1, d2));
              }
              st2(D + (D_DBF + 3) * DCS, limited_slope_k<LIM>(cby[s_][0], fwy[0]), limited_slope_k<LIM>(cby[s_][1], fwy[1]));
              {
                const T d0 = bzc.a - bzm, d1 = bzc.b - bzc.a, d2 = bz2 - bzc.b;
                st2(D + (D_DBF + 4) * DCS, limited_slope_k<LIM>(d0, d1), limited_slope_k<LIM>(d1, d2));
              }
              st2(D + (D_DBF + 5) * DCS, limited_slope_k<LIM>(bzc.a - bzd.a, bzn.a - bzc.a), limited_slope_k<LIM>(bzc.b - bzd.b, bzn.b - bzc.b));
              // half-step faces (Eq. 12 with dt/2) of the two cells and of their +x, +y, +z neighbours:
              // EMFs of planes kd (0) and kd+1 (1) at columns 0..2 and rows 0, +1
              const T *ex0 = e0 + o, *ey0 = e0 + RA + o, *ez0 = e0 + 2 * RA + o;
              const T *ex1 = e1 + o, *ey1 = e1 + RA + o;
              const V2<T> ex0c = ld2(ex0), ex0n = ld2(ex0 + BWX), ex1c = ld2(ex1), ex1n = ld2(ex1 + BWX);
              const V2<T> ey0c = ld2(ey0), ey1c = ld2(ey1);
              const T ey02 = ey0[2], ey12 = ey1[2];
              const V2<T> ez0c = ld2(ez0), ez0n = ld2(ez0 + BWX);
              const T ez02 = ez0[2], ez0n2 = ez0[BWX + 2];
              // bx at columns 0, 1, 2
              const T bxh0 = bxc.a + (ly * (ez0n.a - ez0c.a) - lz * (ey1c.a - ey0c.a));
              const T bxh1 = bxc.b + (ly * (ez0n.b - ez0c.b) - lz * (ey1c.b - ey0c.b));
              const T bxh2 = bx2 + (ly * (ez0n2 - ez02) - lz * (ey12 - ey02));
              // by at rows 0 and +1
              const T byh0 = byc.a + (lz * (ex1c.a - ex0c.a) - lx * (ez0c.b - ez0c.a));
              const T byh1 = byc.b + (lz * (ex1c.b - ex0c.b) - lx * (ez02 - ez0c.b));
              const T byhn0 = byn.a + (lz * (ex1n.a - ex0n.a) - lx * (ez0n.b - ez0n.a));
              const T byhn1 = byn.b + (lz * (ex1n.b - ex0n.b) - lx * (ez0n2 - ez0n.b));
              // bz at planes kd and kd+1
              const T bzh0 = bzc.a + (lx * (ey0c.b - ey0c.a) - ly * (ex0n.a - ex0c.a));
              const T bzh1 = bzc.b + (lx * (ey02 - ey0c.b) - ly * (ex0n.b - ex0c.b));
              const T bzhu0 = bzu.a + (lx * (ey1c.b - ey1c.a) - ly * (ex1n.a - ex1c.a));
              const T bzhu1 = bzu.b + (lx * (ey12 - ey1c.b) - ly * (ex1n.b - ex1c.b));
              st2(D + (D_QH + 0) * DCS, rho_h[0], rho_h[1]);
              st2(D + (D_QH + 1) * DCS, vh[0][0], vh[0][1]);
              st2(D + (D_QH + 2) * DCS, vh[1][0], vh[1][1]);
              st2(D + (D_QH + 3) * DCS, vh[2][0], vh[2][1]);
              st2(D + (D_QH + 4) * DCS, p_h[0], p_h[1]);
              st2(D + (D_BCH + 0) * DCS, h * (bxh0 + bxh1), h * (bxh1 + bxh2));
              st2(D + (D_BCH + 1) * DCS, h * (byh0 + byhn0), h * (byh1 + byhn1));
              st2(D + (D_BCH + 2) * DCS, h * (bzh0 + bzhu0), h * (bzh1 + bzhu1));
              st2(D + (D_BH + 0) * DCS, bxh0, bxh1);
              st2(D + (D_BH + 1) * DCS, byh0, byh1);
              st2(D + (D_BH + 2) * DCS, bzh0, bzh1);
            }
            cbx[s_][0] = fwx[0]; cbx[s_][1] = fwx[1]; cby[s_][0] = fwy[0]; cby[s_][1] = fwy[1];
          }
        }
      }
      __threadfence_block();
      nb_arrive_if(kd >= rlo && kd >= za - 1, NB_FULL + ((kd + 2) & 1), NALL);
      cp_async_wait_all();   // own chunks of hydro plane r and field plane r+1 have landed ...
      nb_sync(NB_P, NP);     // ... and everybody's; the rings are rewritten by the next iteration
    }
    if (nbad) atomicAdd(bad, (unsigned long long)nbad);
    return;
  }

  // =========================================================== roles A and C ==========
  const bool roleA = t >= A0 && t < A0 + NR;
  const int tr = roleA ? t - A0 : t - C0;
  const bool colthr = tr >= C::CB;                        // closing-column warp
  const int fj = colthr ? tr - C::CB : tr / TX;
  const int fi = colthr ? TX : tr - fj * TX;
  const bool valid = colthr ? (fj < C::FH) : (tr < TX * C::FH);
  const bool active = valid && (fi <= tw) && (fj <= th);
  const bool cell = active && (fi < tw) && (fj < th);
  const bool xface = active && (fj < th) && (fi < tw || lastx);   // bx faces of the tile (closing face at the patch end)
  const bool yface = active && (fi < tw) && (fj < th || lasty);
  // the new face fields are also FORMED (not stored) on the tile's upper sides inside the patch: the
  // CFL rate of the last column / row of cells needs both faces of every cell
  const bool xcomp = active && (fj < th), ycomp = active && (fi < tw);
  const int own = (fj + 1) * DP + (fi + 4);          // D cell of (fi, fj): row fj+1, column rc = fi+4
  const int fidx = min(fj, C::FH - 1) * FW + fi;
  const int tyn = colthr ? tr + 1 : tr + TX;              // thread that owns (fi, fj+1)
  const int txn = colthr ? tr : ((fi == TX - 1) ? C::CB + fj : tr + 1);   // thread that owns (fi+1, fj)
  const long long plane = (long long)G.pitch * G.m[1], fs = G.fs;
  const long long ubase = (long long)P.patch(pl) * G.ps + G.lead + (x0 + fi + G.g[0]) +
                          (long long)(y0 + fj + G.g[1]) * G.pitch + (long long)G.g[2] * plane;
  const T cx = dt * P.idx[0], cy = dt * P.idx[1], cz = dt * P.idx[2];
  const int solver = DEFS ? 0 : G.emf_solver, FS = DEFS ? 0 : G.flux_solver;

  if (roleA) {
    // ------------------------------------------------------------- role A -----------
    const bool doFz = cell;
    const bool doEx = active && (fi < tw);      // ex(i, j..j+1): by faces and b_z
    const bool doEy = active && (fj < th);      // ey(i..i+1, j): bx faces and b_z
    Flux5<T> pFz = {};
    T pex = T(0), pey = T(0);
    T bzlo = T(0);                              // new b_z on the lower face of the plane below
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
      if (doFz) Lz = face_state<T, DCS, 2>(dp_, h);
      if (doEx) {   // ex, in-plane (y,z): sw=(j-1,k-1) se=(j,k-1) nw=(j-1,k) ne=(j,k)
        xsw = corner_state<T, DCS, 0>(dp_ - DP, h, h);
        xse = corner_state<T, DCS, 0>(dp_, -h, h);
        xAS = edge_field<T, DCS, 1, 2>(dp_, h);
      }
      if (doEy) {   // ey, in-plane (z,x): sw=(k-1,i-1) se=(k,i-1) nw=(k-1,i) ne=(k,i)
        ysw = corner_state<T, DCS, 1>(dp_ - 1, h, h);
        ynw = corner_state<T, DCS, 1>(dp_, h, -h);
        yBW = edge_field<T, DCS, 0, 2>(dp_, h);
      }
      nb_arrive_if(k + 1 <= zb, NB_EMPTY + ((k + 1) & 1), NALL);   // slot of plane k-1

      Flux5<T> cFz = {};
      T cex = T(0), cey = T(0);
      if (doFz) cFz = riemann_flux(FS, gamma, Lz, face_state<T, DCS, 2>(dc_, -h), dc_[(D_BH + 2) * DCS]);
      // The hydro part of plane k-1 only waits for this flux: finish it now (C is ahead, its
      // partial update is normally there already), so that the previous plane's flux is dead
      // while the two edge problems are solved.
      const long long cu = ubase + (long long)(k - 1) * plane;
      T* pu = PU + fidx;
      nb_sync_if(k >= za + 1, NB_PUF, 2 * NR);
      {
        if (k >= za + 1 && cell) {
          // O8: (U - dt*dFx/dx - dt*dFy/dy) - dt*dFz/dz; z-face frame (mu,mv,mw) = (mz,mx,my).
          // The new values also replace the partial ones in this thread's own PU entries: role C
          // picks them up after NB_PUE for the CFL rate of the new level.
          const T n0 = pu[0] - cz * (cFz.d - pFz.d);
          const T n1 = pu[FA] - cz * (cFz.mv - pFz.mv);
          const T n2 = pu[2 * FA] - cz * (cFz.mw - pFz.mw);
          const T n3 = pu[3 * FA] - cz * (cFz.mu - pFz.mu);
          const T n4 = pu[4 * FA] - cz * (cFz.e - pFz.e);
          P.Un[cu] = n0; P.Un[fs + cu] = n1; P.Un[2 * fs + cu] = n2; P.Un[3 * fs + cu] = n3; P.Un[4 * fs + cu] = n4;
          if (CFLE) { pu[0] = n0; pu[FA] = n1; pu[2 * FA] = n2; pu[3 * FA] = n3; pu[4 * FA] = n4; }
        }
      }
      pFz = cFz;
      if (doEx)
        cex = emf_2d(gamma, solver, xsw, xse, corner_state<T, DCS, 0>(dc_ - DP, h, -h), corner_state<T, DCS, 0>(dc_, -h, -h),
                     xAS, edge_field<T, DCS, 1, 2>(dc_, -h), edge_field<T, DCS, 2, 1>(dc_ - DP, h), edge_field<T, DCS, 2, 1>(dc_, -h));
      if (doEy)
        cey = emf_2d(gamma, solver, ysw, corner_state<T, DCS, 1>(dc_ - 1, -h, h), ynw, corner_state<T, DCS, 1>(dc_, -h, -h),
                     edge_field<T, DCS, 2, 0>(dc_ - 1, h), edge_field<T, DCS, 2, 0>(dc_, -h), yBW, edge_field<T, DCS, 0, 2>(dc_, -h));

      XE[tr] = cex;
      XE[NR + tr] = cey;
      nb_sync(NB_A, NR);
      const T yex = XE[tyn], xey = XE[NR + txn];
      // b_z on the lower z-face of plane k (k = nz: closing face) -- Eq. 12
      // (face zb belongs to the next segment unless it is the patch's closing face)
      const T bzn = u7 + (cx * (xey - cey) - cy * (yex - cex));
      if (cell && (k < zb || zb == nz)) P.Un[7 * fs + ubase + (long long)k * plane] = bzn;
      if (k >= za + 1) {
        // new b_x, b_y of plane k-1; with the cell-centred new b_z they join the new hydro values in
        // the PU entries (every face of the tile, also those another tile stores)
        if (CFLE ? xcomp : xface) {
          const T bxn = pu[5 * FA] - cz * (cey - pey);
          if (xface) P.Un[5 * fs + cu] = bxn;
          if (CFLE) pu[5 * FA] = bxn;
        }
        if (CFLE ? ycomp : yface) {
          const T byn = pu[6 * FA] + cz * (cex - pex);
          if (yface) P.Un[6 * fs + cu] = byn;
          if (CFLE) pu[6 * FA] = byn;
        }
        if (CFLE && cell) pu[7 * FA] = num<T>::xmul(h, num<T>::xadd(bzlo, bzn));
      }
      if (CFLE) __threadfence_block();
      nb_arrive_if(k >= za + 1, NB_PUE, 2 * NR);
      bzlo = bzn;
      pex = cex; pey = cey;
    }
    return;
  }

  // --------------------------------------------------------------- role C -----------
  {
    const bool doFx = active && (fj < th);
    const bool doFy = active && (fi < tw);
    T rmax = T(0);                              // largest CFL rate of the own cells (new level)
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
        if (CFLE ? xcomp : xface) un[5] = P.U[5 * fs + cu];
        if (CFLE ? ycomp : yface) un[6] = P.U[6 * fs + cu];
        const T* dc_ = dslot(kd) + own;
        if (doFx) Fx = riemann_flux(FS, gamma, face_state<T, DCS, 0>(dc_ - 1, h), face_state<T, DCS, 0>(dc_, -h), dc_[(D_BH + 0) * DCS]);
        if (doFy) Fy = riemann_flux(FS, gamma, face_state<T, DCS, 1>(dc_ - DP, h), face_state<T, DCS, 1>(dc_, -h), dc_[(D_BH + 1) * DCS]);
        if (active)   // ez, in-plane (x,y): sw=(i-1,j-1) se=(i,j-1) nw=(i-1,j) ne=(i,j)
          ez = emf_2d(gamma, solver, corner_state<T, DCS, 2>(dc_ - DP - 1, h, h), corner_state<T, DCS, 2>(dc_ - DP, -h, h),
                      corner_state<T, DCS, 2>(dc_ - 1, h, -h), corner_state<T, DCS, 2>(dc_, -h, -h),
                      edge_field<T, DCS, 0, 1>(dc_ - DP, h), edge_field<T, DCS, 0, 1>(dc_, -h),
                      edge_field<T, DCS, 1, 0>(dc_ - 1, h), edge_field<T, DCS, 1, 0>(dc_, -h));
      }
      nb_arrive_if(kd + 2 <= zb, NB_EMPTY + ((kd + 2) & 1), NALL);   // done with plane kd

      // neighbours: +x by warp shuffle (the closing column hands its values over through XC),
      // +y through XY
      if (work) {
        XY[tr] = Fy.d; XY[NR + tr] = Fy.mu; XY[2 * NR + tr] = Fy.mv; XY[3 * NR + tr] = Fy.mw; XY[4 * NR + tr] = Fy.e;
        XY[5 * NR + tr] = ez;
        if (colthr) {
          XC[fj] = Fx.d; XC[32 + fj] = Fx.mu; XC[2 * 32 + fj] = Fx.mv; XC[3 * 32 + fj] = Fx.mw; XC[4 * 32 + fj] = Fx.e;
          XC[5 * 32 + fj] = ez;
        }
      }
      // A has consumed the previous plane's partial update and left the NEW values of that plane
      // in the PU entries: take the ten a cell's CFL rate needs before the entries are rewritten
      const bool newvals = kd >= za + 1;
      nb_sync_if(newvals, NB_PUE, 2 * NR);
      T* pu = PU + fidx;
      T nv[10];
#pragma unroll
      for (int f = 0; f < 10; ++f) nv[f] = T(1);
      if (CFLE && newvals && cell) {
#pragma unroll
        for (int f = 0; f < 5; ++f) nv[f] = pu[f * FA];
        nv[5] = pu[5 * FA]; nv[6] = pu[5 * FA + 1];          // new b_x on both x-faces of the cell
        nv[7] = pu[6 * FA]; nv[8] = pu[6 * FA + FW];         // new b_y on both y-faces
        nv[9] = pu[7 * FA];                                  // cell-centred new b_z
      }
      nb_sync(NB_C, NR);      // every C thread has its XY/XC values out and its new values in
      if (work) {
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
        if (cell) {
          // momentum components by solver frame: x-face (mu,mv,mw)=(mx,my,mz); y-face (mu,mv,mw)=(my,mz,mx)
          pu[0] = un[0] - cx * (xF.d - Fx.d) - cy * (yF.d - Fy.d);
          pu[FA] = un[1] - cx * (xF.mu - Fx.mu) - cy * (yF.mw - Fy.mw);
          pu[2 * FA] = un[2] - cx * (xF.mv - Fx.mv) - cy * (yF.mu - Fy.mu);
          pu[3 * FA] = un[3] - cx * (xF.mw - Fx.mw) - cy * (yF.mv - Fy.mv);
          pu[4 * FA] = un[4] - cx * (xF.e - Fx.e) - cy * (yF.e - Fy.e);
        }
        if (CFLE ? xcomp : xface) pu[5 * FA] = un[5] + cy * (yez - ez);
        if (CFLE ? ycomp : yface) pu[6 * FA] = un[6] - cx * (xez - ez);
      }
      __threadfence_block();
      nb_arrive_if(work, NB_PUF, 2 * NR);
      // CFL rate of the NEW level in cell (fi, fj, kd-1) (O9), off A's critical path:
      // the step's epilogue replaces a separate pass over the state the step has just written
      if (CFLE && newvals && cell) {
        const T rate = cfl_rate<T>(gamma, P.idx[0], P.idx[1], P.idx[2], true, true, true, nv[0], nv[1], nv[2], nv[3], nv[4],
                                   nv[5], nv[6], nv[7], nv[8], nv[9], nv[9]);
        rmax = num<T>::max(rmax, rate);
      }
    }
    // per-patch maximum: warp shuffle, then one integer atomicMax per warp on the bit pattern
    // (positive doubles order like their bits: deterministic, no floating-point atomics)
    if (CFLE) {
      double rd = (double)rmax;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) rd = fmax(rd, __shfl_xor_sync(0xffffffffu, rd, o));
      if ((t & 31) == 0) atomicMax(&rate_next[P.patch(pl)], enc_max(rd));
    }
  }
}

}  // namespace mhd
