// tile_kernel.cuh -- the whole step of a TWO-DIMENSIONAL bunch (n_z = 1: BASELINE.json config 1, the
// paper's Orszag-Tang runs) in ONE kernel: every stage of PAPER.md section 2.1.4
// (L108-116) runs on a tile held in shared memory, so U^n is read once (with its halo) and U^{n+1}
// written once; nothing intermediate touches HBM and one launch replaces the staged path's eleven.
//
// The stages are the SAME device functions the staged kernels run (stage_kernels.cuh: st_prim,
// st_emf0, st_predict, st_flux, st_emf, st_update), fed through an accessor that points into the
// tile instead of the HBM scratch, so the results are the staged path's to rounding (the compiler may
// contract multiply-adds differently in the two instantiations).
//
// A CTA owns a TX x TY tile of one patch.  Tile arrays have rows of TP = TX + 6 cells and TH = TY + 6
// rows: cell (i, j) of the patch sits at column i - x0 + 3, row j - y0 + 3 (guard width 3, PAPER.md
// L212).  42 scratch arrays + the 8 raw fields: the scratch map of bunch_types.cuh with the arrays
// that are dead by then reused (the fluxes and the final EMFs take the place of the primitives and
// the time-n EMFs) and every slope along the collapsed z direction (all zero) in ONE array.
#pragma once
#include "bunch_types.cuh"
#include "mhd_math.cuh"
#include "stage_kernels.cuh"

namespace mhd {

// scratch array of bunch_types.cuh -> slot of the tile (z collapsed)
__host__ __device__ constexpr int tile_slot(int a) {
  return a < W_DQ ? a                                           // W_Q 0..7          -> 0..7
       : a < W_DQ + 16 ? 21 + (a - W_DQ)                        // slopes along x, y -> 21..36
       : a < W_DBF ? 41                                         // slopes along z    -> the zero array
       : a < W_E0 ? ((a - W_DBF) == 0 ? 37 : ((a - W_DBF) == 2 ? 38 : ((a - W_DBF) == 4 ? 39 : ((a - W_DBF) == 5 ? 40 : 41))))
       : a < W_BH ? 8 + (a - W_E0)                              // time-n EMFs       -> 8..10
       : a < W_QH ? 13 + (a - W_BH)                             // half-step faces   -> 13..15
       : a < W_FLUX ? 16 + (a - W_QH)                           // half-step hydro   -> 16..20
       : a < W_FLUX + 10 ? (a - W_FLUX)                         // fluxes along x, y -> 0..9 (over the primitives)
       : a < W_EMF ? 41                                         // fluxes along z: never touched
       : 10 + (a - W_EMF);                                      // final EMFs        -> 10..12 (10 over the time-n e_z)
}
constexpr int TILE_SLOTS = 42;

// NBUF raw-tile buffers: 1 = one tile per CTA, loaded with plain loads; 2 = PERSISTENT CTAs (one per SM) that
// walk the tiles and fetch the next tile's U^n with asynchronous copies (cp.async) while the current one
// is computed -- with one CTA per SM (shared memory) the load of a tile and the drain of its stores are
// otherwise fully exposed (30 % of the kernel's stall samples on a 2048^2 bunch).
template <typename T, int TX, int TY, int NBUF = 1> struct TileCfg {
  static constexpr int TP = TX + 6, TH = TY + 6, AR = TP * TH;
  static constexpr int NTH = sizeof(T) == 4 ? 704 : 384;
  static constexpr size_t smem = sizeof(T) * (size_t)(8 * NBUF + TILE_SLOTS) * AR;
  static_assert(smem <= 227 * 1024, "shared memory of one CTA");
};
__device__ __forceinline__ void tile_cp_async(float* dst, const float* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void tile_cp_async(double* dst, const double* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}

template <typename T, int AR, int TP, int LIM> struct TileAcc {
  static constexpr int lim_kind = LIM < 0 ? 1 : LIM;
  static constexpr bool def_solvers = LIM < 0;      // LIM = -1: minmod AND the default solvers (HLLD, HLLD-2D) at compile time
  const T* raw;   // [8][AR] at the cell
  T* W;           // [TILE_SLOTS][AR] at the cell
  T* Un;          // U^{n+1} in HBM at the cell
  long long ufs;
  __device__ __forceinline__ const T* u(int f) const { return raw + f * AR; }
  __device__ __forceinline__ T* un(int f) const { return Un + f * ufs; }
  __device__ __forceinline__ T* keep(int f) const { return const_cast<T*>(raw) + f * AR; }   // new value over the old one
  __device__ __forceinline__ T* w(int a) const { return W + tile_slot(a) * AR; }
  __device__ __forceinline__ long long s(int d) const { return d == 0 ? 1 : (d == 1 ? TP : 0); }
  __device__ __forceinline__ bool act(int d) const { return d < 2; }      // x, y active; z collapsed: folds at compile time
};

// CFLE: reduce the CFL rates of the NEW level in the kernel's epilogue (per-patch integer atomicMax on the
// bit pattern, as k_cfl does), so that the next mhd_bunch_cfl_dt only runs the bunch-wide reduction: the
// update leaves the new values in the raw tile (each thread over its own old values), the faces on the
// tile's upper sides that another tile stores are formed without being stored, and cfl_rate -- the same
// explicitly rounded function k_cfl evaluates -- gets the same inputs, hence the same bits.
template <typename T, int TX, int TY, bool CFLE, int NBUF, int LIM>
__global__ void __launch_bounds__(TileCfg<T, TX, TY>::NTH, 1)
k_step_tile2d(Params<T> P, const int* __restrict__ nbr, int gather, const double* __restrict__ dtp,
              unsigned long long* __restrict__ bad, unsigned long long* __restrict__ rate_next, int xtiles, int ytiles) {
  using C = TileCfg<T, TX, TY, NBUF>;
  constexpr int TP = C::TP, TH = C::TH, AR = C::AR, NTH = C::NTH;
  extern __shared__ __align__(16) unsigned char tile_smem[];
  T* const raw_all = reinterpret_cast<T*>(tile_smem);
  T* const W = raw_all + NBUF * 8 * AR;
  const Geom& G = P.G;
  const int nx = G.n[0], ny = G.n[1];
  const int t = threadIdx.x;
  const int ntile = xtiles * ytiles * P.npl;

  // U^n of cells [x0-3, x0+tw+2] x [y0-3, y0+th+2] of a tile -> a raw buffer.  GATHER mode: a cell outside the
  // patch is read from the interior of the neighbour of its class (guard fill O1 folded into the load:
  // PAPER.md L124, L188, L241), so the guard shell in HBM is neither written nor read; otherwise the patch's
  // own (already filled) guard cells are read.
  auto fetch = [&](int tile, T* dst) {
    const int pl_ = tile / (xtiles * ytiles), rt = tile - pl_ * (xtiles * ytiles);
    const int yt_ = rt / xtiles, xt_ = rt - yt_ * xtiles;
    const int X0 = xt_ * TX, Y0 = yt_ * TY;
    const long long pb = (long long)P.patch(pl_) * G.ps + G.lead;
    for (int idx = t; idx < AR; idx += NTH) {
      const int lr = idx / TP, lc = idx - lr * TP;
      const int i = X0 - 3 + lc, j = Y0 - 3 + lr;
      if (i <= nx + 2 && j <= ny + 2) {
        long long g = pb + (i + G.g[0]) + (long long)(j + G.g[1]) * G.pitch;
        if (gather) {
          const int ox = i < 0 ? -1 : (i >= nx ? 1 : 0), oy = j < 0 ? -1 : (j >= ny ? 1 : 0);
          if (ox | oy) {
            const int q = nbr[(long long)P.patch(pl_) * 27 + 9 + (oy + 1) * 3 + (ox + 1)];
            g = (long long)q * G.ps + G.lead + (i - ox * nx + G.g[0]) + (long long)(j - oy * ny + G.g[1]) * G.pitch;
          }
        }
#pragma unroll
        for (int f = 0; f < 8; ++f) {
          if (NBUF == 1) dst[f * AR + idx] = P.U[f * G.fs + g];
          else tile_cp_async(dst + f * AR + idx, P.U + f * G.fs + g);
        }
      }
    }
  };
  if (NBUF == 2 && (int)blockIdx.x < ntile) fetch(blockIdx.x, raw_all);

  int nb = 0;
  for (int tile = blockIdx.x; tile < ntile; tile += gridDim.x, nb ^= (NBUF - 1)) {
  T* const raw = raw_all + nb * 8 * AR;
  const int pl = tile / (xtiles * ytiles), rt_ = tile - pl * (xtiles * ytiles);
  const int yt = rt_ / xtiles, xt = rt_ - yt * xtiles;
  const int x0 = xt * TX, y0 = yt * TY;
  const int tw = min(TX, nx - x0), th = min(TY, ny - y0);
  const bool lastx = x0 + tw == nx, lasty = y0 + th == ny;
  const T dt = P.dt_of(pl, dtp);
  const long long pbase = (long long)P.patch(pl) * G.ps + G.lead;
  if (NBUF == 1) {
    fetch(tile, raw);
  } else {
    asm volatile("cp.async.wait_all;" ::: "memory");
  }
  __syncthreads();     // the tile has landed; every thread is done with the previous tile (its W arrays, its raw buffer)
  if (NBUF == 2 && tile + (int)gridDim.x < ntile) fetch(tile + gridDim.x, raw_all + (nb ^ 1) * 8 * AR);

  // a stage over the cells [ilo, ihi] x [jlo, jhi] of the patch
  auto acc = [&](int i, int j) {
    const int o = (j - y0 + 3) * TP + (i - x0 + 3);
    TileAcc<T, AR, TP, LIM> a;
    a.raw = raw + o; a.W = W + o; a.ufs = G.fs;
    a.Un = P.Un + pbase + (i + G.g[0]) + (long long)(j + G.g[1]) * G.pitch;
    return a;
  };
  // Task r of a w x h box -> (di, dj).  The first 32 columns go row by row, 32 tasks = one warp = one tile
  // row (consecutive shared-memory words: no bank conflicts, also for the +-1 and +-TP neighbours); the
  // remaining columns go column by column (stride TP = 38 words: 16 distinct banks before one repeats).
  // Mapping tasks of a 33- to 36-wide box straight onto 38-word rows made 44 % of the kernel's shared-memory
  // wavefronts bank-conflict replays.
  auto task = [&](int r, int w, int h, int& di, int& dj) {
    if (w <= 32) { dj = r / w; di = r - dj * w; }
    else if (r < 32 * h) { dj = r >> 5; di = r & 31; }
    else { r -= 32 * h; di = r / h; dj = r - di * h; di += 32; }
  };
#define TILE_FOR(ilo, ihi, jlo, jhi, BODY)                                   \
  {                                                                          \
    const int ni_ = (ihi) - (ilo) + 1, nj_ = (jhi) - (jlo) + 1;              \
    for (int it_ = t; it_ < ni_ * nj_; it_ += NTH) {                         \
      int di_, dj_;                                                          \
      task(it_, ni_, nj_, di_, dj_);                                         \
      const int i = (ilo) + di_, j = (jlo) + dj_;                            \
      const TileAcc<T, AR, TP, LIM> x = acc(i, j);                                \
      BODY;                                                                  \
    }                                                                        \
  }
  // O2: primitives; only the tile's own cells count towards the bad-cell total
  TILE_FOR(x0 - 2, x0 + tw + 1, y0 - 2, y0 + th + 1,
           st_prim<T>(P, x, (i >= x0 && i < x0 + tw && j >= y0 && j < y0 + th) ? i : -1, j, 0, bad));
  __syncthreads();
  TILE_FOR(x0 - 1, x0 + tw + 1, y0 - 1, y0 + th + 1, st_emf0<T>(P, x));
  __syncthreads();
  TILE_FOR(x0 - 1, x0 + tw + 1, y0 - 1, y0 + th + 1, st_predict<T>(P, x, i, j, 0, dt));
  __syncthreads();
  // the five Riemann problems of the plane as ONE list of tasks over all threads: x faces (tw+1) x th, y faces
  // tw x (th+1), x-directed edges tw x (th+1), y-directed edges (tw+1) x th, z-directed edges (tw+1) x (th+1).
  // The row-by-row parts of all five come first (each a whole number of warps for a full tile), then their
  // 33rd columns.
  {
    // (scalars, not arrays: nothing here may end up in local memory)
    const int wA = tw + 1, wB = tw, hA = th, hB = th + 1;                       // widths / heights of the five boxes
    const int m0 = min(wA, 32) * hA, m1 = min(wB, 32) * hB, m2 = m1, m3 = m0, m4 = min(wA, 32) * hB;
    const int c0 = wA * hA - m0, c1 = wB * hB - m1, c2 = c1, c3 = c0, c4 = wA * hB - m4;
    const int M1 = m0, M2 = M1 + m1, M3 = M2 + m2, M4 = M3 + m3, M5 = M4 + m4;
    const int C1 = M5 + c0, C2 = C1 + c1, C3 = C2 + c2, C4 = C3 + c3, C5 = C4 + c4;
    for (int it = t; it < C5; it += NTH) {
      int q, r;
      if (it < M5) {
        q = (it >= M1) + (it >= M2) + (it >= M3) + (it >= M4);
        r = it - (q == 0 ? 0 : (q == 1 ? M1 : (q == 2 ? M2 : (q == 3 ? M3 : M4))));
      } else {
        q = (it >= C1) + (it >= C2) + (it >= C3) + (it >= C4);
        r = it - (q == 0 ? M5 : (q == 1 ? C1 : (q == 2 ? C2 : (q == 3 ? C3 : C4)))) + (q == 0 ? m0 : (q == 1 ? m1 : (q == 2 ? m2 : (q == 3 ? m3 : m4))));
      }
      const int bwq = (q == 1 || q == 2) ? wB : wA, bhq = (q == 0 || q == 3) ? hA : hB;
      int di, dj;
      task(r, bwq, bhq, di, dj);
      const TileAcc<T, AR, TP, LIM> x = acc(x0 + di, y0 + dj);
      if (q == 0) st_flux<T, 0>(P, x);
      else if (q == 1) st_flux<T, 1>(P, x);
      else if (q == 2) st_emf<T, 0>(P, x);
      else if (q == 3) st_emf<T, 1>(P, x);
      else st_emf<T, 2>(P, x);
    }
  }
  __syncthreads();
  // O8: the tile's cells and lower faces; the closing faces where the tile ends its patch
  TILE_FOR(x0, x0 + tw - 1 + (lastx ? 1 : 0), y0, y0 + th - 1 + (lasty ? 1 : 0), (st_update<T, CFLE>(P, x, i, j, 0, dt)));
  if (CFLE) {
    // b_x on the tile's last column of faces and b_y on its last row, where the next tile stores them
    if (!lastx) TILE_FOR(x0 + tw, x0 + tw, y0, y0 + th - 1, (st_update<T, true>(P, x, i, j, 0, dt, 2, false)));
    if (!lasty) TILE_FOR(x0, x0 + tw - 1, y0 + th, y0 + th, (st_update<T, true>(P, x, i, j, 0, dt, 4, false)));
    __syncthreads();
    T rmax = T(0);
    for (int it = t; it < tw * th; it += NTH) {
      const int jj = it / tw;
      const T* c = raw + (jj + 3) * TP + (it - jj * tw + 3);
      const T rate = cfl_rate<T>(P.gamma, P.idx[0], P.idx[1], P.idx[2], true, true, false, c[0], c[AR], c[2 * AR], c[3 * AR], c[4 * AR],
                                 c[5 * AR], c[5 * AR + 1], c[6 * AR], c[6 * AR + TP], c[7 * AR], c[7 * AR]);
      rmax = num<T>::max(rmax, rate);
    }
    double rd = (double)rmax;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) rd = fmax(rd, __shfl_xor_sync(0xffffffffu, rd, o));
    if ((t & 31) == 0 && rd > 0.0) atomicMax(&rate_next[P.patch(pl)], enc_max(rd));
  }
  }   // tiles of this CTA
#undef TILE_FOR
}

// ---- one-dimensional bunches along x (n_y = n_z = 1: BASELINE.json config 0, the shock-tube runs of PAPER.md
// L186): the same stages on the whole row of a patch, one small CTA per patch, one launch instead of twelve.
// Every scratch array keeps its own slot (75 short rows).
template <typename T, int LIM> struct LineAcc {
  static constexpr int lim_kind = LIM < 0 ? 1 : LIM;
  static constexpr bool def_solvers = LIM < 0;
  const T* raw; T* W; T* Un;
  long long ufs; int L;
  __device__ __forceinline__ const T* u(int f) const { return raw + f * L; }
  __device__ __forceinline__ T* un(int f) const { return Un + f * ufs; }
  __device__ __forceinline__ T* keep(int f) const { return const_cast<T*>(raw) + f * L; }
  __device__ __forceinline__ T* w(int a) const { return W + a * L; }
  __device__ __forceinline__ long long s(int d) const { return d == 0 ? 1 : 0; }
  __device__ __forceinline__ bool act(int d) const { return d == 0; }
};

template <typename T, bool CFLE, int LIM>
__global__ void __launch_bounds__(128)
k_step_line1d(Params<T> P, const int* __restrict__ nbr, int gather, const double* __restrict__ dtp,
              unsigned long long* __restrict__ bad, unsigned long long* __restrict__ rate_next) {
  extern __shared__ __align__(16) unsigned char tile_smem[];
  const Geom& G = P.G;
  const int nx = G.n[0], L = nx + 6, t = threadIdx.x, NTH = blockDim.x;
  T* const raw = reinterpret_cast<T*>(tile_smem);
  T* const W = raw + 8 * L;
  const int pl = blockIdx.x;
  const T dt = P.dt_of(pl, dtp);
  const long long pbase = (long long)P.patch(pl) * G.ps + G.lead;
  for (int idx = t; idx < L; idx += NTH) {
    const int i = idx - 3;
    long long g = pbase + (i + G.g[0]);
    if (gather) {
      const int ox = i < 0 ? -1 : (i >= nx ? 1 : 0);
      if (ox) g = (long long)nbr[(long long)P.patch(pl) * 27 + 13 + ox] * G.ps + G.lead + (i - ox * nx + G.g[0]);
    }
#pragma unroll
    for (int f = 0; f < 8; ++f) raw[f * L + idx] = P.U[f * G.fs + g];
  }
  __syncthreads();
  auto acc = [&](int i) {
    LineAcc<T, LIM> a;
    a.raw = raw + i + 3; a.W = W + i + 3; a.ufs = G.fs; a.L = L;
    a.Un = P.Un + pbase + (i + G.g[0]);
    return a;
  };
  for (int i = -2 + t; i <= nx + 1; i += NTH) st_prim<T>(P, acc(i), (i >= 0 && i < nx) ? i : -1, 0, 0, bad);
  __syncthreads();
  for (int i = -1 + t; i <= nx + 1; i += NTH) st_emf0<T>(P, acc(i));
  __syncthreads();
  for (int i = -1 + t; i <= nx + 1; i += NTH) st_predict<T>(P, acc(i), i, 0, 0, dt);
  __syncthreads();
  // x faces and the y- and z-directed edges at the faces (the x-directed edge EMF only enters through differences
  // that vanish)
  for (int it = t; it < 3 * (nx + 1); it += NTH) {
    const int q = it / (nx + 1), i = it - q * (nx + 1);
    if (q == 0) st_flux<T, 0>(P, acc(i));
    else if (q == 1) st_emf<T, 1>(P, acc(i));
    else st_emf<T, 2>(P, acc(i));
  }
  __syncthreads();
  for (int i = t; i <= nx; i += NTH) st_update<T, CFLE>(P, acc(i), i, 0, 0, dt);
  if (CFLE) {
    __syncthreads();
    T rmax = T(0);
    for (int i = t; i < nx; i += NTH) {
      const T* c = raw + i + 3;
      rmax = num<T>::max(rmax, cfl_rate<T>(P.gamma, P.idx[0], P.idx[1], P.idx[2], true, false, false, c[0], c[L], c[2 * L], c[3 * L],
                                            c[4 * L], c[5 * L], c[5 * L + 1], c[6 * L], c[6 * L], c[7 * L], c[7 * L]));
    }
    double rd = (double)rmax;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) rd = fmax(rd, __shfl_xor_sync(0xffffffffu, rd, o));
    if ((t & 31) == 0 && rd > 0.0) atomicMax(&rate_next[P.patch(pl)], enc_max(rd));
  }
}

}  // namespace mhd
