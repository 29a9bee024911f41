// stage_kernels.cuh -- guard fill, CFL reduction and the staged step kernels (one kernel per
// stage of PAPER.md section 2.1.4 with HBM scratch).  The staged step is the general path
// (any mix of active and collapsed dimensions); fused_kernels.cuh holds the fast 3D path.
#pragma once
#include <math.h>
#include "bunch_types.cuh"
#include "mhd_math.cuh"

namespace mhd {

// -------------------------------------------------------------------- guard fill ----
// O1 (width 3 L212): every guard cell copies all 8 fields from
// the neighbour's interior image, or from the nearest own interior cell (zero gradient).
// Threads enumerate GUARD CELLS ONLY, slab by slab (z-low, z-high, y-low, y-high, x-low,
// x-high) with x fastest, so the full-row slabs read and write contiguous runs; each thread
// moves the 8 fields of one guard cell (8 independent loads in flight, then 8 stores).
struct FillMap {
  int start[7];      // first guard index of each slab; start[6] = guard cells per patch
  int lo[6][3];      // first cell (i,j,k) of the slab, interior-relative
  int ext[6][3];     // extents of the slab
};

inline FillMap make_fill_map(const Geom& G) {
  FillMap M;
  int n = 0, s = 0;
  // the six slabs tile the guard shell: z slabs span the padded x,y range, y slabs the padded
  // x range and interior z, x slabs interior y and z
  for (int d = 2; d >= 0; --d) {
    for (int side = 0; side < 2; ++side) {
      M.start[s] = n;
      for (int a = 0; a < 3; ++a) {
        if (a == d) { M.lo[s][a] = side ? G.n[a] : -G.g[a]; M.ext[s][a] = G.g[a]; }
        else if (a > d) { M.lo[s][a] = 0; M.ext[s][a] = G.n[a]; }
        else { M.lo[s][a] = -G.g[a]; M.ext[s][a] = G.m[a]; }
      }
      n += M.ext[s][0] * M.ext[s][1] * M.ext[s][2];
      ++s;
    }
  }
  M.start[6] = n;
  return M;
}

template <typename T>
__global__ void __launch_bounds__(256) k_fill_guards(Geom G, FillMap M, T* __restrict__ U, const int* __restrict__ nbr) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int per = M.start[6];
  if (t >= (long long)per * G.np) return;
  const int p = (int)(t / per);
  int r = (int)(t - (long long)p * per);
  // slab parameters by an unrolled compare chain: indices into M stay compile-time, so the
  // parameter struct is read from constant space and never copied to local memory
  int st = 0, l0 = M.lo[0][0], l1 = M.lo[0][1], l2 = M.lo[0][2], e0 = M.ext[0][0], e1 = M.ext[0][1];
#pragma unroll
  for (int q = 1; q < 6; ++q) {
    if (r >= M.start[q]) { st = M.start[q]; l0 = M.lo[q][0]; l1 = M.lo[q][1]; l2 = M.lo[q][2]; e0 = M.ext[q][0]; e1 = M.ext[q][1]; }
  }
  r -= st;
  const int exy = e0 * e1;
  const int kk = r / exy; r -= kk * exy;
  const int jj = r / e0;
  const int ii = r - jj * e0;
  const int c[3] = {l0 + ii, l1 + jj, l2 + kk};
  int o[3], src[3], cl[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    o[d] = c[d] < 0 ? -1 : (c[d] >= G.n[d] ? 1 : 0);
    src[d] = c[d] - o[d] * G.n[d];
    cl[d] = min(max(c[d], 0), G.n[d] - 1);
  }
  const int q = nbr[p * 27 + (o[2] + 1) * 9 + (o[1] + 1) * 3 + (o[0] + 1)];
  const long long pitch = G.pitch, plane = (long long)G.pitch * G.m[1];
  const long long dst = (long long)p * G.ps + G.lead + (c[0] + G.g[0]) + (c[1] + G.g[1]) * pitch + (c[2] + G.g[2]) * plane;
  long long from;
  if (q >= 0)
    from = (long long)q * G.ps + G.lead + (src[0] + G.g[0]) + (src[1] + G.g[1]) * pitch + (src[2] + G.g[2]) * plane;
  else
    from = (long long)p * G.ps + G.lead + (cl[0] + G.g[0]) + (cl[1] + G.g[1]) * pitch + (cl[2] + G.g[2]) * plane;
  T v[8];
#pragma unroll
  for (int f = 0; f < 8; ++f) v[f] = U[f * G.fs + from];
#pragma unroll
  for (int f = 0; f < 8; ++f) {
    if (q < 0 && f >= 5) {  // the closing face keeps its evolved value (O8)
      const int a = f - 5, b = (a + 1) % 3, e = (a + 2) % 3;
      if (G.act[a] && c[a] == G.n[a] && o[b] == 0 && o[e] == 0) continue;
    }
    U[f * G.fs + dst] = v[f];
  }
}

// The same fill in 16-byte chunks, for bunches whose every neighbour exists (no zero-gradient side) and
// whose rows are whole chunks (n_x a multiple of 16 / sizeof(T); lead pad + guard width = 4 elements).
// A row of the padded patch is CPR chunks: LG chunks of low x-guards (with the lead pad), n_x / VEC
// interior chunks, HG chunks of high x-guards (with the trailing pad).  Guard ROWS (y or z outside the
// interior) are copied whole, chunk by chunk, from the row of the neighbour of class (o_x of the
// chunk, o_y, o_z); interior rows only get their LG + HG guard chunks.  Every chunk of a destination
// row comes from ONE chunk of a source row (the guard chunks of a row are the interior chunks at the
// far / near end of the x-neighbour's row), so the x-guards -- 12-byte fragments that cost whole
// sectors in the scalar kernel -- move as aligned 16-byte accesses like everything else.  Pad
// elements receive copies of interior values nobody reads.  A thread moves one chunk of FillFpt<T>::N fields.
template <typename T> struct FillFpt { static constexpr int N = sizeof(T) == 4 ? 2 : 8; };
template <typename T>
__global__ void __launch_bounds__(256) k_fill_guards_vec(Geom G, T* __restrict__ U, const int* __restrict__ nbr) {
  constexpr int VEC = 16 / sizeof(T);
  using V = int4;
  const int nx = G.n[0], ny = G.n[1], nz = G.n[2], g1 = G.g[1], g2 = G.g[2], my = G.m[1];
  const int CPR = G.pitch / VEC, LG = (G.lead + G.g[0]) / VEC, NI = nx / VEC, HG = CPR - LG - NI;
  const int nfull = my * G.m[2] - ny * nz;                 // guard rows of a patch
  const int per = nfull * CPR + ny * nz * (LG + HG);
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (long long)per * G.np) return;
  const int p = (int)(t / per);
  int r = (int)(t - (long long)p * per);
  int jj, kk, c;                                           // padded row (jj, kk), chunk of the row
  if (r < nfull * CPR) {
    int fr = r / CPR;
    c = r - fr * CPR;
    if (fr < g2 * my) { kk = fr / my; jj = fr - kk * my; }
    else if (fr < 2 * g2 * my) { fr -= g2 * my; kk = fr / my; jj = fr - kk * my; kk += g2 + nz; }
    else {
      fr -= 2 * g2 * my;
      kk = fr / (2 * g1);
      const int s_ = fr - kk * 2 * g1;
      kk += g2;
      jj = s_ < g1 ? s_ : ny + s_;
    }
  } else {
    r -= nfull * CPR;
    const int ir = r / (LG + HG), cc = r - ir * (LG + HG);
    kk = g2 + ir / ny;
    jj = g1 + ir - (ir / ny) * ny;
    c = cc < LG ? cc : NI + cc;
  }
  const int j = jj - g1, k = kk - g2;
  const int ox = c < LG ? -1 : (c >= LG + NI ? 1 : 0);
  const int oy = j < 0 ? -1 : (j >= ny ? 1 : 0), oz = k < 0 ? -1 : (k >= nz ? 1 : 0);
  const int q = nbr[p * 27 + (oz + 1) * 9 + (oy + 1) * 3 + (ox + 1)];
  const long long plane = (long long)G.pitch * my;
  const long long dst = (long long)p * G.ps + (long long)kk * plane + (long long)jj * G.pitch + (long long)c * VEC;
  const long long from = (long long)q * G.ps + (long long)(kk - oz * nz) * plane + (long long)(jj - oy * ny) * G.pitch +
                         (long long)(c - ox * NI) * VEC;
  // fields per thread (blockIdx.y picks the group): measured best 2 in fp32 (0.34 -> 0.31 ms on config 2: fewer
  // loads queued per warp), all 8 in fp64
  constexpr int FILL_FPT = FillFpt<T>::N;
  const int f0 = (int)blockIdx.y * FILL_FPT;
  V v[FILL_FPT];
#pragma unroll
  for (int f = 0; f < FILL_FPT; ++f) v[f] = *reinterpret_cast<const V*>(U + (f0 + f) * G.fs + from);
#pragma unroll
  for (int f = 0; f < FILL_FPT; ++f) *reinterpret_cast<V*>(U + (f0 + f) * G.fs + dst) = v[f];
}

// O10, local time steps: guard fill of the NEWER slice of each listed
// patch from its neighbours' two slices, linearly interpolated in time to the patch's own time.
// S0/S1: the two state buffers; slot[q]: which of them holds the newer slice of patch q;
// wtab[i][class]: weight of the newer slice for listed patch i and neighbour class (1: take the
// newer slice itself, bit for bit -- equal times).  Same thread-to-guard-cell map as k_fill_guards.
template <typename T>
__global__ void __launch_bounds__(256) k_fill_guards_local(Geom G, FillMap M, T* __restrict__ S0, T* __restrict__ S1,
                                                           const int* __restrict__ nbr, const int* __restrict__ slot,
                                                           const int* __restrict__ plist, const double* __restrict__ wtab,
                                                           int nlist) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int per = M.start[6];
  if (t >= (long long)per * nlist) return;
  const int il = (int)(t / per);
  const int p = plist[il];
  int r = (int)(t - (long long)il * per);
  int st = 0, l0 = M.lo[0][0], l1 = M.lo[0][1], l2 = M.lo[0][2], e0 = M.ext[0][0], e1 = M.ext[0][1];
#pragma unroll
  for (int q = 1; q < 6; ++q) {
    if (r >= M.start[q]) { st = M.start[q]; l0 = M.lo[q][0]; l1 = M.lo[q][1]; l2 = M.lo[q][2]; e0 = M.ext[q][0]; e1 = M.ext[q][1]; }
  }
  r -= st;
  const int exy = e0 * e1;
  const int kk = r / exy; r -= kk * exy;
  const int jj = r / e0;
  const int ii = r - jj * e0;
  const int c[3] = {l0 + ii, l1 + jj, l2 + kk};
  int o[3], src[3], cl[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    o[d] = c[d] < 0 ? -1 : (c[d] >= G.n[d] ? 1 : 0);
    src[d] = c[d] - o[d] * G.n[d];
    cl[d] = min(max(c[d], 0), G.n[d] - 1);
  }
  const int cls = (o[2] + 1) * 9 + (o[1] + 1) * 3 + (o[0] + 1);
  const int q = nbr[p * 27 + cls];
  const long long pitch = G.pitch, plane = (long long)G.pitch * G.m[1];
  T* const mine = slot[p] ? S1 : S0;
  const long long dst = (long long)p * G.ps + G.lead + (c[0] + G.g[0]) + (c[1] + G.g[1]) * pitch + (c[2] + G.g[2]) * plane;
  if (q >= 0) {
    const long long from = (long long)q * G.ps + G.lead + (src[0] + G.g[0]) + (src[1] + G.g[1]) * pitch + (src[2] + G.g[2]) * plane;
    const T* const qn = slot[q] ? S1 : S0;
    const T* const qo = slot[q] ? S0 : S1;
    const double w = wtab[il * 27 + cls];
    T v[8];
#pragma unroll
    for (int f = 0; f < 8; ++f) v[f] = qn[f * G.fs + from];
    if (w != 1.0) {   // never touches the older slice of a neighbour at the patch's own time (it may be written by this call's steps)
      const T wt = (T)w;
#pragma unroll
      for (int f = 0; f < 8; ++f) {
        const T vo = qo[f * G.fs + from];
        v[f] = vo + wt * (v[f] - vo);
      }
    }
#pragma unroll
    for (int f = 0; f < 8; ++f) mine[f * G.fs + dst] = v[f];
  } else {
    const long long from = (long long)p * G.ps + G.lead + (cl[0] + G.g[0]) + (cl[1] + G.g[1]) * pitch + (cl[2] + G.g[2]) * plane;
#pragma unroll
    for (int f = 0; f < 8; ++f) {
      if (f >= 5) {  // the closing face keeps its evolved value (O8)
        const int a = f - 5, b = (a + 1) % 3, e = (a + 2) % 3;
        if (G.act[a] && c[a] == G.n[a] && o[b] == 0 && o[e] == 0) continue;
      }
      mine[f * G.fs + dst] = mine[f * G.fs + from];
    }
  }
}

// The closing faces alone (O8: face n_a of the normal field b_a sits in the first high guard
// slot): the neighbour's face 0 overwrites it, an outflow side keeps the evolved value.
// This is the only part of the guard shell that cfl_dt and the one-pass kernel's update read
// from HBM, so it is all a deferred fill has to do up front.
template <typename T>
__global__ void __launch_bounds__(256) k_sync_closing_faces(Geom G, T* __restrict__ U, const int* __restrict__ nbr,
                                                            int p0, int npl, int zlo, int zhi) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int fx = G.n[1] * G.n[2], fy = G.n[0] * G.n[2], fz = G.n[0] * G.n[1];
  const int per = fx + fy + fz;
  if (t >= (long long)per * npl) return;
  const int p = p0 + (int)(t / per);
  int r = (int)(t % per);
  int a, c[3];
  if (r < fx) { a = 0; c[0] = G.n[0]; c[1] = r % G.n[1]; c[2] = r / G.n[1]; }
  else if (r < fx + fy) { r -= fx; a = 1; c[0] = r % G.n[0]; c[1] = G.n[1]; c[2] = r / G.n[0]; }
  else { r -= fx + fy; a = 2; c[0] = r % G.n[0]; c[1] = r / G.n[0]; c[2] = G.n[2]; }
  if (!G.act[a]) return;
  // planes [zlo, zhi) only (the z closing face belongs to the band that ends at n_z)
  if (a == 2 ? zhi != G.n[2] : (c[2] < zlo || c[2] >= zhi)) return;
  const int cls = 13 + (a == 0 ? 1 : (a == 1 ? 3 : 9));      // neighbour class with offset +1 along a
  const int q = nbr[p * 27 + cls];
  if (q < 0) return;
  const long long pitch = G.pitch, plane = (long long)G.pitch * G.m[1];
  const long long dst = (long long)p * G.ps + G.lead + (c[0] + G.g[0]) + (c[1] + G.g[1]) * pitch + (c[2] + G.g[2]) * plane;
  c[a] = 0;
  const long long from = (long long)q * G.ps + G.lead + (c[0] + G.g[0]) + (c[1] + G.g[1]) * pitch + (c[2] + G.g[2]) * plane;
  U[(5 + a) * G.fs + dst] = U[(5 + a) * G.fs + from];
}

// -------------------------------------------------------------------------- CFL ----
__device__ __forceinline__ unsigned long long enc_max(double x) { return (unsigned long long)__double_as_longlong(x); }

// O9: rate = sum_d (|u_d| + c_f,d)/dx_d over active d; per-patch maximum.
// Positive doubles order like their bit patterns, so the maximum is an integer atomicMax:
// deterministic, no floating-point atomics.
template <typename T>
__global__ void __launch_bounds__(256) k_cfl(Params<T> P, unsigned long long* __restrict__ rate_bits) {
  const Geom& G = P.G;
  const int p = blockIdx.y;
  const long long per = (long long)G.n[0] * G.n[1] * G.n[2];
  double rmax = 0.0;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < per; t += (long long)gridDim.x * blockDim.x) {
    int r = (int)t;
    const int nxy = G.n[0] * G.n[1];
    const int k = r / nxy; r -= k * nxy;
    const int j = r / G.n[0];
    const int i = r - j * G.n[0];
    const long long c = (long long)p * G.ps + G.lead + (i + G.g[0]) + (long long)(j + G.g[1]) * G.pitch +
                        (long long)(k + G.g[2]) * G.pitch * G.m[1];
    const T* U = P.U;
    const T rate = cfl_rate<T>(P.gamma, P.idx[0], P.idx[1], P.idx[2], G.act[0] != 0, G.act[1] != 0, G.act[2] != 0, U[c],
                               U[G.fs + c], U[2 * G.fs + c], U[3 * G.fs + c], U[4 * G.fs + c], U[5 * G.fs + c],
                               U[5 * G.fs + c + G.s[0]], U[6 * G.fs + c], U[6 * G.fs + c + G.s[1]], U[7 * G.fs + c],
                               U[7 * G.fs + c + G.s[2]]);   // a NaN cell comes back as +inf: dt = 0 rather than being ignored
    rmax = fmax(rmax, (double)rate);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) rmax = fmax(rmax, __shfl_xor_sync(0xffffffffu, rmax, o));
  __shared__ double sm[8];
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = rmax;
  __syncthreads();
  if (threadIdx.x < 32) {
    double v = threadIdx.x < (blockDim.x >> 5) ? sm[threadIdx.x] : 0.0;
#pragma unroll
    for (int o = 4; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    if (threadIdx.x == 0) atomicMax(&rate_bits[p], enc_max(v));
  }
}

// second stage: bunch-wide minimum step, optional per-patch steps
__global__ void __launch_bounds__(256) k_cfl_final(const unsigned long long* __restrict__ rate_bits, int np, double courant,
                                                   double* __restrict__ dt_out, double* __restrict__ dt_user,
                                                   double* __restrict__ dt_patch) {
  double rmax = 0.0;
  for (int p = threadIdx.x; p < np; p += blockDim.x) {
    const double r = __longlong_as_double((long long)rate_bits[p]);
    if (dt_patch) dt_patch[p] = courant / r;
    rmax = fmax(rmax, r);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) rmax = fmax(rmax, __shfl_xor_sync(0xffffffffu, rmax, o));
  __shared__ double sm[8];
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = rmax;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w) rmax = fmax(rmax, sm[w]);
    const double dt = courant / rmax;
    *dt_out = dt;
    if (dt_user) *dt_user = dt;
  }
}

__global__ void k_zero_u64(unsigned long long* p, int n) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t < n) p[t] = 0ull;
}

// mhd_bunch_local_end: the newer time slice of every patch whose slot is not `cur` moves into buffer
// `cur` -- all eight fields of all such patches in ONE launch (blockIdx.y = patch, blockIdx.z = field),
// 16 bytes per thread; a patch and a field start on 16-byte boundaries (ps is a multiple of four elements).
__global__ void __launch_bounds__(256) k_gather_slices(uint4* __restrict__ dst, const uint4* __restrict__ src,
                                                       const int* __restrict__ slot, int cur, long long patch_v, long long field_v) {
  const int p = blockIdx.y;
  if (slot[p] == cur) return;
  const long long base = (long long)blockIdx.z * field_v + (long long)p * patch_v;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < patch_v; t += (long long)gridDim.x * blockDim.x)
    dst[base + t] = src[base + t];
}

// FMA-chain microbenchmark: 16 independent chains per thread, used to MEASURE the fp32/fp64
// pipe peak that the ALU roofline of the step kernels is reported against
template <typename T>
__global__ void __launch_bounds__(256) k_fma_peak(T* out, int iters, T a, T b) {
  T x[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) x[i] = T(threadIdx.x + i) * T(1e-3);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = x[i] * a + b;
  }
  T s = T(0);
#pragma unroll
  for (int i = 0; i < 16; ++i) s += x[i];
  if (s == T(-1)) out[blockIdx.x * blockDim.x + threadIdx.x] = s;   // never true: keeps the chains alive
}

// dt for a step, on the device: either the host value or min(*dt_dev, dt_max).  The same launch
// clears the per-patch rate maxima the step's epilogue is about to accumulate for the new level.
__global__ void __launch_bounds__(256) k_set_dt(double* dst, const double* src, double host_dt, double dt_max,
                                                unsigned long long* __restrict__ rate_next, int np) {
  if (threadIdx.x == 0) {
    double dt = src ? *src : host_dt;
    if (dt_max > 0.0 && dt > dt_max) dt = dt_max;
    *dst = dt;
  }
  if (rate_next)
    for (int p = threadIdx.x; p < np; p += blockDim.x) rate_next[p] = 0ull;
}

// ------------------------------------------------------------------- step stages ----
// The body of every stage is a device function over an ACCESSOR x that says where the stage finds the
// state and the scratch arrays at "its" cell: HbmAcc = the bunch's arrays in HBM (the staged kernels
// below: one kernel per stage), TileAcc (tile_kernel.cuh) = a tile held in shared memory (all stages
// in one kernel).  x.u(f): field f of U^n, x.w(a): scratch array a, x.un(f): field f of U^{n+1} (always
// HBM), each a pointer AT the cell; x.s(d): element step for +1 along d (0 if collapsed).  Both paths
// therefore evaluate the same expressions in the same order (results agree to rounding: the compiler
// may contract multiply-adds differently in the two instantiations).
// limited slope of a stage: the accessor fixes the limiter at compile time (lim_kind 1 / 2) or leaves it to the
// descriptor (0).  minmod as a median is four min/max instructions instead of ten (27 slopes per cell in 3D, 18 in 2D).
template <typename X, typename T>
__device__ __forceinline__ T stage_slope(int kind, T a, T b) {
  if constexpr (X::lim_kind != 0) return limited_slope_k<X::lim_kind>(a, b);
  else return limited_slope(kind, a, b);
}
template <typename T> struct HbmAcc {
  static constexpr int lim_kind = 0;
  static constexpr bool def_solvers = false;
  const T* U; T* Un; T* W;
  long long ufs, wfs, cu, cw;
  long long st[3];
  int actv[3];
  __device__ __forceinline__ HbmAcc(const Params<T>& P, int pl, long long c)
      : U(P.U), Un(P.Un), W(P.W), ufs(P.G.fs), wfs(P.wfs), cu((long long)P.patch(pl) * P.G.ps + c), cw((long long)pl * P.G.ps + c) {
    st[0] = P.G.s[0]; st[1] = P.G.s[1]; st[2] = P.G.s[2];
    actv[0] = P.G.act[0]; actv[1] = P.G.act[1]; actv[2] = P.G.act[2];
  }
  __device__ __forceinline__ const T* u(int f) const { return U + f * ufs + cu; }
  __device__ __forceinline__ T* un(int f) const { return Un + f * ufs + cu; }
  __device__ __forceinline__ T* keep(int f) const { return Un + f * ufs + cu; }     // (unused: KEEP is false here)
  __device__ __forceinline__ T* w(int a) const { return W + a * wfs + cw; }
  __device__ __forceinline__ long long s(int d) const { return st[d]; }
  __device__ __forceinline__ bool act(int d) const { return actv[d] != 0; }     // run-time here, compile-time on a tile
};

// O2 (EOS L68): primitives on cells [-2, n+1]
template <typename T, typename X>
__device__ __forceinline__ void st_prim(const Params<T>& P, const X& x, int i, int j, int k, unsigned long long* __restrict__ bad) {
  const Geom& G = P.G;
  const T rho = x.u(0)[0], irho = num<T>::rcp(rho);
  const T u = x.u(1)[0] * irho, v = x.u(2)[0] * irho, w = x.u(3)[0] * irho;
  const T bx = T(0.5) * (x.u(5)[0] + x.u(5)[x.s(0)]);
  const T by = T(0.5) * (x.u(6)[0] + x.u(6)[x.s(1)]);
  const T bz = T(0.5) * (x.u(7)[0] + x.u(7)[x.s(2)]);
  const T pr = (P.gamma - T(1)) *
               (x.u(4)[0] - T(0.5) * rho * (u * u + v * v + w * w) - T(0.5) * (bx * bx + by * by + bz * bz));
  x.w(W_Q + 0)[0] = rho; x.w(W_Q + 1)[0] = u; x.w(W_Q + 2)[0] = v; x.w(W_Q + 3)[0] = w; x.w(W_Q + 4)[0] = pr;
  x.w(W_Q + 5)[0] = bx; x.w(W_Q + 6)[0] = by; x.w(W_Q + 7)[0] = bz;
  if (inside(G, i, j, k, 0, 0) && !(rho > T(0) && pr > T(0) && rho < T(INFINITY) && pr < T(INFINITY)))
    atomicAdd(bad, 1ull);
}

// O4a: Eq. 7-11 and cyclic images, edges [-1, n+1]
template <typename T, typename X>
__device__ __forceinline__ void st_emf0(const Params<T>& P, const X& x) {
  const long long sx = x.s(0), sy = x.s(1), sz = x.s(2);
  const T* u = x.w(W_Q + 1);
  const T* v = x.w(W_Q + 2);
  const T* w = x.w(W_Q + 3);
  const T* bx = x.u(5);
  const T* by = x.u(6);
  const T* bz = x.u(7);
  const T q4 = T(0.25), h = T(0.5);
  {  // ez = <u><By> - <v><Bx> over cells (i-1..i, j-1..j)
    const T ub = q4 * (u[0] + u[-sy] + u[-sx] + u[-sx - sy]);
    const T vb = q4 * (v[0] + v[-sy] + v[-sx] + v[-sx - sy]);
    x.w(W_E0 + 2)[0] = ub * (h * (by[0] + by[-sx])) - vb * (h * (bx[0] + bx[-sy]));
  }
  {  // ex = <v><Bz> - <w><By> over (j-1..j, k-1..k)
    const T vb = q4 * (v[0] + v[-sz] + v[-sy] + v[-sy - sz]);
    const T wb = q4 * (w[0] + w[-sz] + w[-sy] + w[-sy - sz]);
    x.w(W_E0 + 0)[0] = vb * (h * (bz[0] + bz[-sy])) - wb * (h * (by[0] + by[-sz]));
  }
  {  // ey = <w><Bx> - <u><Bz> over (k-1..k, i-1..i)
    const T wb = q4 * (w[0] + w[-sx] + w[-sz] + w[-sz - sx]);
    const T ub = q4 * (u[0] + u[-sx] + u[-sz] + u[-sz - sx]);
    x.w(W_E0 + 1)[0] = wb * (h * (bx[0] + bx[-sz])) - ub * (h * (bz[0] + bz[-sx]));
  }
}

// O3 + O4b + O4c: limited slopes and the half-step predictor
template <typename T, typename X>
__device__ __forceinline__ void st_predict(const Params<T>& P, const X& x, int i, int j, int k, T dt) {
  const Geom& G = P.G;
  const T hdt = T(0.5) * dt;
  const int cc[3] = {i, j, k};

  // half-step face fields: Eq. 12 with dt/2
  {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      const int b = (a + 1) % 3, e = (a + 2) % 3;
      // faces [-1, n+1] along a, [-1, n] transversally
      bool ok = true;
#pragma unroll
      for (int d = 0; d < 3; ++d)
        if (x.act(d)) ok = ok && (d == a ? true : cc[d] <= G.n[d]);
      if (!ok) continue;
      const T* Ee = x.w(W_E0 + e);
      const T* Eb = x.w(W_E0 + b);
      T curl = T(0);  // differences along a collapsed dimension vanish identically
      if (x.act(b)) curl += (Ee[x.s(b)] - Ee[0]) * P.idx[b];
      if (x.act(e)) curl -= (Eb[x.s(e)] - Eb[0]) * P.idx[e];
      x.w(W_BH + a)[0] = x.u(5 + a)[0] + hdt * curl;
    }
  }
  if (!inside(G, i, j, k, 1, 1)) return;

  T qc[8];
#pragma unroll
  for (int f = 0; f < 8; ++f) qc[f] = x.w(W_Q + f)[0];
  T dq[3][8];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
#pragma unroll
    for (int f = 0; f < 8; ++f) {
      T s = T(0);
      if (x.act(d) && f != 5 + d) {
        const T* qf = x.w(W_Q + f);
        s = stage_slope<X>(G.limiter, qc[f] - qf[-x.s(d)], qf[x.s(d)] - qc[f]);
      }
      if (f != 5 + d) x.w(W_DQ + d * 8 + f)[0] = s;  // the normal-field slot is never read
      dq[d][f] = s;
    }
  }
#pragma unroll
  for (int a = 0; a < 3; ++a) {
#pragma unroll
    for (int t = 0; t < 3; ++t) {
      if (t == a) continue;
      T s = T(0);
      if (x.act(t)) {
        const T* bf = x.u(5 + a);
        s = stage_slope<X>(G.limiter, bf[0] - bf[-x.s(t)], bf[x.s(t)] - bf[0]);
      }
      x.w(W_DBF + dbf_index(a, t))[0] = s;
    }
  }
  // primitive half step
  T lam[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) lam[d] = x.act(d) ? hdt * P.idx[d] : T(0);
  const T rho = qc[0], pr = qc[4], irho = num<T>::rcp(rho);
  T rho_h = rho, p_h = pr, vh[3] = {qc[1], qc[2], qc[3]};
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    const T ud = qc[1 + d], dud = dq[d][1 + d];
    rho_h -= lam[d] * (ud * dq[d][0] + rho * dud);
    p_h -= lam[d] * (ud * dq[d][4] + P.gamma * pr * dud);
#pragma unroll
    for (int a = 0; a < 3; ++a) vh[a] -= lam[d] * ud * dq[d][1 + a];
  }
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const int b = (a + 1) % 3, e = (a + 2) % 3;
    const T press = lam[a] * (dq[a][4] + qc[5 + b] * dq[a][5 + b] + qc[5 + e] * dq[a][5 + e]);
    const T tens = lam[b] * qc[5 + b] * dq[b][5 + a] + lam[e] * qc[5 + e] * dq[e][5 + a];
    vh[a] += (tens - press) * irho;
  }
  x.w(W_QH + 0)[0] = rho_h; x.w(W_QH + 1)[0] = vh[0]; x.w(W_QH + 2)[0] = vh[1]; x.w(W_QH + 3)[0] = vh[2]; x.w(W_QH + 4)[0] = p_h;
}

// O5 + O6: face states and HLLD flux through the lower face along D
template <typename T, int D, typename X>
__device__ __forceinline__ void st_flux(const Params<T>& P, const X& x) {
  const Geom& G = P.G;
  constexpr int T1 = (D + 1) % 3, T2 = (D + 2) % 3;
  const long long sd = x.s(D);
  const T h = T(0.5);
  State1D<T> L, R;
  // left state: upper face of cell c - e_D; right state: lower face of cell c
  L.rho = x.w(W_QH)[-sd] + h * x.w(W_DQ + D * 8)[-sd];                   R.rho = x.w(W_QH)[0] - h * x.w(W_DQ + D * 8)[0];
  L.u = x.w(W_QH + 1 + D)[-sd] + h * x.w(W_DQ + D * 8 + 1 + D)[-sd];     R.u = x.w(W_QH + 1 + D)[0] - h * x.w(W_DQ + D * 8 + 1 + D)[0];
  L.v = x.w(W_QH + 1 + T1)[-sd] + h * x.w(W_DQ + D * 8 + 1 + T1)[-sd];   R.v = x.w(W_QH + 1 + T1)[0] - h * x.w(W_DQ + D * 8 + 1 + T1)[0];
  L.w = x.w(W_QH + 1 + T2)[-sd] + h * x.w(W_DQ + D * 8 + 1 + T2)[-sd];   R.w = x.w(W_QH + 1 + T2)[0] - h * x.w(W_DQ + D * 8 + 1 + T2)[0];
  L.p = x.w(W_QH + 4)[-sd] + h * x.w(W_DQ + D * 8 + 4)[-sd];             R.p = x.w(W_QH + 4)[0] - h * x.w(W_DQ + D * 8 + 4)[0];
  // half-step centred transverse fields = mean of the two half-step faces
  const T* b1 = x.w(W_BH + T1);
  const T* b2 = x.w(W_BH + T2);
  L.by = h * (b1[-sd] + b1[-sd + x.s(T1)]) + h * x.w(W_DQ + D * 8 + 5 + T1)[-sd];
  R.by = h * (b1[0] + b1[x.s(T1)]) - h * x.w(W_DQ + D * 8 + 5 + T1)[0];
  L.bz = h * (b2[-sd] + b2[-sd + x.s(T2)]) + h * x.w(W_DQ + D * 8 + 5 + T2)[-sd];
  R.bz = h * (b2[0] + b2[x.s(T2)]) - h * x.w(W_DQ + D * 8 + 5 + T2)[0];
  const Flux5<T> F = riemann_flux(X::def_solvers ? 0 : G.flux_solver, P.gamma, L, R, x.w(W_BH + D)[0]);
  x.w(W_FLUX + D * 5)[0] = F.d; x.w(W_FLUX + D * 5 + 1 + D)[0] = F.mu; x.w(W_FLUX + D * 5 + 1 + T1)[0] = F.mv;
  x.w(W_FLUX + D * 5 + 1 + T2)[0] = F.mw; x.w(W_FLUX + D * 5 + 4)[0] = F.e;
}

// O5 + O7: corner states and the 2D Riemann problem at the edge along E
template <typename T, int E, typename X>
__device__ __forceinline__ void st_emf(const Params<T>& P, const X& x) {
  const Geom& G = P.G;
  constexpr int A = (E + 1) % 3, Bd = (E + 2) % 3;
  const long long sa = x.s(A), sb = x.s(Bd), se = x.s(E);
  const T h = T(0.5);
  // corner of cell at offset o seen with signs (sga, sgb)
  auto corner = [&](long long o, T sga, T sgb) {
    Corner<T> q;
    q.rho = x.w(W_QH)[o] + sga * h * x.w(W_DQ + A * 8)[o] + sgb * h * x.w(W_DQ + Bd * 8)[o];
    q.ua = x.w(W_QH + 1 + A)[o] + sga * h * x.w(W_DQ + A * 8 + 1 + A)[o] + sgb * h * x.w(W_DQ + Bd * 8 + 1 + A)[o];
    q.ub = x.w(W_QH + 1 + Bd)[o] + sga * h * x.w(W_DQ + A * 8 + 1 + Bd)[o] + sgb * h * x.w(W_DQ + Bd * 8 + 1 + Bd)[o];
    q.p = x.w(W_QH + 4)[o] + sga * h * x.w(W_DQ + A * 8 + 4)[o] + sgb * h * x.w(W_DQ + Bd * 8 + 4)[o];
    const T* be = x.w(W_BH + E) + o;
    q.be = h * (be[0] + be[se]) + sga * h * x.w(W_DQ + A * 8 + 5 + E)[o] + sgb * h * x.w(W_DQ + Bd * 8 + 5 + E)[o];
    return q;
  };
  // SW = RT of cell (a-1,b-1), SE = LT of (a,b-1), NW = RB of (a-1,b), NE = LB of (a,b)
  const Corner<T> sw = corner(-sa - sb, T(1), T(1)), se_ = corner(-sb, T(-1), T(1));
  const Corner<T> nw = corner(-sa, T(1), T(-1)), ne = corner(0, T(-1), T(-1));
  const T* dba = x.w(W_DBF + dbf_index(A, Bd));  // slope of b_A along B
  const T* dbb = x.w(W_DBF + dbf_index(Bd, A));  // slope of b_B along A
  const T* ba = x.w(W_BH + A);
  const T* bb = x.w(W_BH + Bd);
  const T AS = ba[-sb] + h * dba[-sb], AN = ba[0] - h * dba[0];
  const T BW = bb[-sa] + h * dbb[-sa], BE = bb[0] - h * dbb[0];
  x.w(W_EMF + E)[0] = emf_2d(P.gamma, X::def_solvers ? 0 : G.emf_solver, sw, se_, nw, ne, AS, AN, BW, BE);
}

// O8: conservative update + constrained transport with the metric factor of each term
// (Eq. 12; L154).  what: bit 0 the hydro fields, bit 1+a the face field b_a; store:
// write U^{n+1}; KEEP: also leave the new values in x.keep(f) (the tile kernel reduces the CFL rates of
// the new level from them, and forms -- without storing -- the faces another tile owns).
template <typename T, bool KEEP, typename X>
__device__ __forceinline__ void st_update(const Params<T>& P, const X& x, int i, int j, int k, T dt, int what = 15, bool store = true) {
  const Geom& G = P.G;
  const int cc[3] = {i, j, k};
  if ((what & 1) && inside(G, i, j, k, 0, 0)) {
#pragma unroll
    for (int f = 0; f < 5; ++f) {
      T v = x.u(f)[0];
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        if (!x.act(d)) continue;
        const T* fl = x.w(W_FLUX + d * 5 + f);
        v -= dt * P.idx[d] * (fl[x.s(d)] - fl[0]);
      }
      if (store) x.un(f)[0] = v;
      if (KEEP) x.keep(f)[0] = v;
    }
  }
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const int b = (a + 1) % 3, e = (a + 2) % 3;
    if (!(what & (2 << a))) continue;
    // faces 0..n along a (n = closing face), interior transversally
    bool ok = true;
#pragma unroll
    for (int d = 0; d < 3; ++d)
      if (x.act(d) && d != a) ok = ok && cc[d] < G.n[d];
    if (!ok) continue;
    const T* Ee = x.w(W_EMF + e);
    const T* Eb = x.w(W_EMF + b);
    T curl = T(0);
    if (x.act(b)) curl += (Ee[x.s(b)] - Ee[0]) * P.idx[b];
    if (x.act(e)) curl -= (Eb[x.s(e)] - Eb[0]) * P.idx[e];
    const T v = x.u(5 + a)[0] + dt * curl;
    if (store) x.un(5 + a)[0] = v;
    if (KEEP) x.keep(5 + a)[0] = v;
  }
}

// ---- the staged kernels: one stage each, arrays in HBM ----
template <typename T>
__global__ void __launch_bounds__(256) k_prim(Params<T> P, Box B, unsigned long long* __restrict__ bad) {
  int pl, i, j, k; long long c;
  if (!decode(P.G, B, P.npl, (long long)blockIdx.x * blockDim.x + threadIdx.x, pl, i, j, k, c)) return;
  st_prim<T>(P, HbmAcc<T>(P, pl, c), i, j, k, bad);
}
template <typename T>
__global__ void __launch_bounds__(256) k_emf0(Params<T> P, Box B) {
  int pl, i, j, k; long long c;
  if (!decode(P.G, B, P.npl, (long long)blockIdx.x * blockDim.x + threadIdx.x, pl, i, j, k, c)) return;
  st_emf0<T>(P, HbmAcc<T>(P, pl, c));
}
template <typename T>
__global__ void __launch_bounds__(256) k_predict(Params<T> P, Box B, const double* __restrict__ dtp) {
  int pl, i, j, k; long long c;
  if (!decode(P.G, B, P.npl, (long long)blockIdx.x * blockDim.x + threadIdx.x, pl, i, j, k, c)) return;
  st_predict<T>(P, HbmAcc<T>(P, pl, c), i, j, k, P.dt_of(pl, dtp));
}
template <typename T, int D>
__global__ void __launch_bounds__(256) k_flux(Params<T> P, Box B) {
  int pl, i, j, k; long long c;
  if (!decode(P.G, B, P.npl, (long long)blockIdx.x * blockDim.x + threadIdx.x, pl, i, j, k, c)) return;
  st_flux<T, D>(P, HbmAcc<T>(P, pl, c));
}
template <typename T, int E>
__global__ void __launch_bounds__(128) k_emf(Params<T> P, Box B) {
  int pl, i, j, k; long long c;
  if (!decode(P.G, B, P.npl, (long long)blockIdx.x * blockDim.x + threadIdx.x, pl, i, j, k, c)) return;
  st_emf<T, E>(P, HbmAcc<T>(P, pl, c));
}
template <typename T>
__global__ void __launch_bounds__(256) k_update(Params<T> P, Box B, const double* __restrict__ dtp) {
  int pl, i, j, k; long long c;
  if (!decode(P.G, B, P.npl, (long long)blockIdx.x * blockDim.x + threadIdx.x, pl, i, j, k, c)) return;
  st_update<T, false>(P, HbmAcc<T>(P, pl, c), i, j, k, P.dt_of(pl, dtp));
}

}  // namespace mhd
