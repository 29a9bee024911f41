// bunch_types.cuh -- geometry of a bunch in HBM, scratch-array map and kernel parameters.
#pragma once
#include <cuda_runtime.h>

namespace mhd {

// ---------------------------------------------------------------------- geometry ----
struct Geom {
  int n[3], g[3], m[3], act[3];
  int pitch, lead;
  long long s[3];      // element step for +1 along d (0 if collapsed)
  long long ps;        // elements per patch
  long long fs;        // elements per field of a state buffer (= npatch*ps)
  int np;
  int limiter, emf_solver, flux_solver;
};

struct Box { int lo[3], ext[3]; long long cells; };

inline Box make_box(const Geom& G, const int a[3], const int b[3]) {
  Box B;
  B.cells = 1;
  for (int d = 0; d < 3; ++d) {
    B.lo[d] = G.act[d] ? -a[d] : 0;
    B.ext[d] = G.act[d] ? G.n[d] + a[d] + b[d] : 1;
    B.cells *= B.ext[d];
  }
  return B;
}
inline Box make_box(const Geom& G, int a, int b) {
  const int aa[3] = {a, a, a}, bb[3] = {b, b, b};
  return make_box(G, aa, bb);
}

// thread -> (local patch, cell) inside a box; returns false past the end
__device__ __forceinline__ bool decode(const Geom& G, const Box& B, int npl, long long t, int& pl, int& i, int& j,
                                       int& k, long long& c) {
  if (t >= B.cells * npl) return false;
  pl = (int)(t / B.cells);
  int r = (int)(t - (long long)pl * B.cells);
  const int exy = B.ext[0] * B.ext[1];
  const int kk = r / exy;
  r -= kk * exy;
  const int jj = r / B.ext[0];
  const int ii = r - jj * B.ext[0];
  i = ii + B.lo[0]; j = jj + B.lo[1]; k = kk + B.lo[2];
  c = (long long)G.lead + (i + G.g[0]) + (long long)(j + G.g[1]) * G.pitch + (long long)(k + G.g[2]) * G.pitch * G.m[1];
  return true;
}

__device__ __forceinline__ bool inside(const Geom& G, int i, int j, int k, int a, int b) {
  const int c[3] = {i, j, k};
  bool ok = true;
#pragma unroll
  for (int d = 0; d < 3; ++d)
    if (G.act[d]) ok = ok && (c[d] >= -a) && (c[d] <= G.n[d] - 1 + b);
  return ok;
}

// scratch arrays of a chunk, all with the patch geometry of the state
enum : int {
  W_Q = 0,      // 8  primitives rho,u,v,w,p,Bcx,Bcy,Bcz
  W_DQ = 8,     // 24 slopes [dir][8] (normal-field slot unused)
  W_DBF = 32,   // 6  face-field transverse slopes: dy bx, dz bx, dx by, dz by, dx bz, dy bz
  W_E0 = 38,    // 3  edge EMFs at time n
  W_BH = 41,    // 3  half-step face fields
  W_QH = 44,    // 5  half-step rho,u,v,w,p
  W_FLUX = 49,  // 15 fluxes [dir][5]
  W_EMF = 64,   // 3  edge EMFs at n+1/2
  W_COUNT = 67,
  W_DCOUNT = 38  // arrays of the separate "D block" of the fused path (fused_kernels.cuh)
};

__host__ __device__ __forceinline__ int dbf_index(int a, int t) {
  // slope of face field b_a along t:  a=0: y->0 z->1; a=1: x->2 z->3; a=2: x->4 y->5
  return a == 0 ? (t == 1 ? 0 : 1) : (a == 1 ? (t == 0 ? 2 : 3) : (t == 0 ? 4 : 5));
}

// The D block (predictor output consumed by the fused Riemann/update kernel) has its own
// geometry: cells [-1, n] in every dimension, cell -1 at column/row/plane 0, row pitch a
// multiple of 16 bytes, so that every TMA box start (x0-1) is 16-byte aligned.
struct DGeom {
  int pitch, ny, nz;     // row pitch (elements), rows (n_y+2), planes (n_z+2)
  long long ps, fs;      // elements per patch, per array (= chunk*ps)
};

template <typename T> struct Params {
  Geom G;
  DGeom DG;
  T* D;            // D block base
  const T* U;      // current level (state origin applied)
  T* Un;           // next level
  T* W;            // scratch base
  long long wfs;   // elements per scratch array (= chunk*ps)
  int p0, npl;     // first patch and number of patches of this chunk
  T gamma, dx[3], idx[3];
  // Local time steps (mhd_bunch_step_local): the launch covers a LIST of patches, each with its
  // own dt; null for the ordinary launches over the patch range [p0, p0+npl) with one dt.
  const int* plist;       // DEVICE, [npl]: patch of local index pl
  const double* dtlist;   // DEVICE, [npl]: its time step
  __device__ __forceinline__ int patch(int pl) const { return plist ? plist[pl] : p0 + pl; }
  __device__ __forceinline__ T dt_of(int pl, const double* __restrict__ dtp) const { return (T)(dtlist ? dtlist[pl] : *dtp); }
};


}  // namespace mhd
