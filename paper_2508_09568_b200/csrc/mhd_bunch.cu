// mhd_bunch.cu -- C ABI (include/mhd_bunch.h) and sm_100a kernels of the bunch MHD update.
//
// Path (section 2.1.4): guard fill -> primitives -> limited slopes ->
// predictor (edge EMF at time n, half-step face fields, primitive half step) -> HLLD at
// faces -> 2D Riemann problem at edges -> conservative + constrained-transport update;
// CFL reduction.  One launch of each kernel covers a whole sub-bunch of patches.
//
// This file never allocates device memory after create and has no CPU fallback.
#include "../../include/mhd_bunch.h"
#include "mhd_math.cuh"

#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <string.h>
#include <new>
#include <vector>

namespace {

using namespace mhd;

thread_local char g_cuda_err[256] = "";

// ---------------------------------------------------------------------- geometry ----
struct Geom {
  int n[3], g[3], m[3], act[3];
  int pitch, lead;
  long long s[3];      // element step for +1 along d (0 if collapsed)
  long long ps;        // elements per patch
  long long fs;        // elements per field of a state buffer (= npatch*ps)
  int np;
  int limiter, emf_solver;
};

struct Box { int lo[3], ext[3]; long long cells; };

static Box make_box(const Geom& G, const int a[3], const int b[3]) {
  Box B;
  B.cells = 1;
  for (int d = 0; d < 3; ++d) {
    B.lo[d] = G.act[d] ? -a[d] : 0;
    B.ext[d] = G.act[d] ? G.n[d] + a[d] + b[d] : 1;
    B.cells *= B.ext[d];
  }
  return B;
}
static Box make_box(const Geom& G, int a, int b) {
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
  W_COUNT = 67
};

__host__ __device__ __forceinline__ int dbf_index(int a, int t) {
  // slope of face field b_a along t:  a=0: y->0 z->1; a=1: x->2 z->3; a=2: x->4 y->5
  return a == 0 ? (t == 1 ? 0 : 1) : (a == 1 ? (t == 0 ? 2 : 3) : (t == 0 ? 4 : 5));
}

template <typename T> struct Params {
  Geom G;
  const T* U;      // current level (state origin applied)
  T* Un;           // next level
  T* W;            // scratch base
  long long wfs;   // elements per scratch array (= chunk*ps)
  int p0, npl;     // first patch and number of patches of this chunk
  T gamma, dx[3], idx[3];
};

// -------------------------------------------------------------------- guard fill ----
// O1 (width 3 L212): every guard cell copies all 8 fields from
// the neighbour's interior image, or from the nearest own interior cell (zero gradient).
template <typename T>
__global__ void __launch_bounds__(256) k_fill_guards(Geom G, T* __restrict__ U, const int* __restrict__ nbr) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long per = (long long)G.m[0] * G.m[1] * G.m[2];
  if (t >= per * G.np) return;
  const int p = (int)(t / per);
  int r = (int)(t - (long long)p * per);
  const int mxy = G.m[0] * G.m[1];
  const int kk = r / mxy; r -= kk * mxy;
  const int jj = r / G.m[0];
  const int ii = r - jj * G.m[0];
  const int c[3] = {ii - G.g[0], jj - G.g[1], kk - G.g[2]};
  int o[3], src[3], cl[3];
  bool guard = false;
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    o[d] = c[d] < 0 ? -1 : (c[d] >= G.n[d] ? 1 : 0);
    guard = guard || (o[d] != 0);
    src[d] = c[d] - o[d] * G.n[d];
    cl[d] = min(max(c[d], 0), G.n[d] - 1);
  }
  if (!guard) return;
  const int q = nbr[p * 27 + (o[2] + 1) * 9 + (o[1] + 1) * 3 + (o[0] + 1)];
  const long long dst = (long long)p * G.ps + G.lead + ii + (long long)jj * G.pitch + (long long)kk * G.pitch * G.m[1];
  long long from;
  if (q >= 0)
    from = (long long)q * G.ps + G.lead + (src[0] + G.g[0]) + (long long)(src[1] + G.g[1]) * G.pitch +
           (long long)(src[2] + G.g[2]) * G.pitch * G.m[1];
  else
    from = (long long)p * G.ps + G.lead + (cl[0] + G.g[0]) + (long long)(cl[1] + G.g[1]) * G.pitch +
           (long long)(cl[2] + G.g[2]) * G.pitch * G.m[1];
#pragma unroll
  for (int f = 0; f < 8; ++f) {
    if (q < 0 && f >= 5) {  // the closing face keeps its evolved value (O8)
      const int a = f - 5, b = (a + 1) % 3, e = (a + 2) % 3;
      if (G.act[a] && c[a] == G.n[a] && o[b] == 0 && o[e] == 0) continue;
    }
    U[f * G.fs + dst] = U[f * G.fs + from];
  }
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
    const T rho = U[c], irho = num<T>::rcp(rho);
    const T u = U[G.fs + c] * irho, v = U[2 * G.fs + c] * irho, w = U[3 * G.fs + c] * irho;
    const T bx = T(0.5) * (U[5 * G.fs + c] + U[5 * G.fs + c + G.s[0]]);
    const T by = T(0.5) * (U[6 * G.fs + c] + U[6 * G.fs + c + G.s[1]]);
    const T bz = T(0.5) * (U[7 * G.fs + c] + U[7 * G.fs + c + G.s[2]]);
    const T b2 = bx * bx + by * by + bz * bz;
    const T pr = (P.gamma - T(1)) * (U[4 * G.fs + c] - T(0.5) * rho * (u * u + v * v + w * w) - T(0.5) * b2);
    const T gp = P.gamma * pr;
    T rate = T(0);
    if (G.act[0]) rate += (num<T>::abs(u) + fast_speed(gp, b2, bx * bx, irho)) * P.idx[0];
    if (G.act[1]) rate += (num<T>::abs(v) + fast_speed(gp, b2, by * by, irho)) * P.idx[1];
    if (G.act[2]) rate += (num<T>::abs(w) + fast_speed(gp, b2, bz * bz, irho)) * P.idx[2];
    double rd = (double)rate;
    if (!(rd == rd)) rd = INFINITY;  // a NaN cell forces dt = 0 rather than being ignored
    rmax = fmax(rmax, rd);
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

// dt for a step, on the device: either the host value or min(*dt_dev, dt_max)
__global__ void k_set_dt(double* dst, const double* src, double host_dt, double dt_max) {
  double dt = src ? *src : host_dt;
  if (dt_max > 0.0 && dt > dt_max) dt = dt_max;
  *dst = dt;
}

// ------------------------------------------------------------------- step stages ----
// O2 (EOS L68): primitives on cells [-2, n+1]
template <typename T>
__global__ void __launch_bounds__(256) k_prim(Params<T> P, Box B, unsigned long long* __restrict__ bad) {
  const Geom& G = P.G;
  int pl, i, j, k; long long c;
  if (!decode(G, B, P.npl, (long long)blockIdx.x * blockDim.x + threadIdx.x, pl, i, j, k, c)) return;
  const long long cu = (long long)(P.p0 + pl) * G.ps + c, cw = (long long)pl * G.ps + c;
  const T* U = P.U;
  const T rho = U[cu], irho = num<T>::rcp(rho);
  const T u = U[G.fs + cu] * irho, v = U[2 * G.fs + cu] * irho, w = U[3 * G.fs + cu] * irho;
  const T bx = T(0.5) * (U[5 * G.fs + cu] + U[5 * G.fs + cu + G.s[0]]);
  const T by = T(0.5) * (U[6 * G.fs + cu] + U[6 * G.fs + cu + G.s[1]]);
  const T bz = T(0.5) * (U[7 * G.fs + cu] + U[7 * G.fs + cu + G.s[2]]);
  const T pr = (P.gamma - T(1)) *
               (U[4 * G.fs + cu] - T(0.5) * rho * (u * u + v * v + w * w) - T(0.5) * (bx * bx + by * by + bz * bz));
  T* q = P.W + W_Q * P.wfs + cw;
  q[0] = rho; q[P.wfs] = u; q[2 * P.wfs] = v; q[3 * P.wfs] = w; q[4 * P.wfs] = pr;
  q[5 * P.wfs] = bx; q[6 * P.wfs] = by; q[7 * P.wfs] = bz;
  if (inside(G, i, j, k, 0, 0) && !(rho > T(0) && pr > T(0) && rho < T(INFINITY) && pr < T(INFINITY)))
    atomicAdd(bad, 1ull);
}

// O4a: Eq. 7-11 and cyclic images, edges [-1, n+1]
template <typename T>
__global__ void __launch_bounds__(256) k_emf0(Params<T> P, Box B) {
  const Geom& G = P.G;
  int pl, i, j, k; long long c;
  if (!decode(G, B, P.npl, (long long)blockIdx.x * blockDim.x + threadIdx.x, pl, i, j, k, c)) return;
  const long long cu = (long long)(P.p0 + pl) * G.ps + c, cw = (long long)pl * G.ps + c;
  const long long sx = G.s[0], sy = G.s[1], sz = G.s[2];
  const T* u = P.W + (W_Q + 1) * P.wfs + cw;
  const T* v = P.W + (W_Q + 2) * P.wfs + cw;
  const T* w = P.W + (W_Q + 3) * P.wfs + cw;
  const T* bx = P.U + 5 * G.fs + cu;
  const T* by = P.U + 6 * G.fs + cu;
  const T* bz = P.U + 7 * G.fs + cu;
  const T q4 = T(0.25), h = T(0.5);
  T* e0 = P.W + W_E0 * P.wfs + cw;
  {  // ez = <u><By> - <v><Bx> over cells (i-1..i, j-1..j)
    const T ub = q4 * (u[0] + u[-sy] + u[-sx] + u[-sx - sy]);
    const T vb = q4 * (v[0] + v[-sy] + v[-sx] + v[-sx - sy]);
    e0[2 * P.wfs] = ub * (h * (by[0] + by[-sx])) - vb * (h * (bx[0] + bx[-sy]));
  }
  {  // ex = <v><Bz> - <w><By> over (j-1..j, k-1..k)
    const T vb = q4 * (v[0] + v[-sz] + v[-sy] + v[-sy - sz]);
    const T wb = q4 * (w[0] + w[-sz] + w[-sy] + w[-sy - sz]);
    e0[0] = vb * (h * (bz[0] + bz[-sy])) - wb * (h * (by[0] + by[-sz]));
  }
  {  // ey = <w><Bx> - <u><Bz> over (k-1..k, i-1..i)
    const T wb = q4 * (w[0] + w[-sx] + w[-sz] + w[-sz - sx]);
    const T ub = q4 * (u[0] + u[-sx] + u[-sz] + u[-sz - sx]);
    e0[P.wfs] = wb * (h * (bx[0] + bx[-sz])) - ub * (h * (bz[0] + bz[-sx]));
  }
}

// O3 + O4b + O4c: limited slopes and the half-step predictor
template <typename T>
__global__ void __launch_bounds__(256) k_predict(Params<T> P, Box B, const double* __restrict__ dtp) {
  const Geom& G = P.G;
  int pl, i, j, k; long long c;
  if (!decode(G, B, P.npl, (long long)blockIdx.x * blockDim.x + threadIdx.x, pl, i, j, k, c)) return;
  const long long cu = (long long)(P.p0 + pl) * G.ps + c, cw = (long long)pl * G.ps + c;
  const T dt = (T)(*dtp);
  const T hdt = T(0.5) * dt;
  const long long wfs = P.wfs;
  const int cc[3] = {i, j, k};

  // half-step face fields: Eq. 12 with dt/2
  {
    const T* e0 = P.W + W_E0 * wfs + cw;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      const int b = (a + 1) % 3, e = (a + 2) % 3;
      // faces [-1, n+1] along a, [-1, n] transversally
      bool ok = true;
#pragma unroll
      for (int d = 0; d < 3; ++d)
        if (G.act[d]) ok = ok && (d == a ? true : cc[d] <= G.n[d]);
      if (!ok) continue;
      const T* Ee = e0 + e * wfs;
      const T* Eb = e0 + b * wfs;
      T curl = T(0);  // differences along a collapsed dimension vanish identically
      if (G.act[b]) curl += (Ee[G.s[b]] - Ee[0]) * P.idx[b];
      if (G.act[e]) curl -= (Eb[G.s[e]] - Eb[0]) * P.idx[e];
      P.W[(W_BH + a) * wfs + cw] = P.U[(5 + a) * G.fs + cu] + hdt * curl;
    }
  }
  if (!inside(G, i, j, k, 1, 1)) return;

  const T* q = P.W + W_Q * wfs + cw;
  T qc[8];
#pragma unroll
  for (int f = 0; f < 8; ++f) qc[f] = q[f * wfs];
  T dq[3][8];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
#pragma unroll
    for (int f = 0; f < 8; ++f) {
      T s = T(0);
      if (G.act[d] && f != 5 + d) {
        const T* qf = q + f * wfs;
        s = limited_slope(G.limiter, qc[f] - qf[-G.s[d]], qf[G.s[d]] - qc[f]);
      }
      if (f != 5 + d) P.W[(W_DQ + d * 8 + f) * wfs + cw] = s;  // the normal-field slot is never read
      dq[d][f] = s;
    }
  }
#pragma unroll
  for (int a = 0; a < 3; ++a) {
#pragma unroll
    for (int t = 0; t < 3; ++t) {
      if (t == a) continue;
      T s = T(0);
      if (G.act[t]) {
        const T* bf = P.U + (5 + a) * G.fs + cu;
        s = limited_slope(G.limiter, bf[0] - bf[-G.s[t]], bf[G.s[t]] - bf[0]);
      }
      P.W[(W_DBF + dbf_index(a, t)) * wfs + cw] = s;
    }
  }
  // primitive half step
  T lam[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) lam[d] = G.act[d] ? hdt * P.idx[d] : T(0);
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
  T* qh = P.W + W_QH * wfs + cw;
  qh[0] = rho_h; qh[wfs] = vh[0]; qh[2 * wfs] = vh[1]; qh[3 * wfs] = vh[2]; qh[4 * wfs] = p_h;
}

// O5 + O6: face states and HLLD flux through the lower face along D
template <typename T, int D>
__global__ void __launch_bounds__(256) k_flux(Params<T> P, Box B) {
  const Geom& G = P.G;
  int pl, i, j, k; long long c;
  if (!decode(G, B, P.npl, (long long)blockIdx.x * blockDim.x + threadIdx.x, pl, i, j, k, c)) return;
  const long long cw = (long long)pl * G.ps + c, wfs = P.wfs;
  constexpr int T1 = (D + 1) % 3, T2 = (D + 2) % 3;
  const long long sd = G.s[D];
  const T* qh = P.W + W_QH * wfs + cw;
  const T* dq = P.W + (W_DQ + D * 8) * wfs + cw;
  const T* bh = P.W + W_BH * wfs + cw;
  const T h = T(0.5);
  State1D<T> L, R;
  // left state: upper face of cell c - e_D; right state: lower face of cell c
  L.rho = qh[-sd] + h * dq[-sd];                               R.rho = qh[0] - h * dq[0];
  L.u = qh[(1 + D) * wfs - sd] + h * dq[(1 + D) * wfs - sd];   R.u = qh[(1 + D) * wfs] - h * dq[(1 + D) * wfs];
  L.v = qh[(1 + T1) * wfs - sd] + h * dq[(1 + T1) * wfs - sd]; R.v = qh[(1 + T1) * wfs] - h * dq[(1 + T1) * wfs];
  L.w = qh[(1 + T2) * wfs - sd] + h * dq[(1 + T2) * wfs - sd]; R.w = qh[(1 + T2) * wfs] - h * dq[(1 + T2) * wfs];
  L.p = qh[4 * wfs - sd] + h * dq[4 * wfs - sd];               R.p = qh[4 * wfs] - h * dq[4 * wfs];
  // half-step centred transverse fields = mean of the two half-step faces
  const T* b1 = bh + T1 * wfs;
  const T* b2 = bh + T2 * wfs;
  L.by = h * (b1[-sd] + b1[-sd + G.s[T1]]) + h * dq[(5 + T1) * wfs - sd];
  R.by = h * (b1[0] + b1[G.s[T1]]) - h * dq[(5 + T1) * wfs];
  L.bz = h * (b2[-sd] + b2[-sd + G.s[T2]]) + h * dq[(5 + T2) * wfs - sd];
  R.bz = h * (b2[0] + b2[G.s[T2]]) - h * dq[(5 + T2) * wfs];
  const Flux5<T> F = hlld_flux(P.gamma, L, R, bh[D * wfs]);
  T* fl = P.W + (W_FLUX + D * 5) * wfs + cw;
  fl[0] = F.d; fl[(1 + D) * wfs] = F.mu; fl[(1 + T1) * wfs] = F.mv; fl[(1 + T2) * wfs] = F.mw; fl[4 * wfs] = F.e;
}

// O5 + O7: corner states and the 2D Riemann problem at the edge along E
template <typename T, int E>
__global__ void __launch_bounds__(128) k_emf(Params<T> P, Box B) {
  const Geom& G = P.G;
  int pl, i, j, k; long long c;
  if (!decode(G, B, P.npl, (long long)blockIdx.x * blockDim.x + threadIdx.x, pl, i, j, k, c)) return;
  const long long cw = (long long)pl * G.ps + c, wfs = P.wfs;
  constexpr int A = (E + 1) % 3, Bd = (E + 2) % 3;
  const long long sa = G.s[A], sb = G.s[Bd], se = G.s[E];
  const T* qh = P.W + W_QH * wfs + cw;
  const T* da = P.W + (W_DQ + A * 8) * wfs + cw;
  const T* db = P.W + (W_DQ + Bd * 8) * wfs + cw;
  const T* bh = P.W + W_BH * wfs + cw;
  const T h = T(0.5);
  // corner of cell at offset o seen with signs (sga, sgb)
  auto corner = [&](long long o, T sga, T sgb) {
    Corner<T> q;
    q.rho = qh[o] + sga * h * da[o] + sgb * h * db[o];
    q.ua = qh[(1 + A) * wfs + o] + sga * h * da[(1 + A) * wfs + o] + sgb * h * db[(1 + A) * wfs + o];
    q.ub = qh[(1 + Bd) * wfs + o] + sga * h * da[(1 + Bd) * wfs + o] + sgb * h * db[(1 + Bd) * wfs + o];
    q.p = qh[4 * wfs + o] + sga * h * da[4 * wfs + o] + sgb * h * db[4 * wfs + o];
    const T* be = bh + E * wfs + o;
    q.be = h * (be[0] + be[se]) + sga * h * da[(5 + E) * wfs + o] + sgb * h * db[(5 + E) * wfs + o];
    return q;
  };
  // SW = RT of cell (a-1,b-1), SE = LT of (a,b-1), NW = RB of (a-1,b), NE = LB of (a,b)
  const Corner<T> sw = corner(-sa - sb, T(1), T(1)), se_ = corner(-sb, T(-1), T(1));
  const Corner<T> nw = corner(-sa, T(1), T(-1)), ne = corner(0, T(-1), T(-1));
  const T* dba = P.W + (W_DBF + dbf_index(A, Bd)) * wfs + cw;  // slope of b_A along B
  const T* dbb = P.W + (W_DBF + dbf_index(Bd, A)) * wfs + cw;  // slope of b_B along A
  const T* ba = bh + A * wfs;
  const T* bb = bh + Bd * wfs;
  const T AS = ba[-sb] + h * dba[-sb], AN = ba[0] - h * dba[0];
  const T BW = bb[-sa] + h * dbb[-sa], BE = bb[0] - h * dbb[0];
  P.W[(W_EMF + E) * wfs + cw] = emf_2d(P.gamma, G.emf_solver, sw, se_, nw, ne, AS, AN, BW, BE);
}

// O8: conservative update + constrained transport with the metric factor of each term
// (Eq. 12; L154)
template <typename T>
__global__ void __launch_bounds__(256) k_update(Params<T> P, Box B, const double* __restrict__ dtp) {
  const Geom& G = P.G;
  int pl, i, j, k; long long c;
  if (!decode(G, B, P.npl, (long long)blockIdx.x * blockDim.x + threadIdx.x, pl, i, j, k, c)) return;
  const long long cu = (long long)(P.p0 + pl) * G.ps + c, cw = (long long)pl * G.ps + c, wfs = P.wfs;
  const T dt = (T)(*dtp);
  const int cc[3] = {i, j, k};
  if (inside(G, i, j, k, 0, 0)) {
#pragma unroll
    for (int f = 0; f < 5; ++f) {
      T v = P.U[f * G.fs + cu];
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        if (!G.act[d]) continue;
        const T* fl = P.W + (W_FLUX + d * 5 + f) * wfs + cw;
        v -= dt * P.idx[d] * (fl[G.s[d]] - fl[0]);
      }
      P.Un[f * G.fs + cu] = v;
    }
  }
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const int b = (a + 1) % 3, e = (a + 2) % 3;
    // faces 0..n along a (n = closing face), interior transversally
    bool ok = true;
#pragma unroll
    for (int d = 0; d < 3; ++d)
      if (G.act[d] && d != a) ok = ok && cc[d] < G.n[d];
    if (!ok) continue;
    const T* Ee = P.W + (W_EMF + e) * wfs + cw;
    const T* Eb = P.W + (W_EMF + b) * wfs + cw;
    T curl = T(0);
    if (G.act[b]) curl += (Ee[G.s[b]] - Ee[0]) * P.idx[b];
    if (G.act[e]) curl -= (Eb[G.s[e]] - Eb[0]) * P.idx[e];
    P.Un[(5 + a) * G.fs + cu] = P.U[(5 + a) * G.fs + cu] + dt * curl;
  }
}

}  // namespace

// ------------------------------------------------------------------------ handle ----
struct mhd_bunch {
  mhd_bunch_desc desc;
  mhd_bunch_layout lay;
  Geom G;
  void* state[2];
  int cur;
  char* ws;
  size_t ws_bytes;
  int chunk;
  // carved from the workspace head
  int* d_nbr;
  unsigned long long* d_rate;  // [npatch]
  unsigned long long* d_bad;   // [1]
  double* d_dt;                // [2]: cfl result, step dt
  char* d_scratch;
  cudaStream_t stream;
  long long launches;
  size_t esz;
  // optional per-kernel-class timing (host-side objects only)
  bool timing;
  struct Ev { int cls; cudaEvent_t a, b; };
  std::vector<Ev>* events;
  double cls_ms[16];
  long long cls_n[16];
};

enum KClass : int { KC_FILL = 0, KC_CFL, KC_PRIM, KC_EMF0, KC_PREDICT, KC_FLUX, KC_EMF, KC_UPDATE, KC_MISC, KC_COUNT };
static const char* const kclass_names[KC_COUNT] = {"fill_guards", "cfl", "prim", "emf0", "predict", "hlld_flux",
                                                   "emf_2d", "update", "misc"};

// brackets one launch with events when timing is on
struct LaunchScope {
  mhd_bunch* b; int cls; cudaEvent_t a, e;
  LaunchScope(mhd_bunch* b_, int cls_) : b(b_), cls(cls_), a(nullptr), e(nullptr) {
    b->launches += 1;
    if (b->timing) {
      cudaEventCreate(&a); cudaEventCreate(&e);
      cudaEventRecord(a, b->stream);
    }
  }
  ~LaunchScope() {
    if (b->timing) {
      cudaEventRecord(e, b->stream);
      b->events->push_back({cls, a, e});
    }
  }
};

namespace {

int fail_cuda(cudaError_t e, const char* what) {
  snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s", what, cudaGetErrorString(e));
  return MHD_ECUDA;
}
#define CUDA_TRY(x)                              \
  do {                                           \
    cudaError_t e_ = (x);                        \
    if (e_ != cudaSuccess) return fail_cuda(e_, #x); \
  } while (0)

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

int build_geom(const mhd_bunch_desc* d, Geom* G) {
  if (!d) return MHD_EINVAL;
  if (d->ng != 3 || d->npatch < 1) return MHD_EINVAL;
  if (d->dtype != MHD_F32 && d->dtype != MHD_F64) return MHD_EINVAL;
  if (d->limiter != 1 && d->limiter != 2) return MHD_EINVAL;
  if (d->emf_solver != 0 && d->emf_solver != 1) return MHD_EINVAL;
  if (!(d->gamma > 1.0) || !isfinite(d->gamma)) return MHD_EINVAL;
  int nact = 0;
  for (int a = 0; a < 3; ++a) {
    if (d->n[a] < 1) return MHD_EINVAL;
    if (d->n[a] > 1 && d->n[a] < d->ng) return MHD_EINVAL;  // a neighbour's interior must fill the whole guard shell
    if (d->n[a] > 1024) return MHD_EINVAL;
    if (!(d->dx[a] > 0.0) || !isfinite(d->dx[a])) return MHD_EINVAL;
    G->n[a] = d->n[a];
    G->act[a] = d->n[a] > 1;
    G->g[a] = G->act[a] ? d->ng : 0;
    G->m[a] = d->n[a] + 2 * G->g[a];
    nact += G->act[a];
  }
  if (nact == 0) return MHD_EINVAL;
  if (G->act[0]) {
    G->lead = (4 - d->ng % 4) % 4;  // interior cell 0 on a 16-byte boundary
    G->pitch = (int)align_up((size_t)(G->lead + G->m[0]), 4);
  } else {
    G->lead = 0;
    G->pitch = 1;
  }
  G->ps = (long long)align_up((size_t)G->pitch * G->m[1] * G->m[2], 4);
  G->s[0] = G->act[0] ? 1 : 0;
  G->s[1] = G->act[1] ? G->pitch : 0;
  G->s[2] = G->act[2] ? (long long)G->pitch * G->m[1] : 0;
  G->np = d->npatch;
  G->fs = (long long)d->npatch * G->ps;
  G->limiter = d->limiter;
  G->emf_solver = d->emf_solver;
  return MHD_OK;
}

size_t head_bytes(int np) {
  return align_up(sizeof(int) * 27 * (size_t)np, 256) + align_up(sizeof(unsigned long long) * (size_t)np, 256) + 256 + 256;
}
size_t scratch_bytes(const Geom& G, size_t esz, int chunk) { return (size_t)W_COUNT * chunk * G.ps * esz; }

template <typename T>
Params<T> make_params(const mhd_bunch* b, int p0, int npl) {
  Params<T> P;
  P.G = b->G;
  P.U = (const T*)b->state[b->cur] ;
  P.Un = (T*)b->state[1 - b->cur];
  P.W = (T*)b->d_scratch;
  P.wfs = (long long)b->chunk * b->G.ps;
  P.p0 = p0;
  P.npl = npl;
  P.gamma = (T)b->desc.gamma;
  for (int a = 0; a < 3; ++a) {
    P.dx[a] = (T)b->desc.dx[a];
    P.idx[a] = (T)(1.0 / b->desc.dx[a]);
  }
  return P;
}

inline unsigned blocks_for(long long threads, int bs) { return (unsigned)((threads + bs - 1) / bs); }

template <typename T>
int launch_fill(mhd_bunch* b) {
  const Geom& G = b->G;
  const long long tot = (long long)G.m[0] * G.m[1] * G.m[2] * G.np;
  { LaunchScope ls(b, KC_FILL);
    k_fill_guards<T><<<blocks_for(tot, 256), 256, 0, b->stream>>>(G, (T*)b->state[b->cur], b->d_nbr); }
  CUDA_TRY(cudaGetLastError());
  return MHD_OK;
}

template <typename T>
int launch_cfl(mhd_bunch* b, double courant, void* dt_dev, void* dt_patch) {
  const Geom& G = b->G;
  Params<T> P = make_params<T>(b, 0, G.np);
  { LaunchScope ls(b, KC_MISC); k_zero_u64<<<blocks_for(G.np, 256), 256, 0, b->stream>>>(b->d_rate, G.np); }
  const long long per = (long long)G.n[0] * G.n[1] * G.n[2];
  int bx = (int)((per + 256 * 8 - 1) / (256 * 8));
  if (bx < 1) bx = 1;
  dim3 grid((unsigned)bx, (unsigned)G.np);
  { LaunchScope ls(b, KC_CFL); k_cfl<T><<<grid, 256, 0, b->stream>>>(P, b->d_rate); }
  { LaunchScope ls(b, KC_MISC);
    k_cfl_final<<<1, 256, 0, b->stream>>>(b->d_rate, G.np, courant, b->d_dt, (double*)dt_dev, (double*)dt_patch); }
  CUDA_TRY(cudaGetLastError());
  return MHD_OK;
}

template <typename T>
int launch_step(mhd_bunch* b) {
  const Geom& G = b->G;
  const double* dtp = b->d_dt + 1;
  for (int p0 = 0; p0 < G.np; p0 += b->chunk) {
    const int npl = (G.np - p0 < b->chunk) ? G.np - p0 : b->chunk;
    Params<T> P = make_params<T>(b, p0, npl);
    cudaStream_t st = b->stream;
    {
      Box B = make_box(G, 2, 2);
      LaunchScope ls(b, KC_PRIM);
      k_prim<T><<<blocks_for(B.cells * npl, 256), 256, 0, st>>>(P, B, b->d_bad);
    }
    {
      Box B = make_box(G, 1, 2);
      { LaunchScope ls(b, KC_EMF0); k_emf0<T><<<blocks_for(B.cells * npl, 256), 256, 0, st>>>(P, B); }
      { LaunchScope ls(b, KC_PREDICT); k_predict<T><<<blocks_for(B.cells * npl, 256), 256, 0, st>>>(P, B, dtp); }
    }
    for (int d = 0; d < 3; ++d) {
      if (!G.act[d]) continue;
      int a[3] = {0, 0, 0}, e[3] = {0, 0, 0};
      e[d] = 1;
      Box B = make_box(G, a, e);
      const unsigned nb = blocks_for(B.cells * npl, 256);
      LaunchScope ls(b, KC_FLUX);
      if (d == 0) k_flux<T, 0><<<nb, 256, 0, st>>>(P, B);
      if (d == 1) k_flux<T, 1><<<nb, 256, 0, st>>>(P, B);
      if (d == 2) k_flux<T, 2><<<nb, 256, 0, st>>>(P, B);
    }
    for (int ed = 0; ed < 3; ++ed) {
      const int A = (ed + 1) % 3, Bd = (ed + 2) % 3;
      if (!G.act[A] && !G.act[Bd]) continue;  // enters the update only through differences that vanish
      int a[3] = {0, 0, 0}, e[3] = {0, 0, 0};
      e[A] = 1; e[Bd] = 1;
      Box B = make_box(G, a, e);
      const unsigned nb = blocks_for(B.cells * npl, 128);
      LaunchScope ls(b, KC_EMF);
      if (ed == 0) k_emf<T, 0><<<nb, 128, 0, st>>>(P, B);
      if (ed == 1) k_emf<T, 1><<<nb, 128, 0, st>>>(P, B);
      if (ed == 2) k_emf<T, 2><<<nb, 128, 0, st>>>(P, B);
    }
    {
      Box B = make_box(G, 0, 1);
      LaunchScope ls(b, KC_UPDATE);
      k_update<T><<<blocks_for(B.cells * npl, 256), 256, 0, st>>>(P, B, dtp);
    }
  }
  CUDA_TRY(cudaGetLastError());
  b->cur = 1 - b->cur;
  return MHD_OK;
}

}  // namespace

// --------------------------------------------------------------------------- ABI ----
extern "C" {

const char* mhd_bunch_strerror(int code) {
  switch (code) {
    case MHD_OK: return "ok";
    case MHD_EINVAL: return "invalid argument or unsupported configuration";
    case MHD_ENOMEM: return "workspace too small";
    case MHD_ECUDA: return "CUDA runtime error";
    case MHD_ESTATE: return "invalid handle state";
    default: return "unknown error";
  }
}

const char* mhd_bunch_last_cuda_error(void) { return g_cuda_err; }

int mhd_bunch_query(const mhd_bunch_desc* desc, mhd_bunch_layout* lay) {
  if (!desc || !lay) return MHD_EINVAL;
  Geom G;
  const int rc = build_geom(desc, &G);
  if (rc != MHD_OK) return rc;
  const size_t esz = desc->dtype == MHD_F64 ? 8 : 4;
  memset(lay, 0, sizeof(*lay));
  lay->stride[0] = G.fs;
  lay->stride[1] = G.ps;
  lay->stride[2] = (long long)G.pitch * G.m[1];
  lay->stride[3] = G.pitch;
  lay->stride[4] = 1;
  lay->origin = G.lead;
  lay->state_elems = 8 * G.fs;
  lay->state_bytes = (size_t)lay->state_elems * esz;
  lay->workspace_min = head_bytes(G.np) + scratch_bytes(G, esz, 1);
  // enough patches per chunk to fill the machine a few times over; capped at 4 GiB of scratch
  int chunk = G.np;
  const size_t cap = (size_t)4 << 30;
  while (chunk > 1 && scratch_bytes(G, esz, chunk) > cap) chunk = (chunk + 1) / 2;
  lay->workspace_best = head_bytes(G.np) + scratch_bytes(G, esz, chunk);
  for (int a = 0; a < 3; ++a) lay->m[a] = G.m[a];
  return MHD_OK;
}

int mhd_bunch_create(const mhd_bunch_desc* desc, const int32_t* nbr, void* state_a, void* state_b, void* workspace,
                     size_t workspace_bytes, mhd_bunch** out) {
  if (!desc || !nbr || !state_a || !state_b || !workspace || !out) return MHD_EINVAL;
  if (state_a == state_b) return MHD_EINVAL;
  if (((uintptr_t)state_a | (uintptr_t)state_b | (uintptr_t)workspace) & 15) return MHD_EINVAL;
  mhd_bunch_layout lay;
  int rc = mhd_bunch_query(desc, &lay);
  if (rc != MHD_OK) return rc;
  {  // the buffers must not overlap
    const char *a = (const char*)state_a, *b2 = (const char*)state_b;
    if ((a < b2 && a + lay.state_bytes > b2) || (b2 < a && b2 + lay.state_bytes > a)) return MHD_EINVAL;
  }
  for (int p = 0; p < desc->npatch; ++p)
    for (int c = 0; c < 27; ++c) {
      const int q = nbr[p * 27 + c];
      if (q < -1 || q >= desc->npatch) return MHD_EINVAL;
    }
  if (workspace_bytes < lay.workspace_min) return MHD_ENOMEM;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= desc->device || desc->device < 0)
    return fail_cuda(cudaErrorNoDevice, "no CUDA device: this library has no CPU fallback");
  CUDA_TRY(cudaSetDevice(desc->device));

  mhd_bunch* b = new (std::nothrow) mhd_bunch;
  if (!b) return MHD_ENOMEM;
  memset(b, 0, sizeof(*b));
  b->events = new (std::nothrow) std::vector<mhd_bunch::Ev>();
  if (!b->events) { delete b; return MHD_ENOMEM; }
  b->desc = *desc;
  b->lay = lay;
  build_geom(desc, &b->G);
  b->esz = desc->dtype == MHD_F64 ? 8 : 4;
  b->state[0] = state_a;
  b->state[1] = state_b;
  b->cur = 0;
  b->ws = (char*)workspace;
  b->ws_bytes = workspace_bytes;
  b->stream = (cudaStream_t)desc->stream;
  char* p = b->ws;
  b->d_nbr = (int*)p;                 p += align_up(sizeof(int) * 27 * (size_t)desc->npatch, 256);
  b->d_rate = (unsigned long long*)p; p += align_up(sizeof(unsigned long long) * (size_t)desc->npatch, 256);
  b->d_bad = (unsigned long long*)p;  p += 256;
  b->d_dt = (double*)p;               p += 256;
  b->d_scratch = p;
  const size_t avail = workspace_bytes - (size_t)(p - b->ws);
  long long chunk = (long long)(avail / scratch_bytes(b->G, b->esz, 1));
  if (chunk > desc->npatch) chunk = desc->npatch;
  if (chunk < 1) { delete b; return MHD_ENOMEM; }
  b->chunk = (int)chunk;
  cudaError_t e = cudaMemcpyAsync(b->d_nbr, nbr, sizeof(int) * 27 * (size_t)desc->npatch, cudaMemcpyHostToDevice, b->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(b->d_bad, 0, 512, b->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(b->stream);
  if (e != cudaSuccess) { delete b; return fail_cuda(e, "create: table upload"); }
  *out = b;
  return MHD_OK;
}

int mhd_bunch_fill_guards(mhd_bunch* b) {
  if (!b) return MHD_ESTATE;
  return b->desc.dtype == MHD_F64 ? launch_fill<double>(b) : launch_fill<float>(b);
}

int mhd_bunch_cfl_dt(mhd_bunch* b, double courant, double* dt_host, void* dt_dev, void* dt_per_patch_dev) {
  if (!b) return MHD_ESTATE;
  if (!(courant > 0.0) || !isfinite(courant)) return MHD_EINVAL;
  const int rc = b->desc.dtype == MHD_F64 ? launch_cfl<double>(b, courant, dt_dev, dt_per_patch_dev)
                                           : launch_cfl<float>(b, courant, dt_dev, dt_per_patch_dev);
  if (rc != MHD_OK) return rc;
  if (dt_host) {
    CUDA_TRY(cudaMemcpyAsync(dt_host, b->d_dt, sizeof(double), cudaMemcpyDeviceToHost, b->stream));
    CUDA_TRY(cudaStreamSynchronize(b->stream));
  }
  return MHD_OK;
}

static int step_common(mhd_bunch* b) {
  return b->desc.dtype == MHD_F64 ? launch_step<double>(b) : launch_step<float>(b);
}

int mhd_bunch_step(mhd_bunch* b, double dt) {
  if (!b) return MHD_ESTATE;
  if (!(dt > 0.0) || !isfinite(dt)) return MHD_EINVAL;
  { LaunchScope ls(b, KC_MISC); k_set_dt<<<1, 1, 0, b->stream>>>(b->d_dt + 1, nullptr, dt, 0.0); }
  return step_common(b);
}

int mhd_bunch_step_dev(mhd_bunch* b, const void* dt_dev, double dt_max) {
  if (!b) return MHD_ESTATE;
  if (!dt_dev || !(dt_max >= 0.0)) return MHD_EINVAL;
  { LaunchScope ls(b, KC_MISC); k_set_dt<<<1, 1, 0, b->stream>>>(b->d_dt + 1, (const double*)dt_dev, 0.0, dt_max); }
  return step_common(b);
}

int mhd_bunch_current(mhd_bunch* b, void** state) {
  if (!b || !state) return MHD_ESTATE;
  *state = b->state[b->cur];
  return MHD_OK;
}

int mhd_bunch_status(mhd_bunch* b, int64_t* bad_cells) {
  if (!b || !bad_cells) return MHD_ESTATE;
  unsigned long long v = 0;
  CUDA_TRY(cudaMemcpyAsync(&v, b->d_bad, sizeof(v), cudaMemcpyDeviceToHost, b->stream));
  CUDA_TRY(cudaStreamSynchronize(b->stream));
  *bad_cells = (int64_t)v;
  return MHD_OK;
}

int mhd_bunch_launch_count(mhd_bunch* b, int64_t* launches) {
  if (!b || !launches) return MHD_ESTATE;
  *launches = b->launches;
  return MHD_OK;
}

int mhd_bunch_chunk(mhd_bunch* b, int32_t* chunk_patches) {
  if (!b || !chunk_patches) return MHD_ESTATE;
  *chunk_patches = b->chunk;
  return MHD_OK;
}

static void drain_events(mhd_bunch* b, bool accumulate) {
  for (auto& ev : *b->events) {
    if (accumulate) {
      float ms = 0.f;
      if (cudaEventElapsedTime(&ms, ev.a, ev.b) == cudaSuccess) {
        b->cls_ms[ev.cls] += ms;
        b->cls_n[ev.cls] += 1;
      }
    }
    cudaEventDestroy(ev.a);
    cudaEventDestroy(ev.b);
  }
  b->events->clear();
}

int mhd_bunch_upload(mhd_bunch* b, const void* host_state) {
  if (!b || !host_state) return MHD_ESTATE;
  CUDA_TRY(cudaMemcpyAsync(b->state[b->cur], host_state, b->lay.state_bytes, cudaMemcpyHostToDevice, b->stream));
  return MHD_OK;
}

int mhd_bunch_download(mhd_bunch* b, void* host_state) {
  if (!b || !host_state) return MHD_ESTATE;
  CUDA_TRY(cudaMemcpyAsync(host_state, b->state[b->cur], b->lay.state_bytes, cudaMemcpyDeviceToHost, b->stream));
  CUDA_TRY(cudaStreamSynchronize(b->stream));
  return MHD_OK;
}

int mhd_bunch_set_timing(mhd_bunch* b, int32_t enable) {
  if (!b) return MHD_ESTATE;
  CUDA_TRY(cudaStreamSynchronize(b->stream));
  drain_events(b, false);
  for (int c = 0; c < 16; ++c) { b->cls_ms[c] = 0.0; b->cls_n[c] = 0; }
  b->timing = enable != 0;
  return MHD_OK;
}

int mhd_bunch_kernel_times(mhd_bunch* b, int32_t cap, const char** names, double* ms, int64_t* count, int32_t* n) {
  if (!b || !n) return MHD_ESTATE;
  CUDA_TRY(cudaStreamSynchronize(b->stream));
  drain_events(b, true);
  int k = 0;
  for (int c = 0; c < KC_COUNT && k < cap; ++c) {
    if (b->cls_n[c] == 0) continue;
    if (names) names[k] = kclass_names[c];
    if (ms) ms[k] = b->cls_ms[c];
    if (count) count[k] = b->cls_n[c];
    ++k;
  }
  *n = k;
  return MHD_OK;
}

int mhd_bunch_destroy(mhd_bunch* b) {
  if (!b) return MHD_ESTATE;
  cudaStreamSynchronize(b->stream);
  drain_events(b, false);
  delete b->events;
  delete b;
  return MHD_OK;
}

}  // extern "C"
