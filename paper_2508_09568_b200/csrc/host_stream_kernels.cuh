// host_stream_kernels.cuh -- pack / unpack kernels of the host-streaming path (SURVEY 8f
// NEXT-1; PAPER.md L162-164 round-robin bunches, L243-247 asynchronous host<->device
// staging).  A host-resident bunch is kept in the COMPACT layout host[field][patch][k][j][i]
// (interior cells only); a chunk of patches crosses PCIe as eight contiguous copies into a
// staging buffer and is scattered into / gathered from the padded HBM layout by these
// kernels (pure data movement, HBM-bound, 16-byte accesses where the row length allows).
// A transfer may carry only the z-planes [k0, k0+nk) of its patches (a PIECE): the lowest or
// highest guard-width planes of a chunk are all its z-neighbours need from it, so they cross
// PCIe ahead of the rest (see hs_plan in mhd_bunch.cu).
#pragma once
#include "bunch_types.cuh"

namespace mhd {

// stage[f][pl][kk][j][i] (npl patches, nk planes)  <->  U[f][p0+pl][k0+kk+g][j+g][i+g]
template <typename T, int VEC, bool PACK>
__global__ void __launch_bounds__(256) k_pack_unpack(Geom G, T* __restrict__ U, T* __restrict__ stage, int p0, int npl, int k0, int nk) {
  const int nxv = G.n[0] / VEC;
  const long long rows = (long long)G.n[1] * nk;
  const long long per = rows * nxv;                       // vectors per (field, patch)
  const long long tot = per * npl * 8;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < tot; t += (long long)gridDim.x * blockDim.x) {
    const long long fp = t / per;
    const int r = (int)(t - fp * per);
    const int f = (int)(fp / npl), pl = (int)(fp - (long long)f * npl);
    const int row = r / nxv, iv = r - row * nxv;
    const int k = row / G.n[1], j = row - k * G.n[1];
    const long long u = (long long)f * G.fs + (long long)(p0 + pl) * G.ps + G.lead + (iv * VEC + G.g[0]) +
                        (long long)(j + G.g[1]) * G.pitch + (long long)(k0 + k + G.g[2]) * G.pitch * G.m[1];
    const long long s = (fp * rows + row) * G.n[0] + (long long)iv * VEC;
    if (VEC == 1) {
      if (PACK) stage[s] = U[u]; else U[u] = stage[s];
    } else {
      using V = typename std::conditional<sizeof(T) * VEC == 16, int4, int2>::type;
      if (PACK) *reinterpret_cast<V*>(stage + s) = *reinterpret_cast<const V*>(U + u);
      else *reinterpret_cast<V*>(U + u) = *reinterpret_cast<const V*>(stage + s);
    }
  }
}

}  // namespace mhd
