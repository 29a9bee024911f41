// mhd_bunch.cu -- C ABI (include/mhd_bunch.h) of the bunch MHD update: host orchestration.
//
// Path (section 2.1.4): guard fill -> primitives -> limited slopes ->
// predictor (edge EMF at time n, half-step face fields, primitive half step) -> HLLD at
// faces -> 2D Riemann problem at edges -> conservative + constrained-transport update;
// CFL reduction.  One launch of each kernel covers a whole sub-bunch of patches.
//
// This file never allocates device memory after create and has no CPU fallback.
#include "../../include/mhd_bunch.h"
#include "bunch_types.cuh"
#include "mhd_math.cuh"
#include "stage_kernels.cuh"
#include "fused_kernels.cuh"
#include "onepass_kernel.cuh"
#include "tile_kernel.cuh"
#include "host_stream_kernels.cuh"

#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <mutex>
#include <new>
#include <vector>
#include <algorithm>
#include <type_traits>

using namespace mhd;

namespace {
thread_local char g_cuda_err[256] = "";
}

// (x,y) tile of the fused kernel per arithmetic type.  fp32: 32 x 8, two CTAs per SM (2 x 38
// arrays of 36 x 10 cells each).  fp64: 16 x 16 with ONE CTA of 10 warps per SM -- a double
// takes two registers, so occupancy is register-bound either way, and the square tile does
// 5 % less halo work than 16 x 8 with two CTAs (riemann_update 7.81 -> 7.24 ms on the
// config-2 shape).
template <typename T> struct FusedTile;
template <> struct FusedTile<float> { static constexpr int TX = 32, TY = 8; };
#ifndef FUSED_F64_TY
#define FUSED_F64_TY 16
#endif
template <> struct FusedTile<double> { static constexpr int TX = 16, TY = FUSED_F64_TY; };
// one-pass kernel (onepass_kernel.cuh): tile and number of predictor warps
#ifndef ONEPASS_NPW
#define ONEPASS_NPW 7
#endif
struct OneTile { static constexpr int TX = 32, TY = 8, NPW = ONEPASS_NPW; };

// ------------------------------------------------------------------------ handle ----
struct mhd_bunch {
  mhd_bunch_desc desc;
  mhd_bunch_layout lay;
  Geom G;
  void* state[2];
  int cur;
  char* ws;
  size_t ws_bytes;
  int chunk;           // patches per sub-bunch of the fused path (D block)
  int chunk_s;         // patches per sub-bunch of the staged path
  // carved from the workspace head
  int* d_nbr;
  unsigned long long* d_rate;  // [npatch] per-patch CFL rate maxima (bit patterns) of the stand-alone pass
  unsigned long long* d_rate_next;  // [npatch] the same for the level a one-pass step is writing (its epilogue)
  bool rate_valid;             // d_rate_next holds the rates of the CURRENT level (set by a one-pass step that
                               // covered the bunch; cleared when the caller may have written the buffer)
  unsigned long long* d_bad;   // [1]
  double* d_dt;                // [2]: cfl result, step dt
  char* d_scratch;
  cudaStream_t stream;
  long long launches;
  size_t esz;
  // optional per-kernel-class timing (host-side objects only)
  int path;            // MHD_PATH_*: 0 = automatic choice
  int nsm;             // multiprocessors of the device
  bool onepass_ok;     // three active dimensions, fp32
  bool tile2d_ok;      // x and y active, z collapsed: the whole step in one kernel on shared-memory tiles
  bool gather_t_ok;    // ... which may read its halos through the neighbour table (consistent table, no -1 side)
  bool gather_ok;      // the one-pass kernel can read halos from the neighbours' interiors: every
                       // neighbour exists (no outflow side) and n_x is a whole number of 16-byte chunks
  bool gather2_ok;     // the two-kernel path can do the same (predictor loads through the neighbour table)
  bool guards_stale;   // fill_guards was deferred: the guard shell of the current level is not in HBM
  bool closing_ok;     // every closing face of the current level equals the neighbour's face 0: true after
                       // any fill and kept by steps (both sides evaluate the same update on the same
                       // data, bit for bit); false once the caller may have written the buffer
  bool fused_ok;       // three active dimensions and the tensor maps could be built
  int pred_ty;         // y-tile of the fused predictor (16, 8 or 4)
  DGeom DG;            // geometry of the D block
  char* d_dblock;
  CUtensorMap tmap_d;  // D block of the scratch: [38][chunk][mz][my][pitch]
  // host-streaming path (mhd_bunch_host_attach / mhd_bunch_step_host)
  struct HostStream {
    char* stage_up[2]; char* stage_dn[2];   // DEVICE staging, two chunk-sized buffers per direction (caller-owned)
    int chunk, nchunk;                      // patches per chunk, number of chunks
    // Library-owned streams: H2D copies alternate between two streams and so do D2H copies -- measured
    // on this box: while the other direction is busy, a copy that has to wait for the COMPLETION of the
    // previous copy of its stream starts ~40 us late (the completion signal queues behind the data);
    // two independent copies in flight keep the link busy.  Unpack and pack kernels have their own streams.
    cudaStream_t s_up[2], s_un, s_pk, s_dn[2];
    cudaEvent_t ev_begin, ev_all_steps;
    std::vector<cudaEvent_t> ev_copied, ev_up;            // per piece: staged / scattered into the state
    std::vector<cudaEvent_t> ev_step, ev_packed, ev_dn;   // per step unit: stepped / gathered / on the host
    std::vector<int> piece_chunk, piece_k0, piece_k1;     // upload pieces in order: planes [k0, k1) of a chunk
    std::vector<int> unit_chunk, unit_za, unit_zb;        // step units in order: planes [za, zb) of a chunk
    std::vector<int> ready;                 // ready[u]: piece after which unit u may step
  };
  HostStream* hs;
  // ring mode (mhd_bunch_ring_attach / mhd_bunch_step_ring): the handle's buffers are a window of
  // chunk slots through which a host-resident bunch LARGER than the buffers streams
  struct Ring {
    int NP, chunk, nchunk, nslot;                 // host bunch, patches per chunk, chunks, chunk slots of the window
    std::vector<int> up_chunk, up_slot, up_step, up_wait;   // planned uploads: chunk, slot, before which step, and the
                                                            // last step that read the slot's previous occupant (-1: none)
    std::vector<int> slot_of_step;                // slot in which chunk c sits when it is stepped
    std::vector<int> rows;                        // [NP][27] neighbour table in SLOT space (patch ids of the window)
    char* stage_up; char* stage_dn;
    cudaStream_t s_up, s_dn;
    std::vector<cudaEvent_t> ev_up, ev_step, ev_dn;   // per upload, per step, per slot
  };
  Ring* ring;
  std::vector<int>* h_nbr;   // HOST copy of the neighbour table (schedules of the host-streaming path)
  bool all_nbr;        // no -1 entry in the neighbour table
  // local time steps (mhd_bunch_local_begin / mhd_bunch_step_local): per-patch times and slots on the
  // host, small device tables carved from the workspace head
  struct Local {
    bool active;
    std::vector<double> t_old, t_new;
    std::vector<int> slot;                 // which state buffer holds the newer slice of a patch
  };
  Local* loc;
  int* d_slot;         // [npatch]
  int* d_plist;        // [npatch]
  double* d_dtlist;    // [npatch]
  double* d_wtab;      // [npatch][27]
  // overrides make_params applies while a list of patches is stepped
  const int* ov_plist; const double* ov_dtlist; int ov_side;
  bool nbr_consistent; // the table composes like translations (see table_is_consistent)
  int tune_zseg;       // MHD_TUNE_ONEPASS_ZSEG: 0 = automatic
  int tune_bands;      // MHD_TUNE_HOST_BANDS: 0 = automatic
  int tune_max_pitch;  // MHD_TUNE_HOST_MAX_PITCH: 0 = the device's limit (max_pitch)
  size_t max_pitch;    // cudaDevAttrMaxPitch of the handle's device: largest pitch a strided copy may name
  bool fused_cfl;      // MHD_TUNE_FUSED_CFL = 1: the one-pass step reduces the new level's CFL rates in its epilogue
  bool fused_cfl_auto; // MHD_TUNE_FUSED_CFL = 2 (default): it does so on small bunches (onepass_cfle)
  bool timing;
  struct Ev { int cls; cudaEvent_t a, b; };
  std::vector<Ev>* events;
  double cls_ms[16];
  long long cls_n[16];
};

enum KClass : int { KC_FILL = 0, KC_CFL, KC_PRIM, KC_EMF0, KC_PREDICT, KC_FLUX, KC_EMF, KC_UPDATE, KC_MISC, KC_RIEMANN, KC_ONEPASS,
                    KC_CLOSING, KC_TILE2D, KC_COUNT };
static const char* const kclass_names[KC_COUNT] = {"fill_guards", "cfl", "prim", "emf0", "predict", "hlld_flux",
                                                   "emf_2d", "update", "misc", "riemann_update", "step_onepass",
                                                   "sync_closing_faces", "step_tile2d"};

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
  if (d->flux_solver != 0 && d->flux_solver != 1) return MHD_EINVAL;
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
  G->flux_solver = d->flux_solver;
  return MHD_OK;
}

size_t head_bytes(int np) {
  return align_up(sizeof(int) * 27 * (size_t)np, 256) + 2 * align_up(sizeof(unsigned long long) * (size_t)np, 256) + 256 + 256 +
         2 * align_up(sizeof(int) * (size_t)np, 256) + align_up(sizeof(double) * (size_t)np, 256) +
         align_up(sizeof(double) * 27 * (size_t)np, 256);
}
DGeom make_dgeom(const Geom& G, size_t esz, int chunk) {
  DGeom D;
  const int ve = (int)(16 / esz);
  D.pitch = (G.n[0] + 2 + ve - 1) / ve * ve;
  D.ny = G.n[1] + 2;
  D.nz = G.n[2] + 2;
  D.ps = (long long)D.pitch * D.ny * D.nz;
  D.fs = D.ps * chunk;
  return D;
}
bool all_active(const Geom& G) { return G.act[0] && G.act[1] && G.act[2]; }
// A chunk smaller than the bunch is rounded down to a multiple of 74 patches: the fused
// kernels run 4 long-lived CTAs per 32^3 patch, so 74 patches fill 148 SMs x 2 CTAs exactly.
int wave_aligned_chunk(const Geom& G, int chunk) {
  if (chunk >= G.np || chunk < 74) return chunk;
  return chunk / 74 * 74;
}
size_t staged_bytes(const Geom& G, size_t esz, int chunk) { return align_up((size_t)W_COUNT * chunk * G.ps * esz, 256); }
size_t dblock_bytes(const Geom& G, size_t esz, int chunk) {
  return align_up((size_t)W_DCOUNT * make_dgeom(G, esz, chunk).fs * esz, 256);
}
// 3D bunches run the fused path: the D block scales with the chunk, the staged scratch (kept
// for cross-checks) only needs a few patches.  Otherwise the staged scratch is all there is.
int staged_patches_3d(const Geom& G) { return G.np < 16 ? G.np : 16; }

template <typename T>
Params<T> make_params(const mhd_bunch* b, int p0, int npl) {
  Params<T> P;
  P.G = b->G;
  P.U = (const T*)b->state[b->cur] ;
  P.Un = (T*)b->state[1 - b->cur];
  P.W = (T*)b->d_scratch;
  P.wfs = (long long)b->chunk_s * b->G.ps;
  P.DG = b->DG;
  P.D = (T*)b->d_dblock;
  P.p0 = p0;
  P.npl = npl;
  P.plist = nullptr;
  P.dtlist = nullptr;
  if (b->ov_plist) {   // a list of patches with their own time steps (local time stepping)
    P.plist = b->ov_plist + p0;
    P.dtlist = b->ov_dtlist + p0;
    P.U = (const T*)b->state[b->ov_side];
    P.Un = (T*)b->state[1 - b->ov_side];
  }
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
  const int vec = (int)(16 / sizeof(T));
  // every neighbour present and rows made of whole 16-byte chunks: the chunked fill (aligned 16-byte
  // accesses, x-guards included); otherwise cell by cell (zero-gradient sides, ragged rows)
  const bool chunked = b->all_nbr && G.act[0] && G.n[0] % vec == 0 && (G.lead + G.g[0]) % vec == 0 && G.pitch % vec == 0 &&
                       G.ps % vec == 0 && G.fs % vec == 0 && ((uintptr_t)b->state[b->cur] & 15) == 0;
  if (chunked) {
    const int cpr = G.pitch / vec, lg = (G.lead + G.g[0]) / vec, ni = G.n[0] / vec;
    const long long per = (long long)(G.m[1] * G.m[2] - G.n[1] * G.n[2]) * cpr + (long long)G.n[1] * G.n[2] * (cpr - ni);
    (void)lg;
    if (per > 0) {
      LaunchScope ls(b, KC_FILL);
      k_fill_guards_vec<T><<<dim3(blocks_for(per * G.np, 256), 8 / FillFpt<T>::N), 256, 0, b->stream>>>(G, (T*)b->state[b->cur], b->d_nbr);
    }
    CUDA_TRY(cudaGetLastError());
    return MHD_OK;
  }
  const FillMap M = make_fill_map(G);
  const long long tot = (long long)M.start[6] * G.np;
  if (tot > 0) {
    LaunchScope ls(b, KC_FILL);
    k_fill_guards<T><<<blocks_for(tot, 256), 256, 0, b->stream>>>(G, M, (T*)b->state[b->cur], b->d_nbr);
  }
  CUDA_TRY(cudaGetLastError());
  return MHD_OK;
}

// closing faces only (the part of the fill that cfl_dt and the one-pass kernel's update read)
template <typename T>
int launch_sync_closing(mhd_bunch* b, int p0 = 0, int npl = -1, int zlo = 0, int zhi = -1) {
  const Geom& G = b->G;
  if (npl < 0) npl = G.np;
  if (zhi < 0) zhi = G.n[2];
  const long long per = (long long)G.n[1] * G.n[2] + (long long)G.n[0] * G.n[2] + (long long)G.n[0] * G.n[1];
  const long long tot = per * npl;
  {
    LaunchScope ls(b, KC_CLOSING);
    k_sync_closing_faces<T><<<blocks_for(tot, 256), 256, 0, b->stream>>>(G, (T*)b->state[b->cur], b->d_nbr, p0, npl, zlo, zhi);
  }
  CUDA_TRY(cudaGetLastError());
  return MHD_OK;
}

// runs a deferred guard fill now (before anything reads the guard shell from HBM)
int materialise_guards(mhd_bunch* b) {
  if (!b->guards_stale) return MHD_OK;
  b->guards_stale = false;
  b->closing_ok = true;
  return b->desc.dtype == MHD_F64 ? launch_fill<double>(b) : launch_fill<float>(b);
}

template <typename T>
int launch_cfl(mhd_bunch* b, double courant, void* dt_dev, void* dt_patch) {
  const Geom& G = b->G;
  Params<T> P = make_params<T>(b, 0, G.np);
  if (b->rate_valid) {
    // the one-pass step that produced this level reduced the rates in its epilogue (same function,
    // same bits as k_cfl): only the bunch-wide reduction is left
    LaunchScope ls(b, KC_MISC);
    k_cfl_final<<<1, 256, 0, b->stream>>>(b->d_rate_next, G.np, courant, b->d_dt, (double*)dt_dev, (double*)dt_patch);
    CUDA_TRY(cudaGetLastError());
    return MHD_OK;
  }
  { LaunchScope ls(b, KC_MISC); k_zero_u64<<<blocks_for(G.np, 256), 256, 0, b->stream>>>(b->d_rate, G.np); }
  const long long per = (long long)G.n[0] * G.n[1] * G.n[2];
#ifndef CFL_CPT
#define CFL_CPT 8
#endif
  int bx = (int)((per + 256 * CFL_CPT - 1) / (256 * CFL_CPT));
  if (bx < 1) bx = 1;
  dim3 grid((unsigned)bx, (unsigned)G.np);
  { LaunchScope ls(b, KC_CFL); k_cfl<T><<<grid, 256, 0, b->stream>>>(P, b->d_rate); }
  { LaunchScope ls(b, KC_MISC);
    k_cfl_final<<<1, 256, 0, b->stream>>>(b->d_rate, G.np, courant, b->d_dt, (double*)dt_dev, (double*)dt_patch); }
  CUDA_TRY(cudaGetLastError());
  return MHD_OK;
}

// which implementation of the step runs: MHD_PATH_ONEPASS, MHD_PATH_TWO_KERNEL or MHD_PATH_STAGED
int effective_path(const mhd_bunch* b) {
  if (b->path == MHD_PATH_STAGED) return MHD_PATH_STAGED;
  if (b->tile2d_ok && (b->path == MHD_PATH_AUTO || b->path == MHD_PATH_TILE2D)) return MHD_PATH_TILE2D;
  if (b->path == MHD_PATH_TWO_KERNEL) return b->fused_ok ? MHD_PATH_TWO_KERNEL : MHD_PATH_STAGED;
  if (b->onepass_ok) return MHD_PATH_ONEPASS;           // automatic, or asked for
  return b->fused_ok ? MHD_PATH_TWO_KERNEL : MHD_PATH_STAGED;
}

// true if the step that would run gathers its halos from the neighbours' interiors, so that the
// guard shell need not exist in HBM (deferred fill)
bool step_gathers(const mhd_bunch* b) {
  const int path = effective_path(b);
  return (path == MHD_PATH_ONEPASS && b->gather_ok) || (path == MHD_PATH_TWO_KERNEL && b->gather2_ok) ||
         (path == MHD_PATH_TILE2D && b->gather_t_ok);
}

// Does the one-pass step reduce the CFL rates of the level it writes in its epilogue?  Asked for
// (MHD_TUNE_FUSED_CFL = 1), or by itself on bunches of at most ONEPASS_CFLE_WAVES waves of tiles: those are bound
// by launch latency, and the epilogue replaces two of the five launches of a step (the rate
// pass and its clear).  Measured (profiles/r3_c4_sweep.md): one 32^3 patch 59 -> 51 us per step, 8 x 32^3 86 -> 79,
// 64 x 16^3 91 -> 85; break-even at one to two waves (64 x 32^3: 465 either way; 64 x 24^3, 1.3 waves: 282 -> 292);
// on bunches that fill the GPU the stand-alone pass is cheaper (config 2: 3.03 against 3.15 ms per step).  The
// choice is made for the WHOLE bunch, so every launch of a step (chunks, bands, patch lists) runs the same variant.
#ifndef ONEPASS_CFLE_WAVES
#define ONEPASS_CFLE_WAVES 1
#endif
bool onepass_cfle(const mhd_bunch* b) {
  if (b->fused_cfl) return true;
  if (!b->fused_cfl_auto) return false;
  const int tx = b->G.n[0] <= 16 ? 16 : OneTile::TX, ty = b->G.n[0] <= 16 ? 16 : OneTile::TY;
  const long long tiles = (long long)((b->G.n[0] + tx - 1) / tx) * ((b->G.n[1] + ty - 1) / ty) * b->G.np;
  return tiles <= (long long)ONEPASS_CFLE_WAVES * b->nsm;
}

template <typename T> struct OnePassLaunch {
  static int prepare(mhd_bunch*) { return MHD_OK; }
  static int run(mhd_bunch*, const double*, int = 0, int = -1, bool = true, int = 0, int = -1) { return MHD_EINVAL; }
};
template <> struct OnePassLaunch<float> {
  // one tile shape: patches [p0, p0+npl) of the bunch
  template <int TX, int TY>
  static int launch(mhd_bunch* b, const double* dtp, int p0, int npl, bool attr_only = false, int zlo = 0, int zhi = -1) {
    using Cfg = OneCfg<float, TX, TY, OneTile::NPW>;
    const Geom& G = b->G;
    if (attr_only) {   // called once from create, on the handle's device (the attribute is per device)
      CUDA_TRY(cudaFuncSetAttribute(k_step_onepass<float, TX, TY, OneTile::NPW, 1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::smem));
      CUDA_TRY(cudaFuncSetAttribute(k_step_onepass<float, TX, TY, OneTile::NPW, 2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::smem));
      CUDA_TRY(cudaFuncSetAttribute(k_step_onepass<float, TX, TY, OneTile::NPW, 1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::smem));
      CUDA_TRY(cudaFuncSetAttribute(k_step_onepass<float, TX, TY, OneTile::NPW, 2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::smem));
      CUDA_TRY(cudaFuncSetAttribute(k_step_onepass<float, TX, TY, OneTile::NPW, 1, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::smem));
      return MHD_OK;
    }
    // the limiter and the CFL epilogue are compile-time parameters of the kernel
    const bool cfle = onepass_cfle(b);
    auto kern = cfle
                    ? (G.limiter == 1 ? k_step_onepass<float, TX, TY, OneTile::NPW, 1, true> : k_step_onepass<float, TX, TY, OneTile::NPW, 2, true>)
                    : (G.limiter == 1 ? k_step_onepass<float, TX, TY, OneTile::NPW, 1, false> : k_step_onepass<float, TX, TY, OneTile::NPW, 2, false>);
    // the default scheme (minmod, HLLD, HLLD-2D) has an instantiation with the solvers fixed at compile time
    if (!cfle && G.limiter == 1 && G.emf_solver == 0 && G.flux_solver == 0)
      kern = k_step_onepass<float, TX, TY, OneTile::NPW, 1, false, true>;
    Params<float> P = make_params<float>(b, p0, npl);
    if (zhi < 0) zhi = G.n[2];
    const int xt = (G.n[0] + TX - 1) / TX, yt = (G.n[1] + TY - 1) / TY;
    // Small launches (fewer than four waves of tiles): the columns are cut into z segments, each a CTA that
    // pays a five-plane run-in.  The cut minimises waves x (planes per segment + 5), segments of at least four
    // planes -- a launch that leaves SMs idle is bound by the latency of one CTA's march (one 32^3 patch:
    // 78 -> 56 us per step with 4-plane segments), a launch that already fills them only loses to the run-in.
    int zseg = 1;
    const long long tiles = (long long)xt * yt * npl;
    if (tiles < 4ll * b->nsm) {
      const int nzr = zhi - zlo;
      long long best = -1;
      for (int z = 1; z <= (nzr / 4 > 1 ? nzr / 4 : 1); ++z) {
        const long long waves = (tiles * z + b->nsm - 1) / b->nsm;
        const long long cost = waves * ((nzr + z - 1) / z + 5);
        if (best < 0 || cost < best) { best = cost; zseg = z; }
      }
    }
    if (b->tune_zseg >= 1) zseg = b->tune_zseg < zhi - zlo ? b->tune_zseg : zhi - zlo;   // mhd_bunch_set_tuning
    {  // no empty segments: the kernel cuts [zlo, zhi) into pieces of ceil(planes / zseg), so e.g. 32 planes in
       // 31 segments would be 16 pieces of two planes and 15 CTAs that start past zhi; ask for the 16
      const int nzr = zhi - zlo, zlen = (nzr + zseg - 1) / zseg;
      zseg = (nzr + zlen - 1) / zlen;
    }
    dim3 grid((unsigned)(xt * yt), (unsigned)npl, (unsigned)zseg);
    {
      LaunchScope ls(b, KC_ONEPASS);
      kern<<<grid, Cfg::NTH, Cfg::smem, b->stream>>>(P, b->d_nbr, (b->gather_ok && !b->ov_plist) ? 1 : 0, dtp, b->d_bad, b->d_rate_next, xt, zseg, zlo, zhi);
    }
    CUDA_TRY(cudaGetLastError());
    return MHD_OK;
  }
  // patches [p0, p0+npl) of the bunch (npl < 0: all); `last` flips the buffers.  Rows of up to
  // 16 cells take the 16 x 16 tile (a 32-wide tile would leave half of every warp idle).
  static int prepare(mhd_bunch* b) {
    return b->G.n[0] <= 16 ? launch<16, 16>(b, nullptr, 0, 0, true) : launch<OneTile::TX, OneTile::TY>(b, nullptr, 0, 0, true);
  }
  static int run(mhd_bunch* b, const double* dtp, int p0 = 0, int npl = -1, bool last = true, int zlo = 0, int zhi = -1) {
    if (npl < 0) npl = b->G.np;
    const int rc = b->G.n[0] <= 16 ? launch<16, 16>(b, dtp, p0, npl, false, zlo, zhi)
                                   : launch<OneTile::TX, OneTile::TY>(b, dtp, p0, npl, false, zlo, zhi);
    if (rc != MHD_OK) return rc;
    if (last) {
      b->cur = 1 - b->cur;
      b->guards_stale = false;   // the new level's guards are undefined until the next fill_guards
      b->rate_valid = onepass_cfle(b);   // every patch went through the epilogue since the last k_set_dt
    }
    return MHD_OK;
  }
};

// 2D bunches: one kernel, every stage on a shared-memory tile (tile_kernel.cuh).  fp32 32 x 16 tiles,
// fp64 32 x 8 (the tile with its halo and 50 arrays has to fit in 227 KB).
template <typename T> struct Tile2D { static constexpr int TX = 32, TY = sizeof(T) == 4 ? 16 : 8; };
// fp32: persistent CTAs with two raw buffers (the next tile is prefetched); fp64: one tile per CTA (a second raw
// buffer does not fit beside the 42 scratch arrays of a 32 x 8 tile)
template <typename T> struct Tile2DBuf { static constexpr int N = sizeof(T) == 4 ? 2 : 1; };
template <typename T>
int prepare_tile2d() {
  constexpr int TX = Tile2D<T>::TX, TY = Tile2D<T>::TY, NB = Tile2DBuf<T>::N;
  using C1 = TileCfg<T, TX, TY, 1>;
  using C2 = TileCfg<T, TX, TY, NB>;
  CUDA_TRY(cudaFuncSetAttribute(k_step_tile2d<T, TX, TY, false, 1, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C1::smem));
  CUDA_TRY(cudaFuncSetAttribute(k_step_tile2d<T, TX, TY, true, 1, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C1::smem));
  CUDA_TRY(cudaFuncSetAttribute(k_step_tile2d<T, TX, TY, false, NB, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C2::smem));
  CUDA_TRY(cudaFuncSetAttribute(k_step_tile2d<T, TX, TY, false, 1, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C1::smem));
  CUDA_TRY(cudaFuncSetAttribute(k_step_tile2d<T, TX, TY, true, 1, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C1::smem));
  CUDA_TRY(cudaFuncSetAttribute(k_step_tile2d<T, TX, TY, false, NB, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C2::smem));
  CUDA_TRY(cudaFuncSetAttribute(k_step_tile2d<T, TX, TY, false, 1, -1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C1::smem));
  CUDA_TRY(cudaFuncSetAttribute(k_step_tile2d<T, TX, TY, true, 1, -1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C1::smem));
  CUDA_TRY(cudaFuncSetAttribute(k_step_tile2d<T, TX, TY, false, NB, -1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C2::smem));
  return MHD_OK;
}
// Small 2D bunches are bound by launch latency: there the tile kernel's CFL epilogue replaces two launches
// of the next cfl_dt (config 1: 31 -> 24 us per step in fp32).  On bunches of many waves the stand-alone
// pass is as cheap (fp64 2048^2: 2.08 against 2.14 ms per step), so the epilogue is used up to 8 waves.
template <typename T> long long tile2d_tiles(const mhd_bunch* b, int npl) {
  return (long long)((b->G.n[0] + Tile2D<T>::TX - 1) / Tile2D<T>::TX) * ((b->G.n[1] + Tile2D<T>::TY - 1) / Tile2D<T>::TY) * npl;
}
template <typename T> bool tile2d_wants_cfl(const mhd_bunch* b) { return tile2d_tiles<T>(b, b->G.np) <= 8ll * b->nsm; }
// cfle: the kernel also reduces the CFL rates of the level it writes into d_rate_next (cleared by k_set_dt)
template <typename T>
int launch_tile2d(mhd_bunch* b, int p0, int npl, bool cfle = false) {
  constexpr int TX = Tile2D<T>::TX, TY = Tile2D<T>::TY, NB = Tile2DBuf<T>::N;
  const Geom& G = b->G;
  Params<T> P = make_params<T>(b, p0, npl);
  const int xt = (G.n[0] + TX - 1) / TX, yt = (G.n[1] + TY - 1) / TY;
  const long long tiles = tile2d_tiles<T>(b, npl);
  const int gather = (b->gather_t_ok && !b->ov_plist) ? 1 : 0;
  if (!G.act[1]) {     // one-dimensional bunch along x: one small CTA per patch
    const size_t smem = (size_t)75 * (G.n[0] + 6) * sizeof(T);
    const int lim = G.limiter == 1 ? ((G.emf_solver == 0 && G.flux_solver == 0) ? -1 : 1) : 2;
    LaunchScope ls(b, KC_TILE2D);
    auto go1 = [&](auto kern) {
      if (smem > 48 * 1024) cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      kern<<<(unsigned)npl, 128, smem, b->stream>>>(P, b->d_nbr, gather, b->d_dt + 1, b->d_bad, b->d_rate_next);
    };
    if (cfle) { if (lim < 0) go1(k_step_line1d<T, true, -1>); else if (lim == 1) go1(k_step_line1d<T, true, 1>); else go1(k_step_line1d<T, true, 2>); }
    else { if (lim < 0) go1(k_step_line1d<T, false, -1>); else if (lim == 1) go1(k_step_line1d<T, false, 1>); else go1(k_step_line1d<T, false, 2>); }
    CUDA_TRY(cudaGetLastError());
    return MHD_OK;
  }
  // more than two waves of tiles: persistent CTAs that prefetch (where a second raw buffer fits)
  const bool persist = NB == 2 && !cfle && tiles > 2ll * b->nsm;
  {
    LaunchScope ls(b, KC_TILE2D);
    // the limiter is a compile-time parameter of the kernel
    auto go = [&](auto kern, unsigned grid, int nth, size_t smem) {
      kern<<<grid, nth, smem, b->stream>>>(P, b->d_nbr, gather, b->d_dt + 1, b->d_bad, b->d_rate_next, xt, yt);
    };
    // limiter: a compile-time parameter (1 minmod, 2 monotonised central); -1 = the default scheme, minmod with the
    // default solvers (HLLD, HLLD-2D) fixed at compile time as well
    const int lim = G.limiter == 1 ? ((G.emf_solver == 0 && G.flux_solver == 0) ? -1 : 1) : 2;
    if (persist) {
      using C = TileCfg<T, TX, TY, NB>;
      if (lim < 0) go(k_step_tile2d<T, TX, TY, false, NB, -1>, (unsigned)b->nsm, C::NTH, C::smem);
      else if (lim == 1) go(k_step_tile2d<T, TX, TY, false, NB, 1>, (unsigned)b->nsm, C::NTH, C::smem);
      else go(k_step_tile2d<T, TX, TY, false, NB, 2>, (unsigned)b->nsm, C::NTH, C::smem);
    } else if (cfle) {
      using C = TileCfg<T, TX, TY, 1>;
      if (lim < 0) go(k_step_tile2d<T, TX, TY, true, 1, -1>, (unsigned)tiles, C::NTH, C::smem);
      else if (lim == 1) go(k_step_tile2d<T, TX, TY, true, 1, 1>, (unsigned)tiles, C::NTH, C::smem);
      else go(k_step_tile2d<T, TX, TY, true, 1, 2>, (unsigned)tiles, C::NTH, C::smem);
    } else {
      using C = TileCfg<T, TX, TY, 1>;
      if (lim < 0) go(k_step_tile2d<T, TX, TY, false, 1, -1>, (unsigned)tiles, C::NTH, C::smem);
      else if (lim == 1) go(k_step_tile2d<T, TX, TY, false, 1, 1>, (unsigned)tiles, C::NTH, C::smem);
      else go(k_step_tile2d<T, TX, TY, false, 1, 2>, (unsigned)tiles, C::NTH, C::smem);
    }
  }
  CUDA_TRY(cudaGetLastError());
  return MHD_OK;
}

// dynamic shared memory opt-in of the fused kernels: per device, so done once per handle in create
template <typename T>
int prepare_fused() {
  CUDA_TRY(cudaFuncSetAttribute(k_riemann_update<T, FusedTile<T>::TX, FusedTile<T>::TY>,
                                cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)FusedCfg<T, FusedTile<T>::TX, FusedTile<T>::TY>::smem));
  CUDA_TRY(cudaFuncSetAttribute(k_predict_fused<T, 16>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
  CUDA_TRY(cudaFuncSetAttribute(k_predict_fused<T, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
  CUDA_TRY(cudaFuncSetAttribute(k_predict_fused<T, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
  return MHD_OK;
}

// The deferred fill trusts that a patch's evolved closing face equals its neighbour's face 0 bit
// for bit, and the gathered halos that what a patch sees across a side is what its neighbour
// sees of itself.  Both hold when the table composes like translations: nbr[p][0] = p and
// nbr[nbr[p][c1]][c2] = nbr[p][c1+c2] whenever c1+c2 is again one of the 27 classes.  Tables
// with -1 entries never take those routes.
bool table_is_consistent(const int32_t* nb, int np) {
  for (int p = 0; p < np; ++p) {
    const int32_t* tp = nb + (size_t)p * 27;
    if (tp[13] != p) return false;
    for (int c1 = 0; c1 < 27; ++c1) {
      const int q = tp[c1];
      if (q < 0) return false;
      const int a[3] = {c1 % 3 - 1, (c1 / 3) % 3 - 1, c1 / 9 - 1};
      for (int c2 = 0; c2 < 27; ++c2) {
        const int e[3] = {a[0] + c2 % 3 - 1, a[1] + (c2 / 3) % 3 - 1, a[2] + c2 / 9 - 1};
        if (e[0] < -1 || e[0] > 1 || e[1] < -1 || e[1] > 1 || e[2] < -1 || e[2] > 1) continue;
        if (nb[(size_t)q * 27 + c2] != tp[(e[2] + 1) * 9 + (e[1] + 1) * 3 + (e[0] + 1)]) return false;
      }
    }
  }
  return true;
}

// the global-step entry points are closed while the handle is in local-time-step mode (the two
// buffers are then time slices per patch, not levels n and n+1 of the whole bunch)
#define NOT_LOCAL(b)                                               \
  do {                                                             \
    if ((b)->loc && (b)->loc->active) return MHD_ESTATE;           \
  } while (0)

// ... and while a ring is attached: the device copy of the neighbour table then holds rows of the BIG
// host bunch in slot numbers (mhd_bunch_step_ring rewrites them chunk by chunk), which the resident,
// host-streaming and local-time-step calls would silently take for the window's own table
#define NOT_RING(b)                                                \
  do {                                                             \
    if ((b)->ring) return MHD_ESTATE;                              \
  } while (0)

// every launching entry point runs on the handle's device, whatever the caller's current one is
#define ENTER(b)                                                   \
  do {                                                             \
    if (!(b)) return MHD_ESTATE;                                   \
    cudaError_t e_ = cudaSetDevice((b)->desc.device);              \
    if (e_ != cudaSuccess) return fail_cuda(e_, "cudaSetDevice");  \
  } while (0)

// two-kernel path on patches [q0, q0+nq): sub-bunches of at most b->chunk patches (D block)
template <typename T>
int launch_fused_range(mhd_bunch* b, int q0, int nq) {
  const Geom& G = b->G;
  const double* dtp = b->d_dt + 1;
  const int gather = (b->gather2_ok && b->guards_stale) ? 1 : 0;   // shell not in HBM: read through the table
  cudaStream_t st = b->stream;
  for (int p0 = q0; p0 < q0 + nq; p0 += b->chunk) {
    const int npl = (q0 + nq - p0 < b->chunk) ? q0 + nq - p0 : b->chunk;
    Params<T> P = make_params<T>(b, p0, npl);
    const int ty = b->pred_ty;
    const int pa = (G.n[0] + 5) * (ty + 5);
    const size_t sm = (size_t)39 * pa * sizeof(T);
    dim3 grid((unsigned)((G.n[1] + ty - 1) / ty), (unsigned)npl);
    const unsigned nth = (unsigned)((pa + 31) / 32 * 32);
    {
      LaunchScope ls(b, KC_PREDICT);
      if (ty == 16) k_predict_fused<T, 16><<<grid, nth, sm, st>>>(P, dtp, b->d_bad, b->d_nbr, gather);
      else if (ty == 8) k_predict_fused<T, 8><<<grid, nth, sm, st>>>(P, dtp, b->d_bad, b->d_nbr, gather);
      else k_predict_fused<T, 4><<<grid, nth, sm, st>>>(P, dtp, b->d_bad, b->d_nbr, gather);
    }
    using Cfg = FusedCfg<T, FusedTile<T>::TX, FusedTile<T>::TY>;
    const int xt = (G.n[0] + FusedTile<T>::TX - 1) / FusedTile<T>::TX, yt = (G.n[1] + FusedTile<T>::TY - 1) / FusedTile<T>::TY;
    dim3 grid2((unsigned)(xt * yt), (unsigned)npl);
    LaunchScope ls(b, KC_RIEMANN);
    k_riemann_update<T, FusedTile<T>::TX, FusedTile<T>::TY><<<grid2, Cfg::NTH, Cfg::smem, st>>>(P, b->tmap_d, dtp, xt);
  }
  CUDA_TRY(cudaGetLastError());
  return MHD_OK;
}

// staged path on patches [q0, q0+nq) (or on that many entries of a patch list): one kernel per stage
template <typename T>
int launch_staged_range(mhd_bunch* b, int q0, int nq) {
  const Geom& G = b->G;
  const double* dtp = b->d_dt + 1;
  const int ch = b->chunk_s;
  for (int p0 = q0; p0 < q0 + nq; p0 += ch) {
    const int npl = (q0 + nq - p0 < ch) ? q0 + nq - p0 : ch;
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
  return MHD_OK;
}

template <typename T>
int launch_step(mhd_bunch* b) {
  const Geom& G = b->G;
  const double* dtp = b->d_dt + 1;
  const int path = effective_path(b);
  b->rate_valid = false;     // set again below if the one-pass kernel (whose epilogue reduces the CFL rates) runs
  if (path == MHD_PATH_ONEPASS && b->gather_ok) return OnePassLaunch<T>::run(b, dtp);
  if (path == MHD_PATH_TWO_KERNEL && b->gather2_ok) {
    // halos come through the neighbour table if the fill was deferred, from the shell otherwise
    const int rc = launch_fused_range<T>(b, 0, G.np);
    if (rc != MHD_OK) return rc;
    b->cur = 1 - b->cur;
    b->guards_stale = false;
    return MHD_OK;
  }
  if (path == MHD_PATH_TILE2D && b->gather_t_ok) {
    const bool cfle = tile2d_wants_cfl<T>(b);
    const int rc = launch_tile2d<T>(b, 0, G.np, cfle);
    if (rc != MHD_OK) return rc;
    b->cur = 1 - b->cur;
    b->guards_stale = false;
    b->rate_valid = cfle;      // every patch went through the tile kernel's CFL epilogue since the last k_set_dt
    return MHD_OK;
  }
  {  // every other route reads the guard shell from HBM
    const int rc = materialise_guards(b);
    if (rc != MHD_OK) return rc;
  }
  if (path == MHD_PATH_ONEPASS) return OnePassLaunch<T>::run(b, dtp);
  if (path == MHD_PATH_TWO_KERNEL) {
    const int rc = launch_fused_range<T>(b, 0, G.np);
    if (rc != MHD_OK) return rc;
    b->cur = 1 - b->cur;
    return MHD_OK;
  }
  {
    const bool cfle = path == MHD_PATH_TILE2D && tile2d_wants_cfl<T>(b);
    const int rc = path == MHD_PATH_TILE2D ? launch_tile2d<T>(b, 0, G.np, cfle) : launch_staged_range<T>(b, 0, G.np);
    if (rc != MHD_OK) return rc;
    b->rate_valid = cfle;
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
  // the whole bunch in one chunk unless that needs more than 48 GiB of scratch
  const size_t cap = (size_t)48 << 30;
  int chunk = G.np;
  if (all_active(G)) {
    lay->workspace_min = head_bytes(G.np) + staged_bytes(G, esz, 1) + dblock_bytes(G, esz, 1);
    while (chunk > 1 && dblock_bytes(G, esz, chunk) > cap) chunk = (chunk + 1) / 2;
    chunk = wave_aligned_chunk(G, chunk);
    lay->workspace_best = head_bytes(G.np) + staged_bytes(G, esz, staged_patches_3d(G)) + dblock_bytes(G, esz, chunk);
  } else {
    lay->workspace_min = head_bytes(G.np) + staged_bytes(G, esz, 1);
    while (chunk > 1 && staged_bytes(G, esz, chunk) > cap) chunk = (chunk + 1) / 2;
    lay->workspace_best = head_bytes(G.np) + staged_bytes(G, esz, chunk);
  }
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
  b->d_rate_next = (unsigned long long*)p; p += align_up(sizeof(unsigned long long) * (size_t)desc->npatch, 256);
  b->rate_valid = false;
  b->d_bad = (unsigned long long*)p;  p += 256;
  b->d_dt = (double*)p;               p += 256;
  b->d_slot = (int*)p;                p += align_up(sizeof(int) * (size_t)desc->npatch, 256);
  b->d_plist = (int*)p;               p += align_up(sizeof(int) * (size_t)desc->npatch, 256);
  b->d_dtlist = (double*)p;           p += align_up(sizeof(double) * (size_t)desc->npatch, 256);
  b->d_wtab = (double*)p;             p += align_up(sizeof(double) * 27 * (size_t)desc->npatch, 256);
  b->loc = nullptr;
  b->ov_plist = nullptr; b->ov_dtlist = nullptr; b->ov_side = 0;
  b->d_scratch = p;
  const size_t avail = workspace_bytes - (size_t)(p - b->ws);
  {
    const bool d3 = all_active(b->G);
    // staged scratch first (a few patches in 3D, everything that fits otherwise), D block after it
    int cs = d3 ? staged_patches_3d(b->G) : desc->npatch;
    while (cs > 1 && staged_bytes(b->G, b->esz, cs) + (d3 ? dblock_bytes(b->G, b->esz, 1) : 0) > avail) --cs;
    b->chunk_s = cs;
    b->chunk = cs;
    if (d3) {
      const size_t left = avail - staged_bytes(b->G, b->esz, cs);
      long long c = (long long)(left / dblock_bytes(b->G, b->esz, 1));
      if (c > desc->npatch) c = desc->npatch;
      if (c < 1) { delete b->events; delete b; return MHD_ENOMEM; }
      while (c < desc->npatch && dblock_bytes(b->G, b->esz, (int)c + 1) <= left) ++c;
      b->chunk = wave_aligned_chunk(b->G, (int)c);
    }
  }
  b->fused_ok = false;
  if (b->G.act[0] && b->G.act[1] && b->G.act[2]) {
    const bool f64 = desc->dtype == MHD_F64;
    b->DG = make_dgeom(b->G, b->esz, b->chunk);
    b->pred_ty = 0;
    for (int ty : {16, 8, 4}) {
      const size_t pa = (size_t)(b->G.n[0] + 5) * (ty + 5);
      if (pa <= (size_t)predict_max_threads(ty) && 39 * pa * b->esz <= (size_t)220 * 1024) { b->pred_ty = ty; break; }
    }
    b->d_dblock = b->d_scratch + staged_bytes(b->G, b->esz, b->chunk_s);
    const int bx = f64 ? FusedCfg<double, FusedTile<double>::TX, FusedTile<double>::TY>::DW
                       : FusedCfg<float, FusedTile<float>::TX, FusedTile<float>::TY>::DW;
    const int by = f64 ? FusedCfg<double, FusedTile<double>::TX, FusedTile<double>::TY>::DH
                       : FusedCfg<float, FusedTile<float>::TX, FusedTile<float>::TY>::DH;
    b->fused_ok = b->pred_ty != 0 && make_bunch_tensor_map(&b->tmap_d, b->d_dblock, f64, b->DG.pitch, b->DG.ny, b->DG.nz, b->chunk, W_DCOUNT,
                                        b->DG.ps, b->DG.fs, bx, by, W_DCOUNT);
  }
  b->onepass_ok = all_active(b->G) && desc->dtype == MHD_F32;
  // x and y active with z collapsed (tile kernel), or x alone (line kernel: the whole row of a patch in shared memory)
  b->tile2d_ok = b->G.act[0] && !b->G.act[2] && (b->G.act[1] || (size_t)75 * (b->G.n[0] + 6) * b->esz <= (size_t)200 * 1024);
  b->nsm = 148;
  cudaDeviceGetAttribute(&b->nsm, cudaDevAttrMultiProcessorCount, desc->device);
  b->gather_ok = b->onepass_ok && b->G.n[0] % (int)(16 / b->esz) == 0;
  b->all_nbr = true;
  for (long long c = 0; c < 27ll * desc->npatch && b->all_nbr; ++c)
    if (nbr[c] < 0) b->all_nbr = false;
  b->nbr_consistent = b->all_nbr && table_is_consistent(nbr, desc->npatch);
  b->gather_ok = b->gather_ok && b->nbr_consistent;
  b->gather2_ok = b->fused_ok && b->nbr_consistent;
  b->gather_t_ok = b->tile2d_ok && b->nbr_consistent;
  b->tune_zseg = 0;
  b->tune_bands = 0;
  b->tune_max_pitch = 0;
  {
    int mp = 0;
    b->max_pitch = (cudaDeviceGetAttribute(&mp, cudaDevAttrMaxPitch, desc->device) == cudaSuccess && mp > 0) ? (size_t)mp
                                                                                                             : (size_t)0x7fffffff;
  }
  b->fused_cfl = false;
  b->fused_cfl_auto = true;
  b->hs = nullptr;
  b->ring = nullptr;
  b->h_nbr = new (std::nothrow) std::vector<int>(nbr, nbr + 27 * (size_t)desc->npatch);
  if (!b->h_nbr) { delete b->events; delete b; return MHD_ENOMEM; }
  b->guards_stale = false;
  b->closing_ok = false;
  cudaError_t e = cudaMemcpyAsync(b->d_nbr, nbr, sizeof(int) * 27 * (size_t)desc->npatch, cudaMemcpyHostToDevice, b->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(b->d_bad, 0, 512, b->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(b->stream);
  if (e != cudaSuccess) { delete b->h_nbr; delete b->events; delete b; return fail_cuda(e, "create: table upload"); }
  {  // dynamic shared memory opt-ins of the kernels this handle can launch, on ITS device
    int ra = MHD_OK;
    if (b->fused_ok) ra = desc->dtype == MHD_F64 ? prepare_fused<double>() : prepare_fused<float>();
    if (ra == MHD_OK && b->onepass_ok) ra = OnePassLaunch<float>::prepare(b);
    if (ra == MHD_OK && b->tile2d_ok) ra = desc->dtype == MHD_F64 ? prepare_tile2d<double>() : prepare_tile2d<float>();
    if (ra != MHD_OK) { delete b->h_nbr; delete b->events; delete b; return ra; }
  }
  *out = b;
  return MHD_OK;
}

int mhd_bunch_fill_guards(mhd_bunch* b) {
  ENTER(b);
  NOT_LOCAL(b);
  NOT_RING(b);
  if (step_gathers(b)) {
    // deferred: the one-pass step reads halos from the neighbours' interiors, so only the
    // closing faces are brought up to date now; the rest of the shell is written if and when
    // something reads it from HBM (materialise_guards)
    b->guards_stale = true;
    if (b->closing_ok) return MHD_OK;
    b->closing_ok = true;
    return b->desc.dtype == MHD_F64 ? launch_sync_closing<double>(b) : launch_sync_closing<float>(b);
  }
  b->guards_stale = false;
  b->closing_ok = true;
  return b->desc.dtype == MHD_F64 ? launch_fill<double>(b) : launch_fill<float>(b);
}

int mhd_bunch_sync_guards(mhd_bunch* b) {
  ENTER(b);
  NOT_RING(b);
  return materialise_guards(b);
}

int mhd_bunch_cfl_dt(mhd_bunch* b, double courant, double* dt_host, void* dt_dev, void* dt_per_patch_dev) {
  ENTER(b);
  NOT_LOCAL(b);
  NOT_RING(b);
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
  ENTER(b);
  NOT_LOCAL(b);
  NOT_RING(b);
  if (!(dt > 0.0) || !isfinite(dt)) return MHD_EINVAL;
  { LaunchScope ls(b, KC_MISC); k_set_dt<<<1, 256, 0, b->stream>>>(b->d_dt + 1, nullptr, dt, 0.0, b->d_rate_next, b->G.np); }
  return step_common(b);
}

int mhd_bunch_step_dev(mhd_bunch* b, const void* dt_dev, double dt_max) {
  ENTER(b);
  NOT_LOCAL(b);
  NOT_RING(b);
  if (!dt_dev || !(dt_max >= 0.0)) return MHD_EINVAL;
  { LaunchScope ls(b, KC_MISC); k_set_dt<<<1, 256, 0, b->stream>>>(b->d_dt + 1, (const double*)dt_dev, 0.0, dt_max, b->d_rate_next, b->G.np); }
  return step_common(b);
}

int mhd_bunch_current(mhd_bunch* b, void** state) {
  if (!b || !state) return MHD_ESTATE;
  ENTER(b);
  const int rc = materialise_guards(b);   // the caller is about to look at the buffer
  if (rc != MHD_OK) return rc;
  b->closing_ok = false;                  // ... and may write it
  b->rate_valid = false;
  *state = b->state[b->cur];
  return MHD_OK;
}

int mhd_bunch_status(mhd_bunch* b, int64_t* bad_cells) {
  if (!b || !bad_cells) return MHD_ESTATE;
  ENTER(b);
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

int mhd_bunch_set_path(mhd_bunch* b, int32_t path) {
  ENTER(b);
  if (path < MHD_PATH_AUTO || path > MHD_PATH_TILE2D) return MHD_EINVAL;
  if (path == MHD_PATH_ONEPASS && !b->onepass_ok) return MHD_EINVAL;
  if (path == MHD_PATH_TILE2D && !b->tile2d_ok) return MHD_EINVAL;
  if (path == MHD_PATH_TWO_KERNEL && !b->fused_ok) return MHD_EINVAL;
  const int rc = materialise_guards(b);   // the other paths read the guard shell from HBM
  if (rc != MHD_OK) return rc;
  b->path = path;
  return MHD_OK;
}

int mhd_bunch_set_tuning(mhd_bunch* b, int32_t key, int32_t value) {
  ENTER(b);
  if (value < 0) return MHD_EINVAL;
  if (key == MHD_TUNE_ONEPASS_ZSEG) {
    b->tune_zseg = value;
    return MHD_OK;
  }
  if (key == MHD_TUNE_HOST_BANDS) {
    b->tune_bands = value;
    return MHD_OK;
  }
  if (key == MHD_TUNE_HOST_MAX_PITCH) {
    b->tune_max_pitch = value;
    return MHD_OK;
  }
  if (key == MHD_TUNE_FUSED_CFL) {
    if (value > 2 || !b->onepass_ok) return MHD_EINVAL;
    b->fused_cfl = value == 1;
    b->fused_cfl_auto = value == 2;
    b->rate_valid = false;
    return MHD_OK;
  }
  if (key == MHD_TUNE_PREDICT_TY) {
    if (!b->fused_ok) return MHD_EINVAL;
    if (value != 16 && value != 8 && value != 4) return MHD_EINVAL;
    const size_t pa = (size_t)(b->G.n[0] + 5) * (value + 5);
    if (!(pa <= (size_t)predict_max_threads(value) && 39 * pa * b->esz <= (size_t)220 * 1024)) return MHD_EINVAL;
    b->pred_ty = value;
    return MHD_OK;
  }
  return MHD_EINVAL;
}

int mhd_bunch_get_path(mhd_bunch* b, int32_t* path) {
  if (!b || !path) return MHD_ESTATE;
  *path = effective_path(b);
  return MHD_OK;
}

int mhd_bunch_measure_alu_peak(int32_t dtype, int32_t device, void* scratch_dev, size_t scratch_bytes, double* tflops) {
  if (!tflops || !scratch_dev || (dtype != MHD_F32 && dtype != MHD_F64)) return MHD_EINVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev)
    return fail_cuda(cudaErrorNoDevice, "no CUDA device");
  CUDA_TRY(cudaSetDevice(device));
  cudaDeviceProp prop;
  CUDA_TRY(cudaGetDeviceProperties(&prop, device));
  void* out = scratch_dev;
  const int blocks = prop.multiProcessorCount * 8, iters = 4096;
  if (scratch_bytes < (size_t)blocks * 256 * 8) return MHD_ENOMEM;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  double best = 0.0;
  for (int rep = 0; rep < 5; ++rep) {
    cudaEventRecord(e0, 0);
    if (dtype == MHD_F64) k_fma_peak<double><<<blocks, 256>>>((double*)out, iters, 1.0000001, 1e-7);
    else k_fma_peak<float><<<blocks, 256>>>((float*)out, iters, 1.0000001f, 1e-7f);
    cudaEventRecord(e1, 0);
    cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    const double fl = 2.0 * 16.0 * iters * (double)blocks * 256.0;
    if (ms > 0.f && rep > 0) best = fmax(best, fl / (ms * 1e-3) / 1e12);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  CUDA_TRY(cudaGetLastError());
  *tflops = best;
  return MHD_OK;
}

int mhd_bunch_chunk(mhd_bunch* b, int32_t* chunk_patches) {
  if (!b || !chunk_patches) return MHD_ESTATE;
  const int path = effective_path(b);
  *chunk_patches = path == MHD_PATH_ONEPASS ? b->G.np : (path == MHD_PATH_TWO_KERNEL ? b->chunk : b->chunk_s);
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
  ENTER(b);
  b->guards_stale = false;   // the whole buffer, guard shell included, is replaced
  b->closing_ok = false;
  b->rate_valid = false;
  CUDA_TRY(cudaMemcpyAsync(b->state[b->cur], host_state, b->lay.state_bytes, cudaMemcpyHostToDevice, b->stream));
  return MHD_OK;
}

int mhd_bunch_download(mhd_bunch* b, void* host_state) {
  if (!b || !host_state) return MHD_ESTATE;
  ENTER(b);
  {
    const int rc = materialise_guards(b);
    if (rc != MHD_OK) return rc;
  }
  CUDA_TRY(cudaMemcpyAsync(host_state, b->state[b->cur], b->lay.state_bytes, cudaMemcpyDeviceToHost, b->stream));
  CUDA_TRY(cudaStreamSynchronize(b->stream));
  return MHD_OK;
}

int mhd_bunch_set_timing(mhd_bunch* b, int32_t enable) {
  ENTER(b);
  CUDA_TRY(cudaStreamSynchronize(b->stream));
  drain_events(b, false);
  for (int c = 0; c < 16; ++c) { b->cls_ms[c] = 0.0; b->cls_n[c] = 0; }
  b->timing = enable != 0;
  return MHD_OK;
}

int mhd_bunch_kernel_times(mhd_bunch* b, int32_t cap, const char** names, double* ms, int64_t* count, int32_t* n) {
  if (!b || !n) return MHD_ESTATE;
  ENTER(b);
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

}  // extern "C"

// ------------------------------------------------------- host-streaming path ----
namespace {

size_t hs_chunk_bytes(const mhd_bunch* b, int chunk) {
  return align_up((size_t)8 * chunk * b->G.n[0] * b->G.n[1] * b->G.n[2] * b->esz, 256);
}

void hs_release(mhd_bunch* b) {
  mhd_bunch::HostStream* h = b->hs;
  if (!h) return;
  for (auto* v : {&h->ev_copied, &h->ev_up, &h->ev_step, &h->ev_packed, &h->ev_dn})
    for (cudaEvent_t e : *v) if (e) cudaEventDestroy(e);
  if (h->ev_begin) cudaEventDestroy(h->ev_begin);
  if (h->ev_all_steps) cudaEventDestroy(h->ev_all_steps);
  for (cudaStream_t st : {h->s_up[0], h->s_up[1], h->s_un, h->s_pk, h->s_dn[0], h->s_dn[1]}) if (st) cudaStreamDestroy(st);
  delete h;
  b->hs = nullptr;
}

// scatter / gather planes [k0, k0+nk) of patches [p0, p0+npl) between the state and a staging buffer
template <typename T, bool PACK>
int launch_pack(mhd_bunch* b, cudaStream_t st, void* state, char* stage, int p0, int npl, int k0 = 0, int nk = -1) {
  const Geom& G = b->G;
  if (nk < 0) nk = G.n[2];
  const int vec = (int)(16 / sizeof(T));
  const long long n = (long long)8 * npl * G.n[0] * G.n[1] * nk;
  b->launches += 1;
  if (G.n[0] % vec == 0) {
    const unsigned blocks = blocks_for(n / vec, 256);
    k_pack_unpack<T, (int)(16 / sizeof(T)), PACK><<<blocks, 256, 0, st>>>(G, (T*)state, (T*)stage, p0, npl, k0, nk);
  } else {
    k_pack_unpack<T, 1, PACK><<<blocks_for(n, 256), 256, 0, st>>>(G, (T*)state, (T*)stage, p0, npl, k0, nk);
  }
  CUDA_TRY(cudaGetLastError());
  return MHD_OK;
}

// host[f][p0 .. p0+npl)[k0 .. k0+nk) <-> stage[f][0 .. npl)[0 .. nk).  Normally ONE strided copy per
// transfer: whole patches are eight contiguous rows (the eight fields: a 2D copy), a z-range of every
// patch is a 3D copy (row = the planes of one patch and field, rows per slice = patches, slices =
// fields).  The host stride between fields is that of the WHOLE host bunch, and CUDA refuses a pitch
// above cudaDevAttrMaxPitch (2^31 - 1 bytes: cudaErrorInvalidPitchValue) -- reached by 4096 patches of
// 64^3 in fp32 and by every bunch that really exceeds HBM, which is what ring mode is for.  From there
// on the transfer is eight copies, one per field, none of which names the field stride: a contiguous
// copy for whole patches, a 2D copy whose pitch is one patch for a z-range.
int hs_copy(mhd_bunch* b, cudaStream_t st, char* stage, char* host, int p0, int npl, bool to_device, int host_np = -1,
            int k0 = 0, int nk = -1) {
  const int nz = b->G.n[2];
  if (nk < 0) nk = nz;
  const size_t plane = (size_t)b->G.n[0] * b->G.n[1] * b->esz, per = plane * nz;
  const size_t hnp = (size_t)(host_np < 0 ? b->G.np : host_np);
  const size_t field = hnp * per;                                   // host bytes between two fields
  const size_t maxp = b->tune_max_pitch > 0 ? (size_t)b->tune_max_pitch : b->max_pitch;
  const cudaMemcpyKind kind = to_device ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToHost;
  if (k0 == 0 && nk == nz) {
    char* h = host + (size_t)p0 * per;
    const size_t dp = (size_t)npl * per;
    if (field <= maxp) {
      if (to_device) CUDA_TRY(cudaMemcpy2DAsync(stage, dp, h, field, dp, 8, kind, st));
      else CUDA_TRY(cudaMemcpy2DAsync(h, field, stage, dp, dp, 8, kind, st));
      return MHD_OK;
    }
    for (int f = 0; f < 8; ++f) {
      if (to_device) CUDA_TRY(cudaMemcpyAsync(stage + f * dp, h + f * field, dp, kind, st));
      else CUDA_TRY(cudaMemcpyAsync(h + f * field, stage + f * dp, dp, kind, st));
    }
    return MHD_OK;
  }
  const size_t w = plane * nk;
  if (field <= maxp) {
    cudaMemcpy3DParms q;
    memset(&q, 0, sizeof q);
    const cudaPitchedPtr hptr = make_cudaPitchedPtr(host, per, per, hnp);
    const cudaPitchedPtr dptr = make_cudaPitchedPtr(stage, w, w, (size_t)npl);
    const cudaPos hpos = make_cudaPos(plane * k0, (size_t)p0, 0), dpos = make_cudaPos(0, 0, 0);
    q.srcPtr = to_device ? hptr : dptr; q.srcPos = to_device ? hpos : dpos;
    q.dstPtr = to_device ? dptr : hptr; q.dstPos = to_device ? dpos : hpos;
    q.extent = make_cudaExtent(w, (size_t)npl, 8);
    q.kind = kind;
    CUDA_TRY(cudaMemcpy3DAsync(&q, st));
    return MHD_OK;
  }
  for (int f = 0; f < 8; ++f) {
    char* h = host + f * field + (size_t)p0 * per + plane * k0;
    char* d = stage + f * (size_t)npl * w;
    if (to_device) CUDA_TRY(cudaMemcpy2DAsync(d, w, h, per, w, (size_t)npl, kind, st));
    else CUDA_TRY(cudaMemcpy2DAsync(h, per, d, w, w, (size_t)npl, kind, st));
  }
  return MHD_OK;
}

// Schedule of one host-streamed step for a chunk size.  STEP UNITS are stepped in order: chunk 0,
// 1, .. C-1, the first chunk and the last two cut into `bands` bands of planes [za, zb) each (the
// one-pass kernel steps any plane range of its patches), every other chunk whole: downloads then start
// early, and what is left to download when the last upload lands is two bands, not two chunks.  What a unit (c, [za, zb))
// needs on the device before it may step (O1: guard zones come from the neighbours' interiors, at
// most `guard` cells deep): planes [za-guard, zb+guard) of its own chunk and of every chunk that holds
// an in-plane neighbour (o_z = 0) of one of its patches; if the range reaches below plane 0, the
// HIGHEST planes of the chunks reached through o_z = -1, and if it reaches beyond n_z, the LOWEST
// planes of the chunks reached through o_z = +1 -- the kernels read nothing else.  Uploads are PIECES
// (chunk, planes [k0, k1)): walking the units in step order, whatever a unit still misses is
// appended, so every plane of every patch crosses PCIe exactly once, the thin layers of the chunks
// ahead arrive early and no step waits for the bulk of a z-neighbour: a periodic stack of slabs
// starts stepping after a band of the first slab and ends with the download of one band of the last
// (the whole-chunk schedule ended with three slabs: the first one waited for the last one's upload).
// ready[u] = index of the last piece unit u needs.  Patches too thin for two disjoint layers
// (n_z < 2 guard + 1, collapsed dimensions) or thicker than 64 planes are needed whole.
struct HsPlan { std::vector<int> piece_chunk, piece_k0, piece_k1, unit_chunk, unit_za, unit_zb, ready; };
bool hs_layered(int nz, int guard) { return guard >= 1 && nz >= 2 * guard + 1 && nz <= 64; }
int hs_bands(int nz, int guard, int bands) {                      // bands of at least eight planes
  if (!hs_layered(nz, guard) || bands < 1) return 1;
  return bands > nz / 8 ? (nz / 8 > 1 ? nz / 8 : 1) : bands;
}
HsPlan hs_plan(const int* nb, int np, int chunk, int nz, int guard, int bands) {
  HsPlan pl;
  const int C = (np + chunk - 1) / chunk;
  const bool layered = hs_layered(nz, guard);
  bands = hs_bands(nz, guard, bands);
  const int NZ = layered ? nz : 1;                               // one bit per plane, or one for the whole patch
  auto planes = [&](int a, int z) -> unsigned long long {
    a = std::max(a, 0); z = std::min(z, NZ);
    if (a >= z) return 0ull;
    return (z - a == 64 ? ~0ull : ((1ull << (z - a)) - 1ull)) << a;
  };
  std::vector<unsigned long long> have(C, 0ull);
  std::vector<unsigned char> reach(C, 0);                        // bit 0: o_z = -1, bit 1: o_z = 0, bit 2: o_z = +1
  std::vector<int> touched;
  for (int c = 0; c < C; ++c) {
    touched.clear();
    auto mark = [&](int q, int bit) { if (!reach[q]) touched.push_back(q); reach[q] |= (unsigned char)bit; };
    mark(c, 2);
    for (int p = c * chunk; p < std::min(np, (c + 1) * chunk); ++p)
      for (int k = 0; k < 27; ++k) {
        const int q = nb[(size_t)p * 27 + k];
        if (q >= 0) mark(q / chunk, 1 << (k / 9));
      }
    std::sort(touched.begin() + 1, touched.end());               // own chunk first, then by index
    const int J = (c == 0 || c >= C - 2) ? bands : 1;
    for (int j = 0; j < J; ++j) {
      const int za = (int)((long long)nz * j / J), zb = (int)((long long)nz * (j + 1) / J);
      const int lo = za - guard, hi = zb + guard;
      for (int q : touched) {
        unsigned long long w = 0ull;
        if (!layered) w = 1ull;
        else {
          if (reach[q] & 2) w |= planes(lo, hi);
          if ((reach[q] & 1) && lo < 0) w |= planes(nz + lo, nz);
          if ((reach[q] & 4) && hi > nz) w |= planes(0, hi - nz);
        }
        unsigned long long miss = w & ~have[q];
        have[q] |= miss;
        while (miss) {                                           // maximal runs of missing planes
          int k0 = 0;
          while (!((miss >> k0) & 1ull)) ++k0;
          int k1 = k0;
          while (k1 < NZ && ((miss >> k1) & 1ull)) ++k1;
          pl.piece_chunk.push_back(q);
          pl.piece_k0.push_back(layered ? k0 : 0);
          pl.piece_k1.push_back(layered ? k1 : nz);
          miss &= ~planes(k0, k1);
        }
      }
      pl.unit_chunk.push_back(c); pl.unit_za.push_back(za); pl.unit_zb.push_back(zb);
      pl.ready.push_back((int)pl.piece_chunk.size() - 1);
    }
    for (int q : touched) reach[q] = 0;
  }
  return pl;
}
// Makespan of that schedule in units of "one patch across PCIe": uploads back to back, a step
// costs HS_ALPHA per patch, a download 1 per patch; fixed costs per upload piece, step and download.
// Calibrated on a B200 / PCIe 5 box with both directions busy (21 us per 32^3 fp32 patch): an H2D
// copy starts ~40 us after the previous one has ended (its completion signal queues behind the
// D2H data), a D2H copy ~15 us, a unit's launches take ~10 us.
constexpr double HS_ALPHA = 0.33, HS_EPS_UP = 2.0, HS_EPS_STEP = 0.5, HS_EPS_DN = 0.7;
double hs_makespan(int np, int chunk, int nz, const HsPlan& pl) {
  const int NU = (int)pl.ready.size(), NPC = (int)pl.piece_chunk.size();
  auto size = [&](int c) { return (double)std::min(chunk, np - c * chunk); };
  std::vector<double> t_up(NPC);
  double t = 0.0;
  for (int u = 0; u < NPC; ++u) {
    t += size(pl.piece_chunk[u]) * (pl.piece_k1[u] - pl.piece_k0[u]) / (double)nz + HS_EPS_UP;
    t_up[u] = t;
  }
  double t_step = 0.0, t_dn = 0.0;
  for (int u = 0; u < NU; ++u) {
    const double sz = size(pl.unit_chunk[u]) * (pl.unit_zb[u] - pl.unit_za[u]) / (double)nz;
    t_step = std::max(t_step, t_up[pl.ready[u]]) + HS_ALPHA * sz + HS_EPS_STEP;
    t_dn = std::max(t_dn, t_step) + sz + HS_EPS_DN;
  }
  return t_dn;
}
// default chunk and bands: the candidate with the shortest simulated step
void hs_default(const int* nb, int np, int nz, int guard, bool can_band, int chunk_fixed, int* chunk_out, int* bands_out) {
  int best = np, best_b = 1;
  double best_t = 1e300;
  for (int k : {1, 2, 3, 4, 6, 8, 12, 16, 24, 32, 48, 64, 96, 128}) {
    const int chunk = chunk_fixed > 0 ? chunk_fixed : (np + k - 1) / k;
    if (chunk < 1) break;
    for (int bands : {1, 2, 4}) {
      if (bands > 1 && !can_band) break;
      const double tt = hs_makespan(np, chunk, nz, hs_plan(nb, np, chunk, nz, guard, bands));
      // near ties (0.2 %) go to more bands of the same chunk: measured 2.4 % faster on config 2
      // (13.47 against 13.80 ms) where the model sees none -- it overestimates the start-up of small copies
      const bool tie = chunk == best && bands > best_b && tt < best_t * 1.002;
      if (tt < best_t - 1e-9 || tie) { best_t = std::min(tt, best_t); best = chunk; best_b = bands; }
    }
    if (chunk == 1 || chunk_fixed > 0) break;
  }
  *chunk_out = best;
  *bands_out = best_b;
}

}  // namespace

extern "C" {

int mhd_bunch_host_query(mhd_bunch* b, int32_t chunk_patches, mhd_bunch_host_layout* out) {
  if (!b || !out) return MHD_ESTATE;
  const bool pipelined = b->all_nbr && step_gathers(b);
  const bool can_band = pipelined && effective_path(b) == MHD_PATH_ONEPASS;    // the one-pass kernel steps plane ranges
  int chunk = chunk_patches > b->G.np ? b->G.np : chunk_patches, bands = 1;
  hs_default(b->h_nbr->data(), b->G.np, b->G.n[2], b->G.g[2], can_band, chunk, &chunk, &bands);
  if (can_band && b->tune_bands >= 1) bands = hs_bands(b->G.n[2], b->G.g[2], b->tune_bands);     // mhd_bunch_set_tuning
  out->chunk_patches = chunk;
  out->nchunk = (b->G.np + chunk - 1) / chunk;
  out->host_bytes = (size_t)8 * b->G.np * b->G.n[0] * b->G.n[1] * b->G.n[2] * b->esz;
  out->staging_bytes = 4 * hs_chunk_bytes(b, chunk);
  out->pipelined = pipelined ? 1 : 0;
  out->bands = bands;
  return MHD_OK;
}

int mhd_bunch_host_schedule(const int32_t* nbr, int32_t npatch, int32_t nz, int32_t guard, int32_t chunk_patches, int32_t bands,
                            int32_t* chunk_out, int32_t* bands_out, int32_t* npiece_out, int32_t* piece_chunk,
                            int32_t* piece_k0, int32_t* piece_k1, int32_t* nunit_out, int32_t* unit_chunk, int32_t* unit_za,
                            int32_t* unit_zb, int32_t* ready, int32_t cap, double* makespan) {
  if (!nbr || npatch < 1 || nz < 1 || guard < 0 || !chunk_out || !bands_out || !npiece_out || !nunit_out) return MHD_EINVAL;
  for (long long c = 0; c < 27ll * npatch; ++c)
    if (nbr[c] < -1 || nbr[c] >= npatch) return MHD_EINVAL;
  int chunk = chunk_patches > npatch ? npatch : chunk_patches, bb = bands;
  if (chunk <= 0 || bands <= 0) {
    int c2, b2;
    hs_default(nbr, npatch, nz, guard, true, chunk > 0 ? chunk : 0, &c2, &b2);
    if (chunk <= 0) chunk = c2;
    if (bands <= 0) bb = b2;
  }
  const HsPlan pl = hs_plan(nbr, npatch, chunk, nz, guard, bb);
  const int NU = (int)pl.ready.size(), NPC = (int)pl.piece_chunk.size();
  *chunk_out = chunk;
  *bands_out = hs_bands(nz, guard, bb);
  *npiece_out = NPC;
  *nunit_out = NU;
  if (makespan) *makespan = hs_makespan(npatch, chunk, nz, pl);
  if (piece_chunk || piece_k0 || piece_k1 || unit_chunk || unit_za || unit_zb || ready) {
    if (cap < NPC || cap < NU) return MHD_ENOMEM;
    for (int u = 0; u < NPC; ++u) {
      if (piece_chunk) piece_chunk[u] = pl.piece_chunk[u];
      if (piece_k0) piece_k0[u] = pl.piece_k0[u];
      if (piece_k1) piece_k1[u] = pl.piece_k1[u];
    }
    for (int u = 0; u < NU; ++u) {
      if (unit_chunk) unit_chunk[u] = pl.unit_chunk[u];
      if (unit_za) unit_za[u] = pl.unit_za[u];
      if (unit_zb) unit_zb[u] = pl.unit_zb[u];
      if (ready) ready[u] = pl.ready[u];
    }
  }
  return MHD_OK;
}

int mhd_bunch_host_attach(mhd_bunch* b, void* staging_dev, size_t staging_bytes, int32_t chunk_patches) {
  ENTER(b);
  NOT_RING(b);
  if (!staging_dev || ((uintptr_t)staging_dev & 15)) return MHD_EINVAL;
  if (!b->all_nbr) return MHD_EINVAL;   // the compact host layout has no room for evolved closing faces
  mhd_bunch_host_layout lay;
  int rc = mhd_bunch_host_query(b, chunk_patches, &lay);
  if (rc != MHD_OK) return rc;
  if (staging_bytes < lay.staging_bytes) return MHD_ENOMEM;
  hs_release(b);
  mhd_bunch::HostStream* h = new (std::nothrow) mhd_bunch::HostStream();
  if (!h) return MHD_ENOMEM;
  h->s_up[0] = h->s_up[1] = h->s_un = h->s_pk = h->s_dn[0] = h->s_dn[1] = nullptr;
  h->ev_begin = h->ev_all_steps = nullptr;
  b->hs = h;                               // owned by the handle from here on: released by detach / destroy,
  struct Guard {                           // or right here if the attach fails half way
    mhd_bunch* b; bool ok;
    ~Guard() { if (!ok) hs_release(b); }
  } guard{b, false};
  h->chunk = lay.chunk_patches;
  h->nchunk = lay.nchunk;
  const size_t cb = hs_chunk_bytes(b, h->chunk);
  for (int i = 0; i < 2; ++i) {
    h->stage_up[i] = (char*)staging_dev + (size_t)i * cb;
    h->stage_dn[i] = (char*)staging_dev + (size_t)(2 + i) * cb;
  }
  HsPlan pl = hs_plan(b->h_nbr->data(), b->G.np, h->chunk, b->G.n[2], b->G.g[2], lay.bands);
  h->piece_chunk = pl.piece_chunk;
  h->piece_k0 = pl.piece_k0;
  h->piece_k1 = pl.piece_k1;
  h->unit_chunk = pl.unit_chunk;
  h->unit_za = pl.unit_za;
  h->unit_zb = pl.unit_zb;
  h->ready = pl.ready;
  CUDA_TRY(cudaSetDevice(b->desc.device));
  for (cudaStream_t* st : {&h->s_up[0], &h->s_up[1], &h->s_un, &h->s_pk, &h->s_dn[0], &h->s_dn[1]})
    CUDA_TRY(cudaStreamCreateWithFlags(st, cudaStreamNonBlocking));
  CUDA_TRY(cudaEventCreateWithFlags(&h->ev_begin, cudaEventDisableTiming));
  CUDA_TRY(cudaEventCreateWithFlags(&h->ev_all_steps, cudaEventDisableTiming));
  const size_t NPC = h->piece_chunk.size();
  h->ev_copied.assign(NPC, nullptr);
  h->ev_up.assign(NPC, nullptr);
  h->ev_step.assign(h->unit_chunk.size(), nullptr);
  h->ev_packed.assign(h->unit_chunk.size(), nullptr);
  h->ev_dn.assign(h->unit_chunk.size(), nullptr);
  for (auto* v : {&h->ev_copied, &h->ev_up, &h->ev_step, &h->ev_packed, &h->ev_dn})
    for (cudaEvent_t& e : *v) CUDA_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
  guard.ok = true;
  return MHD_OK;
}

static int step_host_impl(mhd_bunch* b, const void* host_in, void* host_out, double dt, double courant,
                          double* dt_used, double* dt_next);

int mhd_bunch_step_host(mhd_bunch* b, const void* host_in, void* host_out, double dt, double courant,
                        double* dt_used, double* dt_next) {
  ENTER(b);
  NOT_LOCAL(b);
  NOT_RING(b);
  const int rc = step_host_impl(b, host_in, host_out, dt, courant, dt_used, dt_next);
  if (rc != MHD_OK && b->hs) {
    // copies into / out of the caller's host buffers may still be in flight: drain them before
    // the caller sees the error and reuses the buffers
    cudaStreamSynchronize(b->stream);
    for (cudaStream_t st : {b->hs->s_up[0], b->hs->s_up[1], b->hs->s_un, b->hs->s_pk, b->hs->s_dn[0], b->hs->s_dn[1]})
      if (st) cudaStreamSynchronize(st);
  }
  return rc;
}

static int step_host_impl(mhd_bunch* b, const void* host_in, void* host_out, double dt, double courant,
                          double* dt_used, double* dt_next) {
  mhd_bunch::HostStream* h = b->hs;
  if (!h) return MHD_ESTATE;
  if (!host_in || !host_out) return MHD_EINVAL;
  if (!(courant > 0.0) || !isfinite(courant) || !isfinite(dt) || dt < 0.0) return MHD_EINVAL;
  const bool f64 = b->desc.dtype == MHD_F64;
  const bool have_dt = dt > 0.0;
  const bool pipelined = step_gathers(b);
  const bool onepass = effective_path(b) == MHD_PATH_ONEPASS;
  const Geom& G = b->G;
  const int C = h->nchunk, NPC = (int)h->piece_chunk.size();
  auto range = [&](int c, int& p0, int& npl) { p0 = c * h->chunk; npl = std::min(h->chunk, G.np - p0); };
  int rc;

  // the library's streams start after whatever the caller's stream has enqueued so far
  CUDA_TRY(cudaEventRecord(h->ev_begin, b->stream));
  for (cudaStream_t st : {h->s_up[0], h->s_up[1], h->s_un, h->s_pk, h->s_dn[0], h->s_dn[1]}) CUDA_TRY(cudaStreamWaitEvent(st, h->ev_begin, 0));

  // ---- uploads: host -> staging (copy streams) -> interiors of the current level (unpack stream).
  // Two staging buffers, one per copy stream: piece u+1 crosses PCIe while piece u is scattered.
  int next_piece = 0;
  auto upload_through = [&](int last) -> int {
    for (; next_piece <= last; ++next_piece) {
      const int u = next_piece, p0 = h->piece_chunk[u] * h->chunk, npl = std::min(h->chunk, G.np - p0);
      const int k0 = h->piece_k0[u], nk = h->piece_k1[u] - k0;
      char* st = h->stage_up[u & 1];
      cudaStream_t su = h->s_up[u & 1];
      if (u >= 2) CUDA_TRY(cudaStreamWaitEvent(su, h->ev_up[u - 2], 0));           // the buffer has been scattered
      int r2 = hs_copy(b, su, st, (char*)const_cast<void*>(host_in), p0, npl, true, -1, k0, nk);
      if (r2 != MHD_OK) return r2;
      CUDA_TRY(cudaEventRecord(h->ev_copied[u], su));
      CUDA_TRY(cudaStreamWaitEvent(h->s_un, h->ev_copied[u], 0));
      r2 = f64 ? launch_pack<double, false>(b, h->s_un, b->state[b->cur], st, p0, npl, k0, nk)
               : launch_pack<float, false>(b, h->s_un, b->state[b->cur], st, p0, npl, k0, nk);
      if (r2 != MHD_OK) return r2;
      CUDA_TRY(cudaEventRecord(h->ev_up[u], h->s_un));
    }
    return MHD_OK;
  };
  b->closing_ok = false;
  b->guards_stale = false;
  b->rate_valid = false;

  const bool overlap_up = pipelined && have_dt;   // steps start while later pieces still upload
  if (!overlap_up) {
    if ((rc = upload_through(NPC - 1)) != MHD_OK) return rc;
    CUDA_TRY(cudaStreamWaitEvent(b->stream, h->ev_up[NPC - 1], 0));
    if ((rc = mhd_bunch_fill_guards(b)) != MHD_OK) return rc;    // deferred on the one-pass path: closing faces only
    if (!have_dt) {
      rc = f64 ? launch_cfl<double>(b, courant, nullptr, nullptr) : launch_cfl<float>(b, courant, nullptr, nullptr);
      if (rc != MHD_OK) return rc;
    }
  }
  { LaunchScope ls(b, KC_MISC);
    k_set_dt<<<1, 256, 0, b->stream>>>(b->d_dt + 1, have_dt ? nullptr : b->d_dt, dt, 0.0, b->d_rate_next, b->G.np); }

  // ---- steps, and the way back: interiors of the new level -> staging (pack stream) -> host
  // (copy-out stream), again through two staging buffers
  void* const next = b->state[1 - b->cur];
  const int NU = (int)h->unit_chunk.size();
  auto download = [&](int u, cudaEvent_t after) -> int {
    int p0, npl;
    range(h->unit_chunk[u], p0, npl);
    const int za = h->unit_za[u], nk = h->unit_zb[u] - za;
    char* st = h->stage_dn[u & 1];
    CUDA_TRY(cudaStreamWaitEvent(h->s_pk, after, 0));
    if (u >= 2) CUDA_TRY(cudaStreamWaitEvent(h->s_pk, h->ev_dn[u - 2], 0));        // the buffer has left for the host
    int r2 = f64 ? launch_pack<double, true>(b, h->s_pk, next, st, p0, npl, za, nk)
                 : launch_pack<float, true>(b, h->s_pk, next, st, p0, npl, za, nk);
    if (r2 != MHD_OK) return r2;
    CUDA_TRY(cudaEventRecord(h->ev_packed[u], h->s_pk));
    cudaStream_t sd = h->s_dn[u & 1];
    CUDA_TRY(cudaStreamWaitEvent(sd, h->ev_packed[u], 0));
    if ((r2 = hs_copy(b, sd, st, (char*)host_out, p0, npl, false, -1, za, nk)) != MHD_OK) return r2;
    CUDA_TRY(cudaEventRecord(h->ev_dn[u], sd));
    return MHD_OK;
  };
  if (pipelined) {
    for (int u = 0; u < NU; ++u) {
      int p0, npl;
      range(h->unit_chunk[u], p0, npl);
      const int za = h->unit_za[u], zb = h->unit_zb[u];
      if (overlap_up) {
        // enqueue what this unit needs, then the unit: the host stays just ahead of the device
        if ((rc = upload_through(h->ready[u])) != MHD_OK) return rc;
        CUDA_TRY(cudaStreamWaitEvent(b->stream, h->ev_up[h->ready[u]], 0));
        rc = f64 ? launch_sync_closing<double>(b, p0, npl, za, zb) : launch_sync_closing<float>(b, p0, npl, za, zb);
        if (rc != MHD_OK) return rc;
        b->guards_stale = true;    // halos of this unit come through the neighbour table
      }
      if (onepass) rc = OnePassLaunch<float>::run(b, b->d_dt + 1, p0, npl, false, za, zb);
      else if (za != 0 || zb != G.n[2]) rc = MHD_ESTATE;          // only the one-pass kernel steps plane ranges
      else if (effective_path(b) == MHD_PATH_TILE2D) rc = f64 ? launch_tile2d<double>(b, p0, npl) : launch_tile2d<float>(b, p0, npl);
      else rc = f64 ? launch_fused_range<double>(b, p0, npl) : launch_fused_range<float>(b, p0, npl);
      if (rc != MHD_OK) return rc;
      CUDA_TRY(cudaEventRecord(h->ev_step[u], b->stream));
      if ((rc = download(u, h->ev_step[u])) != MHD_OK) return rc;
    }
    b->cur = 1 - b->cur;
    b->guards_stale = true;   // the new level's shell is owed (deferred fill), its closing faces are current
    b->closing_ok = true;
    b->rate_valid = onepass && onepass_cfle(b);  // every unit went through the one-pass epilogue since k_set_dt
  } else {
    if ((rc = step_common(b)) != MHD_OK) return rc;
    CUDA_TRY(cudaEventRecord(h->ev_all_steps, b->stream));
    for (int u = 0; u < NU; ++u)
      if ((rc = download(u, h->ev_all_steps)) != MHD_OK) return rc;
    if ((rc = mhd_bunch_fill_guards(b)) != MHD_OK) return rc;   // cfl of the new level reads its closing faces
  }

  // ---- CFL step of the new level (overlaps the last downloads) -----------------------
  double dts[2] = {0.0, 0.0};
  CUDA_TRY(cudaMemcpyAsync(&dts[1], b->d_dt + 1, sizeof(double), cudaMemcpyDeviceToHost, b->stream));
  rc = f64 ? launch_cfl<double>(b, courant, nullptr, nullptr) : launch_cfl<float>(b, courant, nullptr, nullptr);
  if (rc != MHD_OK) return rc;
  CUDA_TRY(cudaMemcpyAsync(&dts[0], b->d_dt, sizeof(double), cudaMemcpyDeviceToHost, b->stream));
  CUDA_TRY(cudaStreamSynchronize(b->stream));
  for (cudaStream_t st : {h->s_dn[0], h->s_dn[1], h->s_pk, h->s_un, h->s_up[0], h->s_up[1]}) CUDA_TRY(cudaStreamSynchronize(st));
  if (dt_used) *dt_used = dts[1];
  if (dt_next) *dt_next = dts[0];
  return MHD_OK;
}

int mhd_bunch_host_detach(mhd_bunch* b) {
  ENTER(b);
  hs_release(b);
  return MHD_OK;
}

}  // extern "C"

// ------------------------------------------------------------------ ring mode ----
namespace {

// Plan of one ring step for a host bunch of NP patches cut into chunks of `chunk` consecutive
// patches, stepped in order 0..C-1 through a window of R chunk slots.  need(c) = chunks that hold a
// neighbour of a patch of c (c included); before step c every chunk of need(c) must be resident.  A
// missing chunk goes into a free slot, else into the slot of a resident chunk that step c does not
// need and whose next use lies farthest ahead (it is uploaded again later if it is needed again:
// the first chunks of a periodic bunch are).  Returns false if need(c) does not fit in R slots.
struct RingPlan {
  int C;
  std::vector<int> up_chunk, up_slot, up_step, up_wait, slot_of_step;
  std::vector<std::vector<int>> need;
};
bool ring_plan(const int* nb, int NP, int chunk, int R, RingPlan* pl) {
  const int C = (NP + chunk - 1) / chunk;
  pl->C = C;
  pl->need.assign(C, {});
  for (int c = 0; c < C; ++c) {
    std::vector<char> m(C, 0);
    m[c] = 1;
    for (int p = c * chunk; p < std::min(NP, (c + 1) * chunk); ++p)
      for (int k = 0; k < 27; ++k) {
        const int q = nb[(size_t)p * 27 + k];
        if (q >= 0) m[q / chunk] = 1;
      }
    for (int x = 0; x < C; ++x) if (m[x]) pl->need[c].push_back(x);
    if ((int)pl->need[c].size() > R) return false;
  }
  std::vector<int> slot_chunk(R, -1), where(C, -1), last_read(R, -1);
  pl->slot_of_step.assign(C, -1);
  for (int c = 0; c < C; ++c) {
    std::vector<char> needed(C, 0);
    for (int x : pl->need[c]) needed[x] = 1;
    for (int x : pl->need[c]) {
      if (where[x] >= 0) continue;
      int s = -1;
      for (int r = 0; r < R && s < 0; ++r) if (slot_chunk[r] < 0) s = r;
      if (s < 0) {
        int best = -1;
        for (int r = 0; r < R; ++r) {
          const int e = slot_chunk[r];
          if (needed[e]) continue;
          int next = C + 1;                                   // next step that needs e
          for (int t = c + 1; t < C && next > C; ++t)
            for (int y : pl->need[t]) if (y == e) { next = t; break; }
          if (next > best) { best = next; s = r; }
        }
        if (s < 0) return false;
        where[slot_chunk[s]] = -1;
      }
      pl->up_chunk.push_back(x); pl->up_slot.push_back(s); pl->up_step.push_back(c); pl->up_wait.push_back(last_read[s]);
      slot_chunk[s] = x; where[x] = s;
    }
    for (int x : pl->need[c]) last_read[where[x]] = c;
    pl->slot_of_step[c] = where[c];
  }
  return true;
}

void ring_release(mhd_bunch* b) {
  mhd_bunch::Ring* r = b->ring;
  if (!r) return;
  if (r->s_up) cudaStreamSynchronize(r->s_up);
  if (r->s_dn) cudaStreamSynchronize(r->s_dn);
  for (auto* v : {&r->ev_up, &r->ev_step, &r->ev_dn})
    for (cudaEvent_t e : *v) if (e) cudaEventDestroy(e);
  if (r->s_up) cudaStreamDestroy(r->s_up);
  if (r->s_dn) cudaStreamDestroy(r->s_dn);
  delete r;
  b->ring = nullptr;
  // the window's own neighbour table goes back on the device
  cudaMemcpyAsync(b->d_nbr, b->h_nbr->data(), sizeof(int) * 27 * (size_t)b->G.np, cudaMemcpyHostToDevice, b->stream);
  cudaStreamSynchronize(b->stream);
}

}  // namespace

extern "C" {

int mhd_bunch_ring_plan(const int32_t* nbr, int32_t npatch, int32_t chunk_patches, int32_t ring_chunks, int32_t* nchunk,
                        int32_t* nupload, int32_t* up_chunk, int32_t* up_slot, int32_t* up_step, int32_t* step_slot, int32_t cap) {
  if (!nbr || npatch < 1 || chunk_patches < 1 || ring_chunks < 1 || !nchunk || !nupload) return MHD_EINVAL;
  for (long long c = 0; c < 27ll * npatch; ++c)
    if (nbr[c] < -1 || nbr[c] >= npatch) return MHD_EINVAL;
  RingPlan pl;
  if (!ring_plan(nbr, npatch, chunk_patches, ring_chunks, &pl)) return MHD_ENOMEM;
  *nchunk = pl.C;
  *nupload = (int)pl.up_chunk.size();
  if (up_chunk || up_slot || up_step) {
    if (cap < *nupload) return MHD_ENOMEM;
    for (int u = 0; u < *nupload; ++u) {
      if (up_chunk) up_chunk[u] = pl.up_chunk[u];
      if (up_slot) up_slot[u] = pl.up_slot[u];
      if (up_step) up_step[u] = pl.up_step[u];
    }
  }
  if (step_slot) {
    if (cap < pl.C) return MHD_ENOMEM;
    for (int c = 0; c < pl.C; ++c) step_slot[c] = pl.slot_of_step[c];
  }
  return MHD_OK;
}

int mhd_bunch_ring_attach(mhd_bunch* b, const int32_t* nbr, int32_t npatch, int32_t chunk_patches, void* staging_dev,
                          size_t staging_bytes) {
  ENTER(b);
  NOT_LOCAL(b);
  if (!nbr || npatch < 1 || chunk_patches < 1 || !staging_dev || ((uintptr_t)staging_dev & 15)) return MHD_EINVAL;
  if (!b->onepass_ok || b->G.n[0] % (int)(16 / b->esz) != 0) return MHD_EINVAL;     // the step must gather its halos
  for (long long c = 0; c < 27ll * npatch; ++c)
    if (nbr[c] < 0 || nbr[c] >= npatch) return MHD_EINVAL;                          // no outflow sides (compact host layout)
  if (!table_is_consistent(nbr, npatch)) return MHD_EINVAL;
  const int R = b->G.np / chunk_patches;
  if (R < 1) return MHD_ENOMEM;
  if (staging_bytes < 2 * hs_chunk_bytes(b, chunk_patches)) return MHD_ENOMEM;
  RingPlan pl;
  if (!ring_plan(nbr, npatch, chunk_patches, R, &pl)) return MHD_ENOMEM;
  hs_release(b);
  ring_release(b);
  mhd_bunch::Ring* r = new (std::nothrow) mhd_bunch::Ring();
  if (!r) return MHD_ENOMEM;
  r->s_up = r->s_dn = nullptr;
  b->ring = r;
  struct Guard { mhd_bunch* b; bool ok; ~Guard() { if (!ok) ring_release(b); } } guard{b, false};
  r->NP = npatch; r->chunk = chunk_patches; r->nchunk = pl.C; r->nslot = R;
  r->up_chunk = pl.up_chunk; r->up_slot = pl.up_slot; r->up_step = pl.up_step; r->up_wait = pl.up_wait;
  r->slot_of_step = pl.slot_of_step;
  r->stage_up = (char*)staging_dev;
  r->stage_dn = (char*)staging_dev + hs_chunk_bytes(b, chunk_patches);
  // neighbour rows in slot space: when chunk c is stepped, chunk x of need(c) sits in the slot the
  // plan put it in at that time -- replay the plan
  r->rows.assign((size_t)npatch * 27, 0);
  {
    std::vector<int> where(pl.C, -1), slot_chunk(R, -1);
    size_t u = 0;
    for (int c = 0; c < pl.C; ++c) {
      for (; u < pl.up_chunk.size() && pl.up_step[u] == c; ++u) {
        if (slot_chunk[pl.up_slot[u]] >= 0) where[slot_chunk[pl.up_slot[u]]] = -1;
        slot_chunk[pl.up_slot[u]] = pl.up_chunk[u];
        where[pl.up_chunk[u]] = pl.up_slot[u];
      }
      for (int p = c * chunk_patches; p < std::min(npatch, (c + 1) * chunk_patches); ++p)
        for (int k = 0; k < 27; ++k) {
          const int q = nbr[(size_t)p * 27 + k], cq = q / chunk_patches;
          r->rows[(size_t)p * 27 + k] = where[cq] * chunk_patches + (q - cq * chunk_patches);
        }
    }
  }
  CUDA_TRY(cudaStreamCreateWithFlags(&r->s_up, cudaStreamNonBlocking));
  CUDA_TRY(cudaStreamCreateWithFlags(&r->s_dn, cudaStreamNonBlocking));
  r->ev_up.assign(pl.up_chunk.size(), nullptr);
  r->ev_step.assign(pl.C, nullptr);
  r->ev_dn.assign(R, nullptr);
  for (auto* v : {&r->ev_up, &r->ev_step, &r->ev_dn})
    for (cudaEvent_t& e : *v) CUDA_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
  guard.ok = true;
  return MHD_OK;
}

static int step_ring_body(mhd_bunch* b, const void* host_in, void* host_out, double dt, double courant, double* dt_next) {
  mhd_bunch::Ring* r = b->ring;
  const Geom& G = b->G;
  const int C = r->nchunk;
  { LaunchScope ls(b, KC_MISC);
    k_set_dt<<<1, 256, 0, b->stream>>>(b->d_dt + 1, nullptr, dt, 0.0, b->d_rate_next, G.np); }
  cudaEvent_t ev_begin = r->ev_step[C - 1];      // free at this point: marks "everything enqueued so far"
  CUDA_TRY(cudaEventRecord(ev_begin, b->stream));
  CUDA_TRY(cudaStreamWaitEvent(r->s_up, ev_begin, 0));
  CUDA_TRY(cudaStreamWaitEvent(r->s_dn, ev_begin, 0));
  void* const cur = b->state[b->cur];
  void* const next = b->state[1 - b->cur];
  std::vector<char> dn_pending(r->nslot, 0);
  size_t u = 0;
  for (int c = 0; c < C; ++c) {
    for (; u < r->up_chunk.size() && r->up_step[u] == c; ++u) {
      const int x = r->up_chunk[u], s = r->up_slot[u];
      const int hp0 = x * r->chunk, npl = std::min(r->chunk, r->NP - hp0);
      if (r->up_wait[u] >= 0) CUDA_TRY(cudaStreamWaitEvent(r->s_up, r->ev_step[r->up_wait[u]], 0));   // readers of the slot are done
      int e = hs_copy(b, r->s_up, r->stage_up, (char*)const_cast<void*>(host_in), hp0, npl, true, r->NP);
      if (e != MHD_OK) return e;
      e = launch_pack<float, false>(b, r->s_up, cur, r->stage_up, s * r->chunk, npl);   // into the slot's patches
      if (e != MHD_OK) return e;
      CUDA_TRY(cudaEventRecord(r->ev_up[u], r->s_up));
    }
    const int s = r->slot_of_step[c], p0 = s * r->chunk, hp0 = c * r->chunk, npl = std::min(r->chunk, r->NP - hp0);
    if (u > 0) CUDA_TRY(cudaStreamWaitEvent(b->stream, r->ev_up[u - 1], 0));     // uploads are in order: the latest covers all
    CUDA_TRY(cudaMemcpyAsync(b->d_nbr + (size_t)p0 * 27, r->rows.data() + (size_t)hp0 * 27, sizeof(int) * 27 * npl,
                             cudaMemcpyHostToDevice, b->stream));
    {
      const int e = launch_sync_closing<float>(b, p0, npl);
      if (e != MHD_OK) return e;
    }
    if (dn_pending[s]) CUDA_TRY(cudaStreamWaitEvent(b->stream, r->ev_dn[s], 0));   // the slot's previous result has left
    b->guards_stale = true;
    {
      const int e = OnePassLaunch<float>::run(b, b->d_dt + 1, p0, npl, false);
      if (e != MHD_OK) return e;
    }
    CUDA_TRY(cudaEventRecord(r->ev_step[c], b->stream));
    CUDA_TRY(cudaStreamWaitEvent(r->s_dn, r->ev_step[c], 0));
    {
      int e = launch_pack<float, true>(b, r->s_dn, next, r->stage_dn, p0, npl);
      if (e != MHD_OK) return e;
      e = hs_copy(b, r->s_dn, r->stage_dn, (char*)host_out, hp0, npl, false, r->NP);
      if (e != MHD_OK) return e;
    }
    CUDA_TRY(cudaEventRecord(r->ev_dn[s], r->s_dn));
    dn_pending[s] = 1;
  }
  { LaunchScope ls(b, KC_MISC);
    k_cfl_final<<<1, 256, 0, b->stream>>>(b->d_rate_next, G.np, courant, b->d_dt, nullptr, nullptr); }
  double dts = 0.0;
  CUDA_TRY(cudaMemcpyAsync(&dts, b->d_dt, sizeof(double), cudaMemcpyDeviceToHost, b->stream));
  CUDA_TRY(cudaStreamSynchronize(b->stream));
  CUDA_TRY(cudaStreamSynchronize(r->s_dn));
  CUDA_TRY(cudaStreamSynchronize(r->s_up));
  if (dt_next) *dt_next = dts;
  return MHD_OK;
}

int mhd_bunch_step_ring(mhd_bunch* b, const void* host_in, void* host_out, double dt, double courant, double* dt_next) {
  ENTER(b);
  NOT_LOCAL(b);
  mhd_bunch::Ring* r = b->ring;
  if (!r) return MHD_ESTATE;
  if (!host_in || !host_out || host_in == host_out) return MHD_EINVAL;
  if (!(dt > 0.0) || !isfinite(dt) || !(courant > 0.0) || !isfinite(courant)) return MHD_EINVAL;
  const bool fused_saved = b->fused_cfl, gather_saved = b->gather_ok;
  b->fused_cfl = true;        // the CFL rates of the new level come out of the step's epilogue, slot by slot
  b->gather_ok = true;        // halos through the (slot-space) neighbour rows
  const int rc = step_ring_body(b, host_in, host_out, dt, courant, dt_next);
  if (rc != MHD_OK) {
    cudaStreamSynchronize(b->stream);
    cudaStreamSynchronize(r->s_up);
    cudaStreamSynchronize(r->s_dn);
  }
  b->fused_cfl = fused_saved;
  b->gather_ok = gather_saved;
  b->guards_stale = false;
  b->closing_ok = false;
  b->rate_valid = false;
  return rc;
}

int mhd_bunch_ring_detach(mhd_bunch* b) {
  ENTER(b);
  ring_release(b);
  return MHD_OK;
}

}  // extern "C"

// ------------------------------------------------------- local time steps ----
namespace {

bool times_equal(double a, double b) {
  const double s = fmax(fabs(a), fabs(b));
  return fabs(a - b) <= 1e-12 * (s > 1.0 ? s : 1.0);
}

// steps the patches d_plist[0..n) (all with their newer slice in buffer `side`) by d_dtlist
template <typename T>
int launch_step_list(mhd_bunch* b, int off, int n, int side) {
  b->ov_plist = b->d_plist + off;
  b->ov_dtlist = b->d_dtlist + off;
  b->ov_side = side;
  const int path = effective_path(b);
  int rc;
  if (path == MHD_PATH_ONEPASS) rc = OnePassLaunch<T>::run(b, b->d_dt + 1, 0, n, false);
  else if (path == MHD_PATH_TWO_KERNEL) rc = launch_fused_range<T>(b, 0, n);
  else if (path == MHD_PATH_TILE2D) rc = launch_tile2d<T>(b, 0, n);
  else rc = launch_staged_range<T>(b, 0, n);
  b->ov_plist = nullptr;
  b->ov_dtlist = nullptr;
  return rc;
}

}  // namespace

extern "C" {

int mhd_bunch_local_begin(mhd_bunch* b, double t0) {
  ENTER(b);
  NOT_RING(b);
  if (!isfinite(t0)) return MHD_EINVAL;
  int rc = materialise_guards(b);
  if (rc != MHD_OK) return rc;
  if (!b->loc) {
    b->loc = new (std::nothrow) mhd_bunch::Local();
    if (!b->loc) return MHD_ENOMEM;
  }
  // both slices = the current level
  CUDA_TRY(cudaMemcpyAsync(b->state[1 - b->cur], b->state[b->cur], b->lay.state_bytes, cudaMemcpyDeviceToDevice, b->stream));
  b->loc->active = true;
  b->loc->t_old.assign(b->G.np, t0);
  b->loc->t_new.assign(b->G.np, t0);
  b->loc->slot.assign(b->G.np, b->cur);
  b->rate_valid = false;
  b->closing_ok = false;
  return MHD_OK;
}

int mhd_bunch_local_state(mhd_bunch* b, double* t_old, double* t_new, int32_t* slot) {
  if (!b || !b->loc || !b->loc->active) return MHD_ESTATE;
  for (int p = 0; p < b->G.np; ++p) {
    if (t_old) t_old[p] = b->loc->t_old[p];
    if (t_new) t_new[p] = b->loc->t_new[p];
    if (slot) slot[p] = b->loc->slot[p];
  }
  return MHD_OK;
}

int mhd_bunch_step_local(mhd_bunch* b, const int32_t* patches, int32_t n, const double* dt) {
  ENTER(b);
  if (!b->loc || !b->loc->active) return MHD_ESTATE;
  if (!patches || !dt || n < 1 || n > b->G.np) return MHD_EINVAL;
  mhd_bunch::Local& L = *b->loc;
  const int np = b->G.np;
  const std::vector<int>& nb = *b->h_nbr;
  std::vector<char> seen(np, 0);
  for (int i = 0; i < n; ++i) {
    const int p = patches[i];
    if (p < 0 || p >= np || seen[p] || !(dt[i] > 0.0) || !isfinite(dt[i])) return MHD_EINVAL;
    seen[p] = 1;
  }
  // readiness: guard values are interpolated, never extrapolated (the rule under which DISPATCH
  // updates a task): t_old[q] <= t_new[p] <= t_new[q] for every neighbour q of a listed patch
  for (int i = 0; i < n; ++i) {
    const int p = patches[i];
    for (int c = 0; c < 27; ++c) {
      const int q = nb[(size_t)p * 27 + c];
      if (q < 0 || q == p) continue;
      const bool lo = L.t_old[q] <= L.t_new[p] || times_equal(L.t_old[q], L.t_new[p]);
      const bool hi = L.t_new[p] <= L.t_new[q] || times_equal(L.t_new[p], L.t_new[q]);
      if (!(lo && hi)) return MHD_ESTATE;
    }
  }
  // lists grouped by the buffer that holds the newer slice (one set of launches per group), with
  // the interpolation weights of every (listed patch, neighbour class)
  std::vector<int> plist;
  std::vector<double> dtl, wt;
  plist.reserve(n); dtl.reserve(n); wt.reserve((size_t)n * 27);
  int count[2] = {0, 0};
  for (int side = 0; side < 2; ++side)
    for (int i = 0; i < n; ++i) {
      const int p = patches[i];
      if (L.slot[p] != side) continue;
      ++count[side];
      plist.push_back(p);
      dtl.push_back(dt[i]);
      for (int c = 0; c < 27; ++c) {
        const int q = nb[(size_t)p * 27 + c];
        double w = 1.0;
        if (q >= 0 && !times_equal(L.t_new[p], L.t_new[q]) && !times_equal(L.t_new[q], L.t_old[q]))
          w = (L.t_new[p] - L.t_old[q]) / (L.t_new[q] - L.t_old[q]);
        wt.push_back(w);
      }
    }
  CUDA_TRY(cudaMemcpyAsync(b->d_slot, L.slot.data(), sizeof(int) * np, cudaMemcpyHostToDevice, b->stream));
  CUDA_TRY(cudaMemcpyAsync(b->d_plist, plist.data(), sizeof(int) * n, cudaMemcpyHostToDevice, b->stream));
  CUDA_TRY(cudaMemcpyAsync(b->d_dtlist, dtl.data(), sizeof(double) * n, cudaMemcpyHostToDevice, b->stream));
  CUDA_TRY(cudaMemcpyAsync(b->d_wtab, wt.data(), sizeof(double) * 27 * n, cudaMemcpyHostToDevice, b->stream));
  CUDA_TRY(cudaStreamSynchronize(b->stream));      // the host vectors go out of scope
  const bool f64 = b->desc.dtype == MHD_F64;
  {
    const FillMap M = make_fill_map(b->G);
    const long long tot = (long long)M.start[6] * n;
    if (tot > 0) {
      LaunchScope ls(b, KC_FILL);
      if (f64) k_fill_guards_local<double><<<blocks_for(tot, 256), 256, 0, b->stream>>>(b->G, M, (double*)b->state[0], (double*)b->state[1], b->d_nbr, b->d_slot, b->d_plist, b->d_wtab, n);
      else k_fill_guards_local<float><<<blocks_for(tot, 256), 256, 0, b->stream>>>(b->G, M, (float*)b->state[0], (float*)b->state[1], b->d_nbr, b->d_slot, b->d_plist, b->d_wtab, n);
    }
    CUDA_TRY(cudaGetLastError());
  }
  b->guards_stale = false;
  b->rate_valid = false;
  int off = 0;
  for (int side = 0; side < 2; ++side) {
    if (count[side] == 0) continue;
    const int rc = f64 ? launch_step_list<double>(b, off, count[side], side) : launch_step_list<float>(b, off, count[side], side);
    if (rc != MHD_OK) return rc;
    off += count[side];
  }
  for (int i = 0; i < n; ++i) {
    const int p = patches[i];
    L.slot[p] = 1 - L.slot[p];
    L.t_old[p] = L.t_new[p];
    L.t_new[p] += dt[i];
  }
  return MHD_OK;
}

int mhd_bunch_cfl_local(mhd_bunch* b, double courant, double* dt_patch) {
  ENTER(b);
  if (!b->loc || !b->loc->active) return MHD_ESTATE;
  if (!dt_patch || !(courant > 0.0) || !isfinite(courant)) return MHD_EINVAL;
  const int np = b->G.np;
  // one pass per buffer; a patch's step comes from the buffer that holds its newer slice
  std::vector<unsigned long long> r[2];
  const int cur = b->cur;
  for (int side = 0; side < 2; ++side) {
    b->cur = side;
    b->rate_valid = false;
    const int rc = b->desc.dtype == MHD_F64 ? launch_cfl<double>(b, courant, nullptr, nullptr) : launch_cfl<float>(b, courant, nullptr, nullptr);
    b->cur = cur;
    if (rc != MHD_OK) return rc;
    r[side].resize(np);
    CUDA_TRY(cudaMemcpyAsync(r[side].data(), b->d_rate, sizeof(unsigned long long) * np, cudaMemcpyDeviceToHost, b->stream));
    CUDA_TRY(cudaStreamSynchronize(b->stream));
  }
  for (int p = 0; p < np; ++p) {
    double rate;
    const unsigned long long bits = r[b->loc->slot[p]][p];
    memcpy(&rate, &bits, sizeof(rate));
    dt_patch[p] = courant / rate;
  }
  return MHD_OK;
}

int mhd_bunch_local_end(mhd_bunch* b) {
  ENTER(b);
  if (!b->loc || !b->loc->active) return MHD_ESTATE;
  mhd_bunch::Local& L = *b->loc;
  for (int p = 1; p < b->G.np; ++p)
    if (!times_equal(L.t_new[p], L.t_new[0])) return MHD_ESTATE;      // the bunch is not at one time
  // bring every newer slice into the current buffer: one launch over (patch, field), whatever the bunch size
  const size_t pb = (size_t)b->G.ps * b->esz, fb = (size_t)b->G.fs * b->esz;     // multiples of 16 bytes
  bool any = false;
  for (int p = 0; p < b->G.np && !any; ++p) any = L.slot[p] != b->cur;
  if (any) {
    CUDA_TRY(cudaMemcpyAsync(b->d_slot, L.slot.data(), sizeof(int) * b->G.np, cudaMemcpyHostToDevice, b->stream));
    const long long pv = (long long)(pb / 16);
    unsigned bx = blocks_for(pv, 256);
    if (bx > 64) bx = 64;
    LaunchScope ls(b, KC_MISC);
    k_gather_slices<<<dim3(bx, (unsigned)b->G.np, 8), 256, 0, b->stream>>>((uint4*)b->state[b->cur], (const uint4*)b->state[1 - b->cur],
                                                                          b->d_slot, b->cur, pv, (long long)(fb / 16));
    CUDA_TRY(cudaGetLastError());
  }
  L.active = false;
  b->guards_stale = false;
  b->closing_ok = false;
  b->rate_valid = false;
  return MHD_OK;
}

}  // extern "C"

extern "C" {

int mhd_bunch_destroy(mhd_bunch* b) {
  ENTER(b);
  cudaStreamSynchronize(b->stream);
  drain_events(b, false);
  hs_release(b);
  ring_release(b);
  delete b->loc;
  delete b->h_nbr;
  delete b->events;
  delete b;
  return MHD_OK;
}

}  // extern "C"

// ------------------------------------------------ CFL step without handle or workspace ----
// mhd_bunch_cfl_dt_static (include/mhd_bunch.h): for callers that have nowhere to get scratch from --
// a framework's task-update hook running while other streams are busy (cudaMalloc / cudaFree would
// serialise the device under them), an application whose pool already owns all of HBM, a module that is
// only handed a state pointer.  The per-patch rate maxima between k_cfl and k_cfl_final (what a handle
// keeps in b->d_rate, carved from the caller's workspace) sit in this array instead.  It is part of the
// library image: 8 * MHD_CFL_STATIC_MAX_PATCHES bytes (256 KiB) on every device that loads the library,
// until the process exits.
//
// In HOST code the name g_cfl_static_rate is only a handle for the runtime's symbol calls, not a device
// address: a kernel given `g_cfl_static_rate` from host code would fault (or scribble over host memory
// where the GPU can reach it).  The address a kernel may use comes from cudaGetSymbolAddress, asked for
// once per device with that device current, and is kept in g_cfl_static_ptr.
static __device__ __align__(256) unsigned long long g_cfl_static_rate[MHD_CFL_STATIC_MAX_PATCHES];

namespace {
constexpr int kStaticMaxDev = 64;
unsigned long long* g_cfl_static_ptr[kStaticMaxDev];   // device address of g_cfl_static_rate per ordinal (null: not asked yet)
std::mutex g_cfl_static_mu;

// Device address of the array on `device`, which must be the current device.  No allocation: the array
// came with the module; the lookup may make the runtime load the module, which is why the header asks for
// the first call on a device to come before any stream capture.
int cfl_static_address(int device, unsigned long long** out) {
  std::lock_guard<std::mutex> lock(g_cfl_static_mu);
  if (device < kStaticMaxDev && g_cfl_static_ptr[device]) { *out = g_cfl_static_ptr[device]; return MHD_OK; }
  void* p = nullptr;
  CUDA_TRY(cudaGetSymbolAddress(&p, g_cfl_static_rate));
  if (!p) return fail_cuda(cudaErrorInvalidSymbol, "cudaGetSymbolAddress(g_cfl_static_rate) returned null");
  if (device < kStaticMaxDev) g_cfl_static_ptr[device] = (unsigned long long*)p;   // ordinals past the table: looked up every call
  *out = (unsigned long long*)p;
  return MHD_OK;
}

template <typename T>
int launch_cfl_static(const mhd_bunch_desc* desc, const Geom& G, const void* state, unsigned long long* rate, double courant,
                      double* dt_dev, double* dt_patch) {
  cudaStream_t st = (cudaStream_t)desc->stream;
  Params<T> P;
  memset(&P, 0, sizeof(P));
  P.G = G;
  P.U = (const T*)state;
  P.npl = G.np;
  P.gamma = (T)desc->gamma;
  for (int a = 0; a < 3; ++a) {
    P.dx[a] = (T)desc->dx[a];
    P.idx[a] = (T)(1.0 / desc->dx[a]);
  }
  // the array still holds the previous call's maxima: the slots of this bunch start from zero
  k_zero_u64<<<blocks_for(G.np, 256), 256, 0, st>>>(rate, G.np);
  const long long per = (long long)G.n[0] * G.n[1] * G.n[2];
  int bx = (int)((per + 256 * CFL_CPT - 1) / (256 * CFL_CPT));   // launch shape of launch_cfl
  if (bx < 1) bx = 1;
  k_cfl<T><<<dim3((unsigned)bx, (unsigned)G.np), 256, 0, st>>>(P, rate);
  k_cfl_final<<<1, 256, 0, st>>>(rate, G.np, courant, dt_dev, nullptr, dt_patch);
  CUDA_TRY(cudaGetLastError());
  return MHD_OK;
}
}  // namespace

extern "C" int mhd_bunch_cfl_dt_static(const mhd_bunch_desc* desc, const void* state_dev, double courant, void* dt_dev,
                                       void* dt_per_patch_dev) {
  if (!desc || !state_dev || !dt_dev) return MHD_EINVAL;
  if (((uintptr_t)state_dev & 15) || ((uintptr_t)dt_dev & 7) || ((uintptr_t)dt_per_patch_dev & 7)) return MHD_EINVAL;
  if (!(courant > 0.0) || !isfinite(courant)) return MHD_EINVAL;
  Geom G;
  const int rc = build_geom(desc, &G);
  if (rc != MHD_OK) return rc;
  if (desc->npatch > MHD_CFL_STATIC_MAX_PATCHES) {
    snprintf(g_cuda_err, sizeof(g_cuda_err), "mhd_bunch_cfl_dt_static: %d patches, the built-in scratch holds %d (MHD_CFL_STATIC_MAX_PATCHES)",
             (int)desc->npatch, (int)MHD_CFL_STATIC_MAX_PATCHES);
    return MHD_ENOMEM;
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= desc->device || desc->device < 0)
    return fail_cuda(cudaErrorNoDevice, "no CUDA device: this library has no CPU fallback");
  CUDA_TRY(cudaSetDevice(desc->device));
  unsigned long long* rate = nullptr;
  const int ra = cfl_static_address(desc->device, &rate);
  if (ra != MHD_OK) return ra;
  return desc->dtype == MHD_F64
             ? launch_cfl_static<double>(desc, G, state_dev, rate, courant, (double*)dt_dev, (double*)dt_per_patch_dev)
             : launch_cfl_static<float>(desc, G, state_dev, rate, courant, (double*)dt_dev, (double*)dt_per_patch_dev);
}
