/* include/mhd_bunch.h -- C ABI of the B200-native bunch MHD update.
 *
 * One call advances a whole *bunch* -- many small Cartesian patches with guard zones
 * -- by one step of the MUSCL predictor + HLLD + HLLD-2D +
 * constrained-transport scheme of PAPER.md section 2.1 (L47-116).  The bunch stays
 * resident in HBM; there is no host<->device state traffic (the paper's largest cost,
 * L218, L243) and the number of kernel launches per step does not depend on the bunch
 * size (the launch overhead the paper attacks, L11, L178).
 *
 * Conventions
 *   - Every pointer argument says HOST or DEVICE.  Device memory (both state buffers and
 *     the workspace) is OWNED BY THE CALLER and borrowed for the lifetime of the handle.
 *   - State layout: structure of arrays  state[field][patch][k][j][i]  with the element
 *     strides and origin returned by mhd_bunch_query (x rows are padded so that interior
 *     cell 0 sits on a 16-byte boundary).  Indices (i,j,k) are guard-inclusive:
 *     0 <= i < m_x, m_d = n_d + 2*ng in an active dimension, m_d = 1 in a collapsed one
 *     (n_d == 1, "collapsed dimension").  Element (f,p,k,j,i) lives at
 *         origin + f*stride[0] + p*stride[1] + k*stride[2] + j*stride[3] + i*stride[4].
 *   - Field order is Eq. 6's: rho, rho*u, rho*v, rho*w, E, Bx, By, Bz.
 *     B components are LOWER-face values (Eq. 10-12); face n of a
 *     patch (the closing face) is stored in the first high-side guard slot.
 *   - All functions return MHD_OK (0) or a negative error code; they never throw or
 *     abort.  Unless stated otherwise a call only enqueues work on desc.stream.
 *   - No CPU fallback: without a CUDA device every compute call returns MHD_ECUDA.
 */
#ifndef MHD_BUNCH_H
#define MHD_BUNCH_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MHD_OK       0
#define MHD_EINVAL  -1   /* bad argument / unsupported configuration            */
#define MHD_ENOMEM  -2   /* workspace too small                                 */
#define MHD_ECUDA   -3   /* CUDA runtime error (mhd_bunch_last_cuda_error)      */
#define MHD_ESTATE  -4   /* call sequence error (e.g. destroyed handle)         */

#define MHD_F32 0
#define MHD_F64 1

typedef struct mhd_bunch mhd_bunch; /* opaque, owned by the library */

/* Statement of the problem (PAPER.md: patch dimensions and guard width L212, gamma L68,
 * bunch size L162).                                                                    */
typedef struct {
  int32_t n[3];        /* interior cells per patch (x,y,z); n[d]==1 => collapsed        */
  int32_t ng;          /* guard width in active dimensions; must be 3   */
  int32_t npatch;      /* bunch size                                                    */
  int32_t dtype;       /* MHD_F32 or MHD_F64: storage AND arithmetic type               */
  int32_t limiter;     /* 1 = minmod (default), 2 = monotonised central */
  int32_t emf_solver;  /* 0 = HLLD-2D (default), 1 = HLL-2D          */
  int32_t device;      /* CUDA ordinal                                                  */
  int32_t flux_solver; /* 0 = HLLD (default, PAPER.md 2.1.2), 1 = HLL (PAPER.md 2.1.1)  */
  double  gamma;       /* adiabatic index                                               */
  double  dx[3];       /* cell sizes, uniform over the bunch                            */
  void   *stream;      /* cudaStream_t supplied by the caller (0 = default stream)      */
} mhd_bunch_desc;

typedef struct {
  int64_t stride[5];       /* element strides of state[field][patch][k][j][i]           */
  int64_t origin;          /* elements from the buffer start to (0,0,0,0,0)             */
  int64_t state_elems;     /* elements per state buffer                                 */
  size_t  state_bytes;     /* bytes per state buffer (allocate two)                     */
  size_t  workspace_min;   /* bytes: smallest workspace mhd_bunch_create accepts        */
  size_t  workspace_best;  /* bytes: workspace that avoids sub-bunch chunking overhead  */
  int32_t m[3];            /* guard-inclusive extents                                   */
  int32_t reserved;
} mhd_bunch_layout;

/* HOST only.  Fills *layout for the given description.  MHD_EINVAL if the description is
 * not supported (ng != 3, an active dimension with n_d < ng, npatch < 1, ...).          */
int mhd_bunch_query(const mhd_bunch_desc *desc, mhd_bunch_layout *layout);

/* Creates a handle.
 *   nbr        HOST, int32 [npatch][27]; entry (oz+1)*9+(oy+1)*3+(ox+1) is the patch whose
 *              interior supplies the guard cells on that side, or -1 for zero-gradient
 *              outflow (the framework supplies neighbours).  Copied.
 *   state_a/b  DEVICE, state_bytes each, 16-byte aligned.  state_a holds time level n.
 *   workspace  DEVICE, workspace_bytes >= layout.workspace_min, 16-byte aligned.  Nothing
 *              is allocated or freed after create (static work arrays).
 * Synchronises desc.stream once (table upload).
 * The fast routes that read halos through the table (deferred fill, below) are taken only if
 * the table has no -1 entry and composes like translations: nbr[p][centre] = p and
 * nbr[nbr[p][c1]][c2] = nbr[p][c1+c2] wherever c1+c2 is again one of the 27 classes (true for
 * any periodic arrangement of patches).  Any other table is still handled correctly, by an
 * explicit guard fill before every step.  Every later call runs on desc.device, whatever the
 * caller's current device is.                                                            */
int mhd_bunch_create(const mhd_bunch_desc *desc, const int32_t *nbr, void *state_a, void *state_b,
                     void *workspace, size_t workspace_bytes, mhd_bunch **out);

/* Guard fill of the current level: same-time, same-resolution copy of neighbour
 * interiors into the 3-deep guard shell, edges and corners included; -1 neighbours give
 * zero-gradient values and leave the closing face untouched (
 * DESIGN.md O1).  Must precede mhd_bunch_step and mhd_bunch_cfl_dt.
 *
 * Deferred fill.  When the next step will run the one-pass kernel on a bunch all of whose
 * neighbours exist, that kernel reads every halo straight from the neighbours' interiors,
 * so this call only brings the closing faces up to date (if the caller may have written
 * the buffer since the last fill) and marks the rest of the guard shell as owed.  The shell is written to HBM the moment anything reads it from there:
 * mhd_bunch_current, mhd_bunch_download, mhd_bunch_sync_guards, mhd_bunch_set_path or a
 * step by another path.  A caller that looks at guard cells of its own buffer must
 * therefore go through one of those calls first (the Python binding always does).  What
 * every entry point returns is identical to an immediate fill.                         */
int mhd_bunch_fill_guards(mhd_bunch *b);

/* Writes a deferred guard fill of the current level to HBM now (no-op if none is owed).  */
int mhd_bunch_sync_guards(mhd_bunch *b);

/* CFL time step of the current level: courant / max over interior cells of
 * sum_d (|u_d| + c_fast,d)/dx_d over active d (O9).
 *   dt_host          HOST, nullable.  If given, the stream is synchronised and *dt_host set.
 *   dt_dev           DEVICE double*, nullable: receives dt without any synchronisation.
 *   dt_per_patch_dev DEVICE double[npatch], nullable: per-patch steps.  */
int mhd_bunch_cfl_dt(mhd_bunch *b, double courant, double *dt_host, void *dt_dev, void *dt_per_patch_dev);

/* One step: current level n -> other buffer (interior cells and closing faces), which
 * becomes the current level.  Guards of the new level are stale until the next
 * mhd_bunch_fill_guards.  dt <= 0 or non-finite -> MHD_EINVAL.                         */
int mhd_bunch_step(mhd_bunch *b, double dt);

/* Same, with dt read on the device (DEVICE const double*), optionally clipped to
 * dt_max > 0 (pass 0 for no clip): no host round trip between cfl_dt and step.          */
int mhd_bunch_step_dev(mhd_bunch *b, const void *dt_dev, double dt_max);

/* Host-buffer path (the paper's per-bunch offload): copy a whole
 * state buffer between HOST memory (same layout as the device buffer, state_bytes long;
 * pinned memory makes the copy asynchronous) and the current level.  Enqueued on the
 * stream; mhd_bunch_download synchronises the stream before returning.                   */
int mhd_bunch_upload(mhd_bunch *b, const void *host_state);
int mhd_bunch_download(mhd_bunch *b, void *host_state);

/* Host-streaming path (bunches handed to the GPU
 * round-robin with several in flight; L243-247: asynchronous host<->device staging).  The
 * bunch lives in HOST memory in the COMPACT layout  host[field][patch][k][j][i]  (interior
 * cells only, n_z*n_y*n_x per patch and field, fields in Eq. 6's order; B components on the
 * lower faces; host_bytes long; pinned memory lets the copies run asynchronously).  One
 * call advances it by one step: pieces of chunks of patches cross PCIe on library-owned copy
 * streams (through two staging buffers per direction, so the link never waits for a kernel),
 * are scattered into the padded HBM layout, stepped chunk by chunk as soon as what their
 * neighbours must provide has arrived (the neighbour table decides), gathered and copied
 * back -- so uploads, kernels and downloads overlap.  Guard zones never cross PCIe.  A chunk
 * needs the chunks of its in-plane neighbours whole, but of a chunk it reaches only through
 * o_z = +1 (-1) just the lowest (highest) guard-width planes: those thin layers are uploaded
 * ahead of the rest, so a chunk never waits for the bulk of its z-neighbours (and the first
 * chunk of a periodic stack not for the last one).
 *
 *   mhd_bunch_host_query   HOST out *layout for a chunk size (<= 0: library default):
 *                          host_bytes, the staging size, the number of chunks, and whether
 *                          the fully overlapped schedule applies (one-pass path with every
 *                          neighbour present); otherwise uploads, a whole-bunch step and
 *                          downloads run back to back, still through the same chunks.
 *   mhd_bunch_host_attach  staging_dev: DEVICE, caller-owned, >= staging_bytes, 16-byte
 *                          aligned, borrowed until detach/destroy.  MHD_EINVAL for bunches
 *                          with outflow (-1) neighbours: their evolved closing faces have
 *                          no slot in the compact layout.  Creates the streams and events.
 *   mhd_bunch_step_host    host_in: HOST const, time level n; host_out: HOST, receives level
 *                          n+1 (may equal host_in only if dt == 0 or the schedule is not
 *                          overlapped -- keep them distinct).  dt > 0: step with this dt
 *                          (uploads and steps overlap); dt == 0: the step is the CFL step
 *                          courant/max rate of level n, which needs every chunk on the
 *                          device first.  HOST out, nullable: *dt_used, and *dt_next =
 *                          the CFL step of level n+1 (so the next call can pass dt > 0).
 *                          Synchronises: on return host_out is complete.  The device keeps
 *                          level n+1 as the current level.
 */
typedef struct {
  size_t  host_bytes;      /* bytes of a compact host state                                */
  size_t  staging_bytes;   /* bytes of device staging mhd_bunch_host_attach needs          */
  int32_t chunk_patches;   /* patches per chunk                                            */
  int32_t nchunk;          /* chunks per bunch                                             */
  int32_t pipelined;       /* 1: uploads, steps and downloads overlap chunk by chunk       */
  int32_t bands;           /* z-bands the first chunk and the last two are stepped in      */
} mhd_bunch_host_layout;
int mhd_bunch_host_query(mhd_bunch *b, int32_t chunk_patches, mhd_bunch_host_layout *layout);
int mhd_bunch_host_attach(mhd_bunch *b, void *staging_dev, size_t staging_bytes, int32_t chunk_patches);
int mhd_bunch_step_host(mhd_bunch *b, const void *host_in, void *host_out, double dt, double courant,
                        double *dt_used, double *dt_next);
int mhd_bunch_host_detach(mhd_bunch *b);

/* HOST only, no device needed: the schedule mhd_bunch_step_host would follow for a neighbour
 * table (HOST int32 [npatch][27]), patches of nz planes, a guard width, a chunk size and a number
 * of bands (each <= 0: the library's choice, the candidate with the shortest simulated makespan).
 * STEP UNITS are stepped in order: chunks 0 .. nchunk-1, the first chunk and the last two in
 * `bands` bands of planes each (so that downloads start early and the step ends with the download
 * of two bands, not of two chunks), the others whole.  Outputs (HOST; the arrays nullable, capacity `cap` >= *npiece
 * and >= *nunit else MHD_ENOMEM): upload piece i carries planes [piece_k0[i], piece_k1[i]) of
 * every patch of chunk piece_chunk[i]; the pieces of a chunk partition its planes (every plane
 * crosses PCIe once); unit u = planes [unit_za[u], unit_zb[u]) of chunk unit_chunk[u]; ready[u] =
 * index of the last piece unit u needs before it may step (planes [za-guard, zb+guard) of itself
 * and of its in-plane neighbours' chunks; the lowest planes of chunks reached through o_z = +1 if
 * the range passes nz, the highest of those reached through o_z = -1 if it passes 0; everything
 * whole if nz < 2 guard + 1 or nz > 64); *makespan = simulated length of the step in units of
 * "one patch across PCIe" (a step costs 0.33 per patch; fixed costs: 2.0 per upload piece, 0.5
 * per step, 0.7 per download -- measured on a B200 / PCIe 5 box).                               */
int mhd_bunch_host_schedule(const int32_t *nbr, int32_t npatch, int32_t nz, int32_t guard, int32_t chunk_patches, int32_t bands,
                            int32_t *chunk_out, int32_t *bands_out, int32_t *npiece_out, int32_t *piece_chunk,
                            int32_t *piece_k0, int32_t *piece_k1, int32_t *nunit_out, int32_t *unit_chunk, int32_t *unit_za,
                            int32_t *unit_zb, int32_t *ready, int32_t cap, double *makespan);

/* Ring mode: a host-resident bunch LARGER than the device buffers (PAPER.md
 * L164: bunches filled round-robin with several in flight; L243-247: asynchronous staging).  The
 * handle is created for a WINDOW of patches (its npatch, its two state buffers); the bunch itself --
 * `npatch` patches with their own neighbour table, compact host layout as for mhd_bunch_step_host --
 * streams through the window in chunks of `chunk_patches` consecutive patches: the window holds
 * R = (handle npatch) / chunk_patches chunk slots.  Chunks are stepped in order; before a chunk is
 * stepped every chunk that holds one of its neighbours is resident in some slot (the kernels read
 * halos through a neighbour table rewritten in slot numbers), a chunk nobody needs any more gives up
 * its slot to the next upload, and results leave through the second buffer's slots -- uploads,
 * kernels and downloads overlap as in mhd_bunch_step_host.  Chunks that are needed again after they
 * were evicted (the first ones of a periodic bunch) are uploaded twice.
 *
 *   mhd_bunch_ring_plan    HOST only: the schedule for a table, a chunk size and R slots: number of
 *                          chunks, number of uploads, and (nullable, capacity `cap`) per upload the
 *                          chunk, its slot and the step it precedes, per step the slot of the chunk
 *                          stepped.  MHD_ENOMEM if some chunk's neighbourhood does not fit in R slots.
 *   mhd_bunch_ring_attach  nbr: HOST int32[npatch][27], no -1 entries, translation-consistent (see
 *                          mhd_bunch_create); staging_dev: DEVICE, caller-owned, 16-byte aligned,
 *                          >= 2 * 8 * chunk_patches * n_x n_y n_z * sizeof(real) bytes.  Needs the
 *                          one-pass step (float32, three active dimensions, n_x a multiple of 4):
 *                          MHD_EINVAL otherwise.
 *   mhd_bunch_step_ring    host_in / host_out: HOST (pinned for overlap), distinct, compact layout
 *                          of the WHOLE bunch; dt > 0; HOST out, nullable: *dt_next = CFL step of the
 *                          new level (from the step's own epilogue).  Synchronises.  Results are bit
 *                          for bit those of the resident step.
 *   mhd_bunch_ring_detach  releases the streams; the handle is a plain window-sized bunch again.
 * While a ring is attached the device copy of the neighbour table belongs to it, so the calls that
 * would read it as the window's own table -- mhd_bunch_fill_guards, sync_guards, cfl_dt, step, step_dev,
 * host_attach, step_host, local_begin -- return MHD_ESTATE until mhd_bunch_ring_detach; ring_attach
 * ends an attached host-streaming mode itself, and neither ring call is accepted in local-time-step
 * mode.                                                                                           */
int mhd_bunch_ring_plan(const int32_t *nbr, int32_t npatch, int32_t chunk_patches, int32_t ring_chunks, int32_t *nchunk,
                        int32_t *nupload, int32_t *up_chunk, int32_t *up_slot, int32_t *up_step, int32_t *step_slot, int32_t cap);
int mhd_bunch_ring_attach(mhd_bunch *b, const int32_t *nbr, int32_t npatch, int32_t chunk_patches, void *staging_dev,
                          size_t staging_bytes);
int mhd_bunch_step_ring(mhd_bunch *b, const void *host_in, void *host_out, double dt, double courant, double *dt_next);
int mhd_bunch_ring_detach(mhd_bunch *b);

/* Local time steps (a patch holds several time slices, its
 * own time and its own time step; L188, L200: ghost zones of neighbours that sit at other times are
 * interpolated).  The two state buffers become two TIME SLICES per patch: slot[p] says which buffer
 * holds the newer slice of patch p (time t_new[p]), the other one holds the older (t_old[p]).
 *
 *   mhd_bunch_local_begin  both slices of every patch := the current level, all times = t0.
 *   mhd_bunch_step_local   patches: HOST int32[n], distinct; dt: HOST double[n], > 0.  For every
 *                          listed patch p: the guard shell of its newer slice is filled from its
 *                          neighbours' slices LINEARLY INTERPOLATED IN TIME to t_new[p]
 *                          (v_old + w (v_new - v_old), w = (t_new[p] - t_old[q]) / (t_new[q] - t_old[q]);
 *                          a neighbour at the patch's own time contributes its newer slice bit for
 *                          bit; -1 neighbours: zero gradient as in mhd_bunch_fill_guards), then the
 *                          patch is advanced by its own dt into its older slice, which becomes the
 *                          newer one.  The number of launches does not depend on the list's size: one
 *                          guard fill, then one set of step launches per buffer that holds newer slices
 *                          of listed patches (so up to two sets).  Synchronises the stream once (the
 *                          lists are staged through pageable memory).
 *                          MHD_ESTATE unless every neighbour q of every listed p satisfies
 *                          t_old[q] <= t_new[p] <= t_new[q] (values are interpolated, never
 *                          extrapolated -- the rule under which DISPATCH updates a task); nothing is
 *                          changed then.  With one dt and every patch listed this is the global
 *                          step, bit for bit.  Totals are not conserved across patches that step
 *                          with different dt (the paper describes no flux correction).
 *   mhd_bunch_cfl_local    HOST out double[npatch]: the CFL step of each patch's newer slice;
 *                          synchronises.
 *   mhd_bunch_local_state  HOST out (each nullable) t_old, t_new: double[npatch]; slot: int32[npatch]
 *                          (0: state_a, 1: state_b holds the newer slice).
 *   mhd_bunch_local_end    all patches must be at one time (else MHD_ESTATE): their newer slices are
 *                          gathered into the current level and the handle is back in global mode.  */
int mhd_bunch_local_begin(mhd_bunch *b, double t0);
int mhd_bunch_step_local(mhd_bunch *b, const int32_t *patches, int32_t n, const double *dt);
int mhd_bunch_cfl_local(mhd_bunch *b, double courant, double *dt_patch);
int mhd_bunch_local_state(mhd_bunch *b, double *t_old, double *t_new, int32_t *slot);
int mhd_bunch_local_end(mhd_bunch *b);

/* HOST out: which of state_a/state_b holds the current level.  This is the call through
 * which a caller gets at the state between library calls: a deferred guard fill is written
 * out first, and the library assumes the caller may then modify the buffer (so the next
 * mhd_bunch_fill_guards re-reads the closing faces).  Do not read or write the buffers
 * behind the library's back without it (or mhd_bunch_upload / mhd_bunch_download).       */
int mhd_bunch_current(mhd_bunch *b, void **state);

/* Synchronises.  *bad_cells = number of interior cells met so far whose density or
 * pressure was not positive and finite (the scheme has no floors: DESIGN.md Q19).       */
int mhd_bunch_status(mhd_bunch *b, int64_t *bad_cells);

/* The step has four CUDA implementations, all on the GPU:
 *   MHD_PATH_ONEPASS     the whole step in one kernel, nothing intermediate in HBM (three
 *                        active dimensions, float32): the default where it applies;
 *   MHD_PATH_TILE2D      the whole step of a two-dimensional bunch (n_z = 1, x and y active) or of
 *                        a one-dimensional one along x (n_y = n_z = 1) in one kernel on
 *                        shared-memory tiles / rows, any type: the default there (the
 *                        staged path's stage functions on a tile: same result to rounding);
 *   MHD_PATH_TWO_KERNEL  predictor kernel + Riemann/update kernel with one scratch block in
 *                        HBM (three active dimensions, any type);
 *   MHD_PATH_STAGED      one kernel per stage of PAPER.md section 2.1.4 (general: collapsed
 *                        dimensions, cross-checks).
 * MHD_PATH_AUTO picks the first one that applies.  Asking for a path that does not apply to
 * this bunch returns MHD_EINVAL.  mhd_bunch_get_path reports the one a step would run.    */
#define MHD_PATH_AUTO        0
#define MHD_PATH_STAGED      1
#define MHD_PATH_TWO_KERNEL  2
#define MHD_PATH_ONEPASS     3
#define MHD_PATH_TILE2D      4
int mhd_bunch_set_path(mhd_bunch *b, int32_t path);
int mhd_bunch_get_path(mhd_bunch *b, int32_t *path);

int mhd_bunch_destroy(mhd_bunch *b);

/* CFL time step WITHOUT a handle and WITHOUT a workspace (same quantity as mhd_bunch_cfl_dt:
 * PAPER.md L122; O9).
 *
 * Who this is for.  Everything above needs device memory from the caller: a workspace handed
 * to mhd_bunch_create, which somebody had to cudaMalloc.  Some callers cannot do that at the
 * point where they need a time step:
 *   - a task-update hook of a host framework (DISPATCH updates a patch from inside a worker
 *     thread) that runs while other streams are busy: cudaMalloc and
 *     cudaFree serialise the whole device, so one allocation there stalls every bunch in flight;
 *   - an application that gave all of HBM to its own pool at start-up, where a late cudaMalloc
 *     simply fails, and whose pool is not reachable from the place the call is made;
 *   - code that is only handed a state pointer (a diagnostics or restart module checking the
 *     time step of a dump it mapped) and owns no handle and no scratch at all.
 * For them the per-patch rate maxima that the two-stage reduction needs between its kernels live
 * in an array that is PART OF THE LIBRARY IMAGE: MHD_CFL_STATIC_MAX_PATCHES 8-byte slots
 * (256 KiB), present on every GPU that loads libmhd_bunch.so, from load until the process ends,
 * whether or not this call is ever made.  The call makes no cudaMalloc / cudaFree and uses no
 * allocating library routine; it launches the same three kernels as mhd_bunch_cfl_dt and the
 * results are the same bits.
 *
 *   desc             HOST.  n, ng, npatch, dtype, gamma, dx, device and stream are read (limiter
 *                    and solver choices must be valid but play no part).
 *                    npatch > MHD_CFL_STATIC_MAX_PATCHES -> MHD_ENOMEM, nothing is launched
 *                    (mhd_bunch_last_cuda_error then says what the limit is).
 *   state_dev        DEVICE const, the layout mhd_bunch_query returns for desc, 16-byte aligned,
 *                    with the closing faces up to date (after mhd_bunch_fill_guards, or straight
 *                    after a step: a rate reads the upper face of a cell).  Not modified.
 *   dt_dev           DEVICE double*, required: receives courant / (largest rate of the bunch).
 *   dt_per_patch_dev DEVICE double[npatch], nullable: per-patch steps.
 * Only enqueues on desc.stream; read the outputs after synchronising it yourself.
 *
 * First call on a device.  The first call for a given desc.device looks up the device address
 * of the array (with that device current) and remembers it; that lookup may load the library's
 * device code.  Make this first call early, outside any stream capture; later calls on that
 * device only launch kernels.
 *
 * Sharing.  Every call on a device uses the SAME array, whatever its stream, thread or bunch,
 * and the array keeps what the previous call left there: each call clears the slots it is going
 * to use before reducing into them, but two calls whose kernels can overlap on the GPU (different
 * streams without an ordering event between them) overwrite each other's maxima and both results
 * are then garbage.  Order such calls yourself, or use handles (mhd_bunch_cfl_dt), whose
 * scratch is private.                                                                        */
#define MHD_CFL_STATIC_MAX_PATCHES 32768
int mhd_bunch_cfl_dt_static(const mhd_bunch_desc *desc, const void *state_dev, double courant, void *dt_dev,
                            void *dt_per_patch_dev);

const char *mhd_bunch_strerror(int code);
const char *mhd_bunch_last_cuda_error(void);

/* ------------------------------------------------------------------------------------------
 * Diagnostics and tuning -- NOT part of the method.  A caller of the paper's problem statement
 * (create / fill_guards / cfl_dt / step and the host, ring and local variants above) never needs
 * these six calls; bench.py and the tests use them to time kernel classes, count launches, force
 * launch shapes and measure the ALU peak the roofline is quoted against.
 * ------------------------------------------------------------------------------------------ */

/* Per-kernel-class device timing for roofline reports.  While enabled, every launch is
 * bracketed by CUDA events on the stream (a few microseconds of overhead per launch, so
 * leave it off in throughput runs).  mhd_bunch_kernel_times synchronises, fills up to
 * `cap` entries (name: HOST const char* owned by the library; ms: total device time;
 * count: launches) accumulated since timing was enabled, and returns the number of
 * classes through *n.                                                                    */
int mhd_bunch_set_timing(mhd_bunch *b, int32_t enable);
int mhd_bunch_kernel_times(mhd_bunch *b, int32_t cap, const char **names, double *ms, int64_t *count, int32_t *n);

/* Number of kernel launches issued so far through this handle (for bench.py).           */
int mhd_bunch_launch_count(mhd_bunch *b, int64_t *launches);

/* Launch-shape knobs (tests and tuning runs; the library reads no environment variables).
 *   MHD_TUNE_ONEPASS_ZSEG  z segments per tile column of the one-pass kernel (0 = automatic:
 *                          1 unless the bunch has fewer tiles than the device has SMs);
 *                          results do not depend on it, bit for bit.
 *   MHD_TUNE_PREDICT_TY    y-tile of the two-kernel path's predictor: 16, 8 or 4.
 *   MHD_TUNE_FUSED_CFL     1: the one-pass step also reduces the CFL rates of the level it writes
 *                          (in its epilogue, from registers), so that the next mhd_bunch_cfl_dt
 *                          only runs the bunch-wide reduction instead of re-reading the state
 *                          (three launches per step instead of five); 0: mhd_bunch_cfl_dt always
 *                          makes its own pass; 2 (default): the library chooses -- the epilogue
 *                          on bunches of at most one wave of tiles, which are bound by launch
 *                          latency, the pass on larger ones, where it is cheaper.  Same dt, bit
 *                          for bit, either way (both evaluate one explicitly rounded function);
 *                          the stepped state of the two kernel variants agrees to rounding.
 *   MHD_TUNE_HOST_BANDS    z-bands in which mhd_bunch_step_host steps the first chunk and the last
 *                          two (0 = automatic; clipped to bands of at least eight planes; only
 *                          the one-pass path steps plane ranges).  Read by host_query / attach;
 *                          results do not depend on it, bit for bit.
 *   MHD_TUNE_HOST_MAX_PITCH  largest host pitch in bytes that one strided host<->device copy of
 *                          mhd_bunch_step_host / mhd_bunch_step_ring may name (0 = the device's
 *                          cudaDevAttrMaxPitch, 2^31 - 1).  Host bunches whose fields are further
 *                          apart than this are moved field by field (eight copies per transfer
 *                          instead of one); tests set it to 1 to run that route on small bunches.
 *                          Results do not depend on it, bit for bit.
 * MHD_EINVAL for an unknown key or a value the bunch cannot run.                           */
#define MHD_TUNE_HOST_MAX_PITCH 5
#define MHD_TUNE_HOST_BANDS   4
#define MHD_TUNE_ONEPASS_ZSEG 1
#define MHD_TUNE_PREDICT_TY   2
#define MHD_TUNE_FUSED_CFL    3
int mhd_bunch_set_tuning(mhd_bunch *b, int32_t key, int32_t value);

/* Measures the plain-ALU peak of the device with an FMA-chain microbenchmark (FMA counted
 * as 2 flops), for the roofline bench.py reports: HOST out *tflops.  Synchronous.
 *   scratch_dev  DEVICE, caller-owned, >= 8 * 256 * 8 * (number of SMs) bytes (4 MiB is
 *                always enough; MHD_ENOMEM otherwise): the library allocates nothing.     */
int mhd_bunch_measure_alu_peak(int32_t dtype, int32_t device, void *scratch_dev, size_t scratch_bytes, double *tflops);

/* Names and device times are not part of the ABI; this reports the sub-bunch chunk (in
 * patches) the workspace allows.                                                        */
int mhd_bunch_chunk(mhd_bunch *b, int32_t *chunk_patches);

#ifdef __cplusplus
}
#endif
#endif /* MHD_BUNCH_H */
