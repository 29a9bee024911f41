/* oracle/mhd_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded CPU statement of the per-bunch ideal-MHD update of
 * arxiv 2508.09568 (PAPER.md sections 2.1.1-2.1.4, L47-116; L154; L212), written
 * stage by stage in the paper's order.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code
 * with paper_2508_09568_b200/ (the CUDA path) and neither imports the other.
 *
 * `real` is double unless the file is compiled with -DORACLE_REAL=float (diagnostic).
 *
 * Layout (dense): U[field][patch][k][j][i] with guard-inclusive extents
 * m_d = n_d + 2*ng in an active dimension, m_d = 1 in a collapsed one (n_d == 1).
 * Field order is Eq. 6's: rho, rho*u, rho*v, rho*w, E, Bx, By, Bz.
 * Bx(i,j,k) is the value on the cell's LOWER x-face (Eq. 10-12).
 *
 * Parity status: every function is pinned in tests/test_oracle_*.py EXCEPT the
 * match of orc_emf2d (HLLD-2D) to the RAMSES routine the paper copied, whose
 * formulas the paper does not print: "parity unpinned" for that match.  What IS
 * pinned for orc_emf2d: planar reduction to orc_hlld's induction flux, uniform
 * state, x<->y antisymmetry, supersonic upwinding, the upwind weighting of the
 * edge-side star fields (step 5: one-way supersonic flow reduces the edge to the
 * upwind row's / column's 1D problem) and a second typing of the whole reading
 * (see DESIGN.md).  tests/test_oracle_mutations.py compiles deliberately broken
 * copies of this file and requires every one of them to fail a pin.
 *
 * The `#pragma omp parallel for` lines over patches are inert in the builds the
 * tests use; oracle/build.py's build_omp() (-fopenmp) activates them for bench.py's
 * all-cores timing leg.  Patches are independent between guard fills (PAPER.md
 * L124), so the arithmetic is the same (checked bit for bit in the tests).
 */
#ifndef MHD_ORACLE_H
#define MHD_ORACLE_H
#include <stdint.h>

#ifndef ORACLE_REAL
#define ORACLE_REAL double
#endif
typedef ORACLE_REAL real;

typedef struct {
  int32_t n[3];       /* interior cells per patch (x,y,z); n[d]==1 => collapsed        */
  int32_t ng;         /* guard width in active dimensions (paper: 3)     */
  int32_t npatch;     /* bunch size                                      */
  int32_t limiter;    /* 1 = minmod, 2 = monotonised central                             */
  int32_t emf_solver; /* 0 = HLLD-2D, 1 = HLL-2D                                         */
  int32_t flux_solver;/* 0 = HLLD (PAPER.md 2.1.2), 1 = HLL (PAPER.md 2.1.1)            */
  double gamma;       /* adiabatic index                                  */
  double dx[3];       /* cell sizes                                                      */
} orc_desc;

/* number of per-patch scratch arrays exported by orc_stages, in this order:
 *  q[8], dq[3][8], dbf[6], e0[3], bh[3], qh[8], flux[3][5], emf[3]                     */
#define ORC_NSTAGE 70

int     orc_sizeof_real(void);
/* OpenMP build only (-fopenmp, bench.py's all-cores leg): set (want > 0) and return the number
 * of threads the per-patch loops use; the plain build returns 1.                              */
int     orc_threads(int want);
int64_t orc_patch_cells(const orc_desc *d);              /* m_x*m_y*m_z                 */
int64_t orc_state_elems(const orc_desc *d);              /* 8*npatch*patch_cells        */

/* O1  guard fill (width L212).  nbr[npatch][27], class index
 *     (oz+1)*9+(oy+1)*3+(ox+1), value = source patch or -1 (zero-gradient outflow).    */
void orc_fill_guards(const orc_desc *d, const int32_t *nbr, real *U);

/* O9  CFL step: courant / max_cells sum_d (|u_d|+c_f,d)/dx_d.
 *     per_patch (nullable) receives npatch per-patch values.                            */
double orc_cfl_dt(const orc_desc *d, const real *U, double courant, double *per_patch);

/* O2-O8  one MUSCL / HLLD / HLLD-2D / CT step of the whole bunch.
 *     Guards of U must be filled.  Unew receives a copy of U with the interior cells
 *     and the closing faces advanced; its other guard cells are stale.                  */
void orc_step(const orc_desc *d, const real *U, real *Unew, double dt);

/* the same stages for one patch, exporting every scratch array: out[ORC_NSTAGE][M]     */
void orc_stages(const orc_desc *d, const real *U, int32_t patch, double dt, real *out);

/* O10  local time steps with time-interpolated guard fill (patches hold several
 *     time slices, their own time and time step; L188, L200: ghost zones of neighbours at other
 *     times are interpolated).  S0, S1: two full bunch arrays; cur[p] = which of them holds the
 *     newer slice of patch p (time t_new[p]); the other holds the older one (t_old[p]).
 *     orc_step_local advances list[0..n) by dt[0..n): guard fill of each listed patch's newer
 *     slice from its neighbours' slices, linearly interpolated in time to t_new[p]
 *     (v_old + w (v_new - v_old), w = (t_new[p]-t_old[q])/(t_new[q]-t_old[q]); equal times: the newer
 *     slice itself, bit for bit), then O2-O8 into the older slice, which becomes the newer one.
 *     Returns -1 and changes nothing unless every neighbour q of every listed p has
 *     t_old[q] <= t_new[p] <= t_new[q] (orc_local_ready).  Mass, momentum and energy are NOT
 *     conserved across patches that step with different dt (no flux correction in the paper).   */
int  orc_local_ready(const orc_desc *d, const int32_t *nbr, const double *t_old, const double *t_new,
                     const int32_t *list, int32_t n);
void orc_fill_guards_local(const orc_desc *d, const int32_t *nbr, real *S0, real *S1, const int32_t *cur,
                           const double *t_old, const double *t_new, int32_t p);
int  orc_step_local(const orc_desc *d, const int32_t *nbr, real *S0, real *S1, int32_t *cur, double *t_old,
                    double *t_new, const int32_t *list, int32_t n, const double *dt);

/* pointwise pieces, exported for the pins */
real orc_limiter(int32_t kind, real a, real b);                               /* O3 */
void orc_hlld(double gamma, const real L[7], const real R[7], real bn, real F[7]); /* O6 */
void orc_hll(double gamma, const real L[7], const real R[7], real bn, real F[7]);  /* PAPER.md 2.1.1 */
/* O7: corner c = 0:SW 1:SE 2:NW 3:NE, each (rho, ua, ub, ue, p, Be);
 *     A = in-plane field along a (south, north), B = in-plane field along b (west, east) */
real orc_emf2d(double gamma, int32_t solver, const real c[4][6],
               real AS, real AN, real BW, real BE);
real orc_fast_speed(double gamma, real rho, real p, real bn, real bt1, real bt2);

#endif
