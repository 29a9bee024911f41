"""Helpers shared by the GPU parity tests: the error metric of DESIGN.md (Q21) and
drivers that run the same seeded workload through the oracle and through the C ABI."""
import numpy as np

import oracle
from paper_2508_09568_b200 import workloads as W

GROUPS = [(0, 1), (1, 4), (4, 5), (5, 8)]      # rho; momentum; E; B

TOL_STEP = {"f64": 1e-12, "f32": 2e-5}         # BASELINE.json north_star: per-cell relative error after one step
TOL_TOTALS_F64 = 1e-12                         # conserved totals after N steps
TOL_L1_F32 = 1e-4                              # L1 field norms after N steps
# Regression bounds, a decade above what the kernels are observed to do (Q21):
# the north_star tolerances leave two to four orders of headroom, these do not.
TIGHT_STEP = {"f64": 2e-14, "f32": 2e-6}
# Secondary metric of Q21: PURE relative error |g-o|/|o|, per component, over cells with
# |o| > PURE_FLOOR * s_f, held to the same north_star tolerance.  (In fp32 the update U - dt*dF/dx
# of a small component cancels fluxes of the group's magnitude, so this is the tighter of the two
# statements there: observed 1.2e-5 at worst against 1.4e-7 for the scale-relative metric.)
PURE_FLOOR = 1e-3
TOL_PURE = {"f64": 1e-12, "f32": 2e-5}


def rel_err(g, o):
    """Q21, primary: max over cells of |g-o| / max(|o|, s_f), s_f = max|o| of the field group
    (rho; momentum; E; B) over the bunch, 1 if the group is identically zero.  Since |o| <= s_f this
    is the maximum-norm error of the group in units of its scale; the per-cell statement proper is
    rel_err_pure."""
    worst = 0.0
    for a, b in GROUPS:
        s = np.abs(o[a:b]).max()
        s = s if s > 0 else 1.0
        e = np.abs(g[a:b].astype(np.float64) - o[a:b]) / np.maximum(np.abs(o[a:b]), s)
        worst = max(worst, float(e.max()))
    return worst


def rel_err_pure(g, o, floor=PURE_FLOOR):
    """Q21, secondary: max over components f and cells with |o_f| > floor * s_f of |g_f-o_f|/|o_f|
    (s_f = max|o| of the component's field group).  A cell at a thousandth of the scale that is
    wrong by a percent fails this, which the primary metric alone would not notice."""
    worst = 0.0
    for a, b in GROUPS:
        s = np.abs(o[a:b]).max()
        if not s > 0:
            continue
        for f in range(a, b):
            of = o[f]
            m = np.abs(of) > floor * s
            if m.any():
                e = np.abs(g[f].astype(np.float64)[m] - of[m]) / np.abs(of[m])
                worst = max(worst, float(e.max()))
    return worst


# Where the secondary metric can be asserted, and with which floor (Q21; measured in round 3).
# Its worst cell always sits just above the floor, in a transverse field component that nearly cancels (By, Bz of the
# turbulence field at 1.0-1.4e-3 of the group scale): the absolute error there is the fp32 rounding of the update's
# terms, 1-4e-8 of the SCALE, so the metric is (1-4e-8) / floor and grows with the number of cells over which the
# maximum is taken and with the steps taken: 1.0e-5 (8 x 16^3 or 8 x 32^3, one step), 2.1e-5 (8 x 64^3, one step),
# 3.6e-5 (8 x 32^3, three steps).  With the floor 1e-3 it is held to 2e-5 on the small one-step cases only
# (assert_step_parity); full-size bunches and multi-step runs use the floor 1e-2 below, where the same absolute
# errors give (1-4)e-6 -- still a statement the primary metric does not make (a cell at a hundredth of the scale
# that is wrong by a tenth of a percent fails it).
PURE_FLOOR_LARGE = 1e-2


def assert_pure_large(g, o, dtype, what=()):
    """Secondary metric of Q21 on full-size bunches and after several steps: floor 1e-2, north_star tolerance."""
    e = rel_err_pure(g, o, floor=PURE_FLOOR_LARGE)
    assert e <= TOL_PURE[dtype], (what, dtype, "pure relative (floor 1e-2)", e)
    return e


def assert_step_parity(g, o, dtype, what=(), tight=True):
    """Both Q21 metrics of a stepped state against the oracle's, at the north_star tolerance and
    (tight) at the regression bound; returns (primary, secondary)."""
    e1, e2 = rel_err(g, o), rel_err_pure(g, o)
    assert e1 <= (TIGHT_STEP if tight else TOL_STEP)[dtype], (what, dtype, "scale-relative", e1)
    assert e2 <= TOL_PURE[dtype], (what, dtype, "pure relative", e2)
    return e1, e2


def assert_nstep_parity(g, o, dtype, what=()):
    """north_star's N-step criteria on interior data [8, ...]: conserved totals of rho, m, E to 1e-12
    relative in fp64, relative L1 norm of each field group to 1e-4 in fp32 (and in fp64, where it is
    far smaller)."""
    g = g.astype(np.float64)
    ax = tuple(range(1, g.ndim))
    tg, to = g[:5].sum(axis=ax), o[:5].sum(axis=ax)
    msum = np.abs(o[1:4]).sum()
    scale = np.array([abs(to[0]), msum, msum, msum, abs(to[4])])
    if dtype == "f64":
        assert np.all(np.abs(tg - to) <= TOL_TOTALS_F64 * scale), (what, (tg - to) / scale)
    for a, b in GROUPS:
        l1 = np.abs(g[a:b] - o[a:b]).sum() / max(np.abs(o[a:b]).sum(), 1e-300)
        assert l1 <= TOL_L1_F32, (what, dtype, a, l1)


def updated_mask(n, ng=3):
    """Boolean [8, mz, my, mx]: cells a step writes (interior; closing faces for B)."""
    mx, my, mz = W.padded(n, ng)
    g = [ng if k > 1 else 0 for k in n]
    m = np.zeros((8, mz, my, mx), dtype=bool)
    I = (slice(g[2], g[2] + n[2]), slice(g[1], g[1] + n[1]), slice(g[0], g[0] + n[0]))
    m[(slice(None),) + I] = True
    if n[0] > 1: m[5, I[0], I[1], g[0] + n[0]] = True
    if n[1] > 1: m[6, I[0], g[1] + n[1], I[2]] = True
    if n[2] > 1: m[7, g[2] + n[2], I[1], I[2]] = True
    return m


def make_oracle(w, limiter=1, emf_solver=0, flux_solver=0):
    return oracle.Oracle(w.n, w.npatch, w.gamma, w.dx, limiter=limiter, emf_solver=emf_solver, flux_solver=flux_solver)


def make_gpu(w, dtype, limiter=1, emf_solver=0, workspace_bytes=None, path="auto", flux_solver=0):
    from paper_2508_09568_b200.binding import MhdBunch
    b = MhdBunch(w.n, w.npatch, w.nbr, w.gamma, w.dx, dtype=dtype, limiter=limiter, emf_solver=emf_solver,
                 workspace_bytes=workspace_bytes, flux_solver=flux_solver)
    b.set_path(path)
    b.load(w.U)
    return b


def masked(U, n):
    """Zero everything a step does not define, for whole-array comparisons."""
    m = updated_mask(n)
    return np.where(m[:, None], U, 0)
