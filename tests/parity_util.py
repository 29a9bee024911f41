"""Helpers shared by the GPU parity tests: the error metric of DESIGN.md (Q21) and
drivers that run the same seeded workload through the oracle and through the C ABI."""
import numpy as np

import oracle
from paper_2508_09568_b200 import workloads as W

GROUPS = [(0, 1), (1, 4), (4, 5), (5, 8)]      # rho; momentum; E; B

TOL_STEP = {"f64": 1e-12, "f32": 2e-5}         # BASELINE.json north_star: per-cell relative error after one step
TOL_TOTALS_F64 = 1e-12                         # conserved totals after N steps
TOL_L1_F32 = 1e-4                              # L1 field norms after N steps


def rel_err(g, o):
    """max over cells of |g-o| / max(|o|, s_f), s_f = max|o| of the field group (1 if 0)."""
    worst = 0.0
    for a, b in GROUPS:
        s = np.abs(o[a:b]).max()
        s = s if s > 0 else 1.0
        # compare at the scale of the group: a cell near zero is measured against s_f
        e = np.abs(g[a:b].astype(np.float64) - o[a:b]) / np.maximum(np.abs(o[a:b]), s)
        worst = max(worst, float(e.max()))
    return worst


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
