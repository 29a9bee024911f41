"""Pins of the oracle's local-time-step extension (reading O10 of DESIGN.md; patches
hold several time slices and their own time and time step; L188, L200: ghost zones of neighbours that
sit at other times are interpolated).  Nothing here calls the oracle twice to compare it with itself:
expected values come from the global step (already pinned), from closed forms of the interpolation,
and from an exact solution."""
import numpy as np
import pytest

import oracle
from paper_2508_09568_b200 import workloads as W


def _oracle(w, **kw):
    return oracle.Oracle(w.n, w.npatch, w.gamma, w.dx, **kw)


def test_uniform_dt_reproduces_the_global_step_bitwise():
    """All patches listed, one dt: every neighbour is at the patch's own time, guard values are the
    neighbours' newer slices themselves, so the scheme is the global one -- bit for bit, over steps."""
    w = W.turbulence(N=16, n=8, dtype=np.float64)
    o = _oracle(w)
    U = w.U.copy()
    st = o.local_state(w.U)
    allp = np.arange(w.npatch)
    for _ in range(4):
        o.fill_guards(U, w.nbr)
        dt = o.cfl_dt(U, 0.4)
        U = o.step(U, dt)
        assert o.step_local(st, w.nbr, allp, dt)
    new = o.local_newest(st)
    I = o.interior
    assert np.array_equal(I(new), I(U))
    assert np.all(st["cur"] == 0) and np.allclose(st["t_new"] - st["t_old"], dt)


def test_guard_values_are_linear_in_time_between_the_two_slices():
    """Neighbour slices F0 at t = 2 and F1 at t = 3 (random, dyadic so that the arithmetic is exact):
    a patch at time 2.25 must see F0 + 0.25 (F1 - F0) in every guard cell that has a neighbour, at the
    cell's periodic image; at the end points it must see the slices themselves bit for bit."""
    n, P = (4, 3, 5), (2, 2, 2)
    nbr = W.neighbour_table(P, (True, True, True))
    o = oracle.Oracle(n, 8, 5 / 3, (1, 1, 1))
    rng = np.random.default_rng(3)
    F0 = rng.integers(-64, 64, size=o.shape).astype(np.float64) / 16
    F1 = rng.integers(-64, 64, size=o.shape).astype(np.float64) / 16
    p = 5
    for tp, expect in ((2.25, F0 + 0.25 * (F1 - F0)), (2.0, F0), (3.0, F1), (2.5, 0.5 * (F0 + F1))):
        st = {"S": [F0.copy(), F1.copy()], "cur": np.ones(8, dtype=np.int32), "t_old": np.full(8, 2.0), "t_new": np.full(8, 3.0)}
        st["t_new"][p] = tp
        st["t_old"][p] = 1.5
        mine = st["S"][1][:, p].copy()
        o.fill_guards_local(st, nbr, p)
        got = st["S"][1][:, p]
        # expected guard shell: the global periodic image of `expect`
        g = W.gather(expect, n, P)
        ref = np.empty_like(got)
        px, py, pz = p % 2, (p // 2) % 2, p // 4
        for k in range(n[2] + 6):
            for j in range(n[1] + 6):
                for i in range(n[0] + 6):
                    ref[:, k, j, i] = g[:, (pz * n[2] + k - 3) % (2 * n[2]), (py * n[1] + j - 3) % (2 * n[1]), (px * n[0] + i - 3) % (2 * n[0])]
        ref[:, 3:3 + n[2], 3:3 + n[1], 3:3 + n[0]] = mine[:, 3:3 + n[2], 3:3 + n[1], 3:3 + n[0]]   # own interior untouched
        assert np.array_equal(got, ref), tp
        # nobody else's data moved
        for q in range(8):
            if q != p:
                assert np.array_equal(st["S"][1][:, q], F1[:, q]) and np.array_equal(st["S"][0][:, q], F0[:, q])


def test_readiness_rule_is_enforced_and_a_refused_call_changes_nothing():
    w = W.turbulence(N=16, n=8, dtype=np.float64)
    o = _oracle(w)
    st = o.local_state(w.U)
    assert o.step_local(st, w.nbr, np.arange(8), 1e-3)
    assert o.step_local(st, w.nbr, [0], 5e-4)                    # 0 -> 1.5e-3, neighbours at 1e-3
    before = [s.copy() for s in st["S"]], st["cur"].copy(), st["t_new"].copy()
    assert not o.local_ready(st, w.nbr, [0])                     # its neighbours are behind it now
    assert not o.step_local(st, w.nbr, [0], 5e-4)
    assert all(np.array_equal(a, b) for a, b in zip(before[0], st["S"])) and np.array_equal(before[1], st["cur"])
    assert np.array_equal(before[2], st["t_new"])
    assert o.local_ready(st, w.nbr, [1, 2, 3, 4, 5, 6, 7])       # the others may catch up (0 brackets their time)
    assert not o.local_ready(st, w.nbr, [99]) and not o.local_ready(st, w.nbr, [-1])


def _subcycled_run(w, o, fine, t_end, dt):
    """Scheduler of the test: patches in `fine` step with dt/2, the others with dt; always advance the
    patches with the smallest time (they are the ready ones)."""
    st = o.local_state(o.fill_guards(w.U.copy(), w.nbr))
    steps = 0
    while st["t_new"].min() < t_end * (1 - 1e-12):
        tmin = st["t_new"].min()
        lst = [p for p in range(w.npatch) if abs(st["t_new"][p] - tmin) <= 1e-12]
        dts = [dt / 2 if p in fine else dt for p in lst]
        assert o.step_local(st, w.nbr, lst, dts), (lst, st["t_new"])
        steps += 1
    assert np.allclose(st["t_new"], t_end)
    return o.local_newest(st), steps


def test_subcycled_patches_track_the_uniformly_stepped_solution():
    """A circularly polarised Alfven wave (exact solution, period 1) on four patches, two of which
    take two half steps per step of the others: the run must be stable and as accurate as the
    uniformly stepped runs that bracket it (error against the exact solution between those of dt and
    dt/2 everywhere, within 20 %), and it need not conserve exactly: the fluxes through the faces
    between a fine and a coarse patch are evaluated at different times on the two sides."""
    w = W.alfven_wave(N=64, n=16)
    o = _oracle(w, limiter=2)
    dt = 1.0 / 256
    exact = W.gather(w.U, w.n, w.P)          # after one period the wave is back

    def err(U):
        g = W.gather(U, w.n, w.P)
        return np.abs(g[6] - exact[6]).mean() + np.abs(g[7] - exact[7]).mean()
    coarse, _ = _subcycled_run(w, o, set(), 1.0, dt)
    fine, _ = _subcycled_run(w, o, {0, 1, 2, 3}, 1.0, dt)
    mixed, steps = _subcycled_run(w, o, {1, 2}, 1.0, dt)
    assert steps == 2 * 256
    e_c, e_f, e_m = err(coarse), err(fine), err(mixed)
    assert np.isfinite(mixed).all()
    assert e_m <= 1.2 * max(e_c, e_f) and e_m >= 0.8 * min(e_c, e_f), (e_c, e_f, e_m)
    I = o.interior
    drift = abs(I(mixed)[4].sum() - I(w.U)[4].sum()) / I(w.U)[4].sum()
    assert drift < 1e-3                       # small, but not round-off: no flux correction (PAPER.md is silent)


def test_subcycling_equal_split_is_the_uniform_run_bitwise():
    """If every patch is "fine" the subcycled scheduler is the uniform run with dt/2 -- the same bits
    as the global step: the list-driven path has no arithmetic of its own besides the interpolation."""
    w = W.turbulence(N=16, n=8, dtype=np.float64)
    o = _oracle(w)
    dt = 2e-3
    a, _ = _subcycled_run(w, o, set(range(8)), 4 * dt, dt)
    U = w.U.copy()
    for _ in range(8):
        o.fill_guards(U, w.nbr)
        U = o.step(U, dt / 2)
    assert np.array_equal(o.interior(a), o.interior(U))
