"""GPU parity of the local-time-step calls (mhd_bunch_local_*, reading O10) against
the extended oracle, on every implementation of the step."""
import numpy as np
import pytest

from parity_util import TOL_STEP, assert_nstep_parity, assert_pure_large, make_gpu, make_oracle, masked, rel_err
from paper_2508_09568_b200 import workloads as W

pytestmark = pytest.mark.gpu
NPD = {"f32": np.float32, "f64": np.float64}


def _workload(name, dtype):
    t = NPD[dtype]
    return {"turb8": lambda: W.turbulence(N=16, n=8, dtype=t),                 # 2 x 2 x 2 patches
            "turb16": lambda: W.turbulence(N=32, n=16, dtype=t),
            "turb_ragged": lambda: W.turbulence(N=(24, 20, 36), n=(12, 10, 9), dtype=t),
            "ot64": lambda: W.orszag_tang(64, 32, dtype=t),
            "sod_x": lambda: W.sod(256, 8, dtype=t)}[name]()


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("name,path", [("turb16", "auto"), ("turb16", "two_kernel"), ("turb16", "staged"),
                                       ("turb_ragged", "auto"), ("ot64", "auto"), ("sod_x", "auto")])
def test_uniform_dt_over_all_patches_is_the_global_step_bitwise(name, path, dtype):
    w = _workload(name, dtype)
    a = make_gpu(w, dtype, path=path)
    b = make_gpu(w, dtype, path=path)
    b.local_begin(0.0)
    allp = np.arange(w.npatch)
    for _ in range(3):
        a.fill_guards(); dt = a.cfl_dt(0.4, sync=True); a.step(dt)
        assert b.cfl_local(0.4).min() == dt                     # the same reduction over the same slices
        assert b.step_local(allp, dt)
    t0, t1, slot = b.local_state()
    assert np.all(t1 == t1[0]) and np.all(slot == slot[0])
    assert np.array_equal(masked(b.local_newest(), w.n), masked(a.download(), w.n))
    b.local_end()
    assert np.array_equal(masked(b.download(), w.n), masked(a.download(), w.n))
    a.close(); b.close()


def _subcycle(step, ready_times, fine, npatch, t_end, dt):
    """The scheduler of the tests: patches in `fine` take dt/2, the others dt; always advance the
    patches with the smallest time."""
    calls = 0
    while True:
        t = ready_times()
        if t.min() >= t_end * (1 - 1e-12):
            return calls
        lst = [p for p in range(npatch) if abs(t[p] - t.min()) <= 1e-12 * max(1.0, t.min())]
        assert step(lst, [dt / 2 if p in fine else dt for p in lst]), (lst, t)
        calls += 1


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("name,path,fine", [("turb8", "auto", {0, 3, 5}), ("turb8", "two_kernel", {7}), ("turb8", "staged", {0, 3, 5}),
                                            ("turb16", "auto", {1, 2, 4, 7}), ("turb_ragged", "auto", {0, 5, 6}),
                                            ("ot64", "auto", {0}), ("sod_x", "auto", {2, 3, 4})])
def test_two_distinct_time_steps_against_the_oracle(name, path, fine, dtype):
    """A bunch whose patches step with dt or dt/2 (neighbours of both kinds next to each other, guard
    values interpolated half way between the coarse patches' slices): every call against the extended
    oracle, which runs the same schedule."""
    w = _workload(name, dtype)
    o = make_oracle(w)
    U0 = o.fill_guards(w.U.astype(np.float64), w.nbr)
    dt = 0.8 * o.cfl_dt(U0, 0.4)
    st = o.local_state(w.U.astype(np.float64))
    b = make_gpu(w, dtype, path=path)
    b.local_begin(0.0)
    n1 = _subcycle(lambda l, d: o.step_local(st, w.nbr, l, d), lambda: st["t_new"], fine, w.npatch, 3 * dt, dt)
    n2 = _subcycle(lambda l, d: b.step_local(l, d), lambda: b.local_state()[1], fine, w.npatch, 3 * dt, dt)
    assert n1 == n2 == 6
    t0, t1, slot = b.local_state()
    assert np.allclose(t1, st["t_new"], rtol=0, atol=1e-15) and np.array_equal(slot, st["cur"])
    got, ref = b.local_newest(), o.local_newest(st)
    assert rel_err(masked(got, w.n), masked(ref, w.n)) <= TOL_STEP[dtype], (name, path, dtype)
    assert_pure_large(masked(got, w.n), masked(ref, w.n), dtype, (name, path))
    assert_nstep_parity(W.gather(got, w.n, w.P), W.gather(ref, w.n, w.P), dtype, name)
    # per-patch CFL steps of the newer slices
    dts = b.cfl_local(0.4)
    _, ref_dts = o.cfl_dt(ref, 0.4, per_patch=True)
    assert np.all(np.abs(dts - ref_dts) <= (1e-13 if dtype == "f64" else 2e-6) * ref_dts)
    assert b.status() == 0
    # the coarse patches flipped buffers three times, the fine ones six: local_end gathers the newer slices
    # from both buffers into the current level (one launch over patches and fields)
    assert len(set(slot.tolist())) == 2
    b.local_end()
    assert np.array_equal(masked(b.download(), w.n), masked(got, w.n))
    b.close()


def test_a_patch_that_is_not_ready_is_refused_and_nothing_changes():
    w = _workload("turb8", "f32")
    b = make_gpu(w, "f32")
    b.local_begin(1.0)
    assert b.step_local(np.arange(8), 1e-3)
    assert b.step_local([0], 5e-4)                      # patch 0 is now ahead of its neighbours
    before, state = b.local_newest(), b.local_state()
    assert not b.step_local([0], 5e-4)                  # ... and must wait for them
    assert np.array_equal(before, b.local_newest())
    assert all(np.array_equal(x, y) for x, y in zip(state, b.local_state()))
    assert b.step_local([1, 2, 3, 4, 5, 6, 7], 5e-4)    # they are bracketed by patch 0's slices
    assert b.lib.mhd_bunch_step_local(b.h, None, 1, None) == -1
    assert b.lib.mhd_bunch_step(b.h, 1e-3) == -4        # the global step is closed in local mode
    assert b.lib.mhd_bunch_local_end(b.h) == 0          # all at 1.0015 again
    assert b.lib.mhd_bunch_local_end(b.h) == -4
    b.close()
