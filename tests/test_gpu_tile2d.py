"""GPU parity of the one-kernel step of two-dimensional bunches (MHD_PATH_TILE2D, csrc/tile_kernel.cuh;
BASELINE.json config 1 = the paper's Orszag-Tang runs): every stage of PAPER.md section
2.1.4 on a shared-memory tile.  Checked against the CPU oracle and, bit for bit, against the staged path
(the two run the same stage functions: they agree to rounding -- not always bit for bit, the compiler is free
to contract multiply-adds differently in the two instantiations)."""
import numpy as np
import pytest

from parity_util import TOL_STEP, assert_nstep_parity, assert_step_parity, make_gpu, make_oracle, masked, rel_err
from paper_2508_09568_b200 import workloads as W

pytestmark = pytest.mark.gpu
NPD = {"f32": np.float32, "f64": np.float64}


def workloads_2d(dtype):
    t = NPD[dtype]
    w = {
        "ot64": W.orszag_tang(64, 32, dtype=t),              # 2 x 2 patches of 32^2: whole tiles in x
        "ot_ragged": W.orszag_tang(60, 20, dtype=t),         # 20^2 patches: ragged tiles in x and y
        "ot_wide": W.orszag_tang(80, 40, dtype=t),           # 40^2 patches: two x-tiles, several y-tiles
        "ot_tiny": W.orszag_tang(12, 3, dtype=t),            # n = guard width: the thinnest legal patch
        "ot_self": W.orszag_tang(24, 24, dtype=t),           # one patch, its own neighbour
    }
    # a 2.5D state: out-of-plane velocity and field, so that e_x, e_y and the b_z update do work
    rng = np.random.default_rng(7)
    for k in ("ot64", "ot_ragged"):
        u = w[k].U
        u[3] += (0.3 * u[0] * (1 + 0.2 * rng.standard_normal(u[0].shape))).astype(t)      # m_z (zero in the guard shell)
        u[7] += t(0.2)                                                                       # b_z
        u[4] += (0.5 * u[3] ** 2 / np.where(u[0] > 0, u[0], 1) + 0.5 * 0.04).astype(t)
    return w


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("limiter,emf_solver,flux_solver", [(1, 0, 0), (2, 1, 1)])
@pytest.mark.parametrize("name", ["ot64", "ot_ragged", "ot_wide", "ot_tiny", "ot_self"])
def test_tile2d_step_matches_oracle_and_the_staged_path(name, dtype, limiter, emf_solver, flux_solver):
    w = workloads_2d(dtype)[name]
    o = make_oracle(w, limiter, emf_solver, flux_solver=flux_solver)
    outs = {}
    for path in ("tile2d", "staged"):
        b = make_gpu(w, dtype, limiter, emf_solver, path=path, flux_solver=flux_solver)
        assert b.path == path
        U = w.U.astype(np.float64)
        for s in range(3):
            U = o.fill_guards(U, w.nbr)
            dt = o.cfl_dt(U, 0.4)
            U = o.step(U, dt)
            b.fill_guards()
            b.step(dt)
            if s == 0:
                assert_step_parity(masked(b.download(), w.n), masked(U, w.n), dtype, (name, path))
        outs[path] = b.download()
        assert b.status() == 0
        b.close()
    got = outs["tile2d"]
    assert rel_err(masked(got, w.n), masked(U, w.n)) <= TOL_STEP[dtype]
    assert_nstep_parity(W.gather(got, w.n, w.P), W.gather(U, w.n, w.P), dtype, name)
    close = {"f64": 1e-14, "f32": 2e-6}[dtype]
    assert rel_err(masked(got, w.n), masked(outs["staged"], w.n).astype(np.float64)) <= close


def test_tile2d_is_the_default_for_2d_bunches_and_one_launch():
    w = W.orszag_tang(64, 32, dtype=np.float32)
    b = make_gpu(w, "f32")
    assert b.path == "tile2d"
    b.fill_guards()
    l0 = b.launches
    b.step(1e-3)
    assert b.launches - l0 == 2                 # k_set_dt + the step
    with pytest.raises(RuntimeError):
        make_gpu(W.turbulence(N=32, n=16, dtype=np.float32), "f32", path="tile2d")     # 3D: not applicable
    b.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_tile2d_with_outflow_sides(dtype):
    """-1 neighbours: guard cells are zero-gradient copies (k_fill_guards) and a patch evolves its own
    closing faces (O8)."""
    w = W.orszag_tang(64, 32, dtype=NPD[dtype])
    w.nbr = W.neighbour_table(w.P, (False, True, True))
    o = make_oracle(w)
    b = make_gpu(w, dtype)
    U = w.U.astype(np.float64)
    for _ in range(3):
        U = o.fill_guards(U, w.nbr)
        dt = o.cfl_dt(U, 0.4)
        U = o.step(U, dt)
        b.fill_guards()
        b.step(dt)
    got = b.download()
    assert rel_err(masked(got, w.n), masked(U, w.n)) <= TOL_STEP[dtype]
    assert b.status() == 0
    b.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("name", ["ot64", "ot_ragged", "ot_self"])
def test_tile2d_defers_the_fill_too(name, dtype):
    """Periodic 2D bunches: the tile kernel reads its halo from the neighbours' interiors through the
    neighbour table, so mhd_bunch_fill_guards launches nothing in the loop.  What a caller sees equals an
    immediate fill (the shell after download, bit for bit against the oracle's fill), and steps with and
    without the shell written first agree bit for bit."""
    w = workloads_2d(dtype)[name]
    o = make_oracle(w)
    outs, launches = [], []
    for force in (False, True):
        b = make_gpu(w, dtype)
        assert b.path == "tile2d"
        l0 = b.launches
        for _ in range(3):
            b.fill_guards()
            if force:
                b.sync_guards()
            b.cfl_dt(0.4, sync=False)
            b.step_dev()
        launches.append(b.launches - l0)
        b.fill_guards()
        outs.append(b.download())
        b.close()
    assert np.array_equal(outs[0], outs[1])
    assert launches[0] < launches[1]                                   # no k_fill_guards in the deferred loop
    ref = o.fill_guards(outs[0].astype(np.float64).copy(), w.nbr)
    assert np.array_equal(outs[0].astype(np.float64), ref)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("name", ["ot64", "ot_ragged", "ot_wide"])
def test_tile2d_cfl_epilogue_gives_the_standalone_pass_bit_for_bit(name, dtype):
    """The tile kernel reduces the CFL rates of the level it writes (O9), so the next cfl_dt is
    one small launch; the step it returns equals, bit for bit, the one k_cfl computes from the stored state."""
    w = workloads_2d(dtype)[name]
    b = make_gpu(w, dtype)
    for _ in range(2):
        b.fill_guards(); b.cfl_dt(0.4, sync=False); b.step_dev()
    b.fill_guards()
    l0 = b.launches
    dt1 = b.cfl_dt(0.4, sync=True)
    assert b.launches - l0 == 1                      # k_cfl_final only
    U = b.download()
    b.load(U)                                        # the caller wrote the buffer: the rates are no longer trusted
    b.fill_guards()
    l0 = b.launches
    dt2 = b.cfl_dt(0.4, sync=True)
    assert b.launches - l0 >= 3                      # zero, k_cfl, k_cfl_final
    assert dt1 == dt2
    o = make_oracle(w)
    ref = o.cfl_dt(o.fill_guards(U.astype(np.float64), w.nbr), 0.4)
    assert abs(dt1 - ref) <= (1e-13 if dtype == "f64" else 2e-6) * ref
    b.close()


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("N,n", [(512, 32), (480, 20)])
def test_tile2d_on_bunches_of_many_waves(N, n, dtype):
    """More than two waves of tiles: in fp32 persistent CTAs walk the tiles and prefetch the next tile's U^n
    with asynchronous copies while the current one is computed (two raw buffers); the CFL epilogue is off
    beyond eight waves.  Two chained steps against the oracle, and the staged path to rounding."""
    w = W.orszag_tang(N, n, dtype=NPD[dtype])
    o = make_oracle(w)
    U = w.U.astype(np.float64)
    outs = {}
    for path in ("tile2d", "staged"):
        b = make_gpu(w, dtype, path=path)
        V = U
        for _ in range(2):
            V = o.fill_guards(V, w.nbr) if path == "tile2d" else V
            if path == "tile2d":
                dt = o.cfl_dt(V, 0.4)
                V = o.step(V, dt)
                dts = outs.setdefault("dts", [])
                dts.append(dt)
            b.fill_guards()
            b.step(outs["dts"][len(outs.get("n_" + path, []))])
            outs.setdefault("n_" + path, []).append(1)
        outs[path] = b.download()
        if path == "tile2d":
            ref = V
        assert b.status() == 0
        b.close()
    assert rel_err(masked(outs["tile2d"], w.n), masked(ref, w.n)) <= TOL_STEP[dtype]
    assert_nstep_parity(W.gather(outs["tile2d"], w.n, w.P), W.gather(ref, w.n, w.P), dtype, (N, n))
    close = {"f64": 1e-14, "f32": 2e-6}[dtype]
    assert rel_err(masked(outs["tile2d"], w.n), masked(outs["staged"], w.n).astype(np.float64)) <= close


# ------------------------------------------------------------------ one-dimensional bunches along x ----
def workloads_1d(dtype):
    t = NPD[dtype]
    return {
        "sod": W.sod(256, 8, dtype=t),                                             # config 0: outflow ends
        "tube": W.mhd_tube((1.0, 0.2, 0.3, -0.1, 1.0, 1.0, 0.4), (0.125, -0.1, -0.2, 0.25, 0.1, -1.0, 0.2), 0.75, 2.0,
                           ncell=120, npatch=3, axis=0, dtype=t),                   # all seven waves, ragged n = 40
        "alfven": W.alfven_wave(N=64, n=16, dtype=t),                               # periodic: halo gathered through the table
        "alfven_self": W.alfven_wave(N=24, n=24, dtype=t),                          # one patch, its own neighbour
    }


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("limiter,emf_solver,flux_solver", [(1, 0, 0), (2, 1, 1)])
@pytest.mark.parametrize("name", ["sod", "tube", "alfven", "alfven_self"])
def test_line_kernel_on_1d_bunches_matches_oracle_and_the_staged_path(name, dtype, limiter, emf_solver, flux_solver):
    """1D bunches along x (config 0) step in one kernel too (k_step_line1d: the stages on the whole row of a patch);
    three chained steps against the oracle, the staged path to rounding, the CFL step from the kernel's epilogue bit
    for bit the stand-alone pass's."""
    w = workloads_1d(dtype)[name]
    o = make_oracle(w, limiter, emf_solver, flux_solver=flux_solver)
    outs = {}
    for path in ("tile2d", "staged"):
        b = make_gpu(w, dtype, limiter, emf_solver, path=path, flux_solver=flux_solver)
        assert b.path == path
        U = w.U.astype(np.float64)
        for s in range(3):
            U = o.fill_guards(U, w.nbr)
            dt = o.cfl_dt(U, 0.4)
            U = o.step(U, dt)
            b.fill_guards()
            b.step(dt)
        if path == "tile2d":
            b.fill_guards()
            dt1 = b.cfl_dt(0.4, sync=True)
            V = b.download()
            b.load(V)
            b.fill_guards()
            assert b.cfl_dt(0.4, sync=True) == dt1
        outs[path] = b.download()
        assert b.status() == 0
        b.close()
    got = outs["tile2d"]
    assert rel_err(masked(got, w.n), masked(U, w.n)) <= TOL_STEP[dtype]
    assert_nstep_parity(W.gather(got, w.n, w.P), W.gather(U, w.n, w.P), dtype, name)
    close = {"f64": 1e-14, "f32": 2e-6}[dtype]
    assert rel_err(masked(got, w.n), masked(outs["staged"], w.n).astype(np.float64)) <= close


def test_1d_bunches_along_y_or_z_stay_on_the_staged_path():
    b = make_gpu(W.sod(96, 3, dtype=np.float64, axis=1), "f64")
    assert b.path == "staged"
    b.close()
