"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by
element on the same seeded inputs.  Tolerances are BASELINE.json's: one step <= 1e-12
(fp64) / 2e-5 (fp32) per cell; N steps: totals 1e-12 (fp64), L1 norms 1e-4 (fp32).
fp32 runs are compared with the fp64 oracle on the same fp32-representable inputs."""
import numpy as np
import pytest

import exact_riemann
from parity_util import (TOL_L1_F32, TOL_STEP, TOL_TOTALS_F64, assert_nstep_parity, assert_pure_large, assert_step_parity, make_gpu,
                         make_oracle, masked, rel_err)
from paper_2508_09568_b200 import workloads as W

pytestmark = pytest.mark.gpu
NPD = {"f32": np.float32, "f64": np.float64}


def small_workloads(dtype):
    t = NPD[dtype]
    return {
        "sod_x": W.sod(256, 8, dtype=t),
        "sod_y": W.sod(96, 3, dtype=t, axis=1),
        "tube_z": W.mhd_tube((1.0, 0.2, 0.3, -0.1, 1.0, 1.0, 0.4), (0.125, -0.1, -0.2, 0.25, 0.1, -1.0, 0.2), 0.75, 2.0,
                             ncell=120, npatch=3, axis=2, dtype=t),
        "ot64": W.orszag_tang(64, 32, dtype=t),
        "ot_ragged": W.orszag_tang(60, 20, dtype=t),
        "turb16": W.turbulence(N=32, n=16, dtype=t),
        "turb_ragged": W.turbulence(N=(24, 20, 36), n=(12, 10, 9), dtype=t),
        "turb_self": W.turbulence(N=16, n=16, dtype=t),          # one patch, its own neighbour
        # rows that are not a whole number of 16-byte chunks, every neighbour present: the one-pass
        # kernel reads the patch's own guard cells (no gather) with ragged x-tiles
        "turb_nx10": W.turbulence(N=(20, 24, 18), n=(10, 12, 9), dtype=t),
        "turb_nx38": W.turbulence(N=(38, 16, 16), n=(38, 8, 8), dtype=t),
        "turb_thin": W.turbulence(N=6, n=3, dtype=t),            # n == ng: the thinnest legal patch
    }

THREE_D = ["turb16", "turb_ragged", "turb_self", "turb_nx10", "turb_nx38", "turb_thin"]


# ---------------------------------------------------------------- guard fill -------
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("name", ["sod_x", "sod_y", "tube_z", "ot64", "ot_ragged"] + THREE_D)
def test_fill_guards_bit_exact(name, dtype):
    w = small_workloads(dtype)[name]
    rng = np.random.default_rng(5)
    U = rng.normal(size=w.U.shape).astype(NPD[dtype])            # every slot distinct, guards included
    w.U = U
    o = make_oracle(w)
    ref = o.fill_guards(U.astype(np.float64).copy(), w.nbr)
    b = make_gpu(w, dtype)
    b.fill_guards()
    got = b.download()
    assert np.array_equal(got.astype(np.float64), ref)
    b.close()


def test_fill_guards_mixed_outflow_periodic_3d():
    P = (2, 1, 3)
    n = (4, 5, 6)
    nbr = W.neighbour_table(P, (False, True, False))
    w = W.Workload("mix", n, P, 5 / 3, (1, 1, 1), (False, True, False),
                   np.random.default_rng(6).normal(size=(8, 6) + tuple(reversed(W.padded(n)))), nbr)
    ref = make_oracle(w).fill_guards(w.U.copy(), nbr)
    b = make_gpu(w, "f64")
    b.fill_guards()
    assert np.array_equal(b.download(), ref)
    b.close()


@pytest.mark.parametrize("name", ["turb16", "turb_ragged", "turb_self"])
def test_deferred_fill_is_indistinguishable_from_an_immediate_one(name):
    """fp32 periodic 3D bunches defer the fill (the one-pass kernel reads halos from the
    neighbours' interiors; include/mhd_bunch.h).  Whatever the caller can see must equal an
    immediate fill: (a) the guard shell after download, bit for bit against the oracle's
    fill, also after steps; (b) a step that read neighbours' interiors equals, bit for bit,
    the same steps with the guard shell written first; the launch count shows which route
    ran."""
    w = small_workloads("f32")[name]
    o = make_oracle(w)
    # (a) random data, guards included
    rng = np.random.default_rng(11)
    w.U = rng.normal(size=w.U.shape).astype(np.float32)
    b = make_gpu(w, "f32")
    assert b.path == "onepass"
    b.fill_guards()
    l0 = b.launches
    got = b.download()
    deferred = (b.launches - l0) == 1          # the owed fill ran when the buffer was looked at
    assert deferred == (bool((w.nbr >= 0).all()) and w.n[0] % 4 == 0)
    assert np.array_equal(got.astype(np.float64), o.fill_guards(w.U.astype(np.float64).copy(), w.nbr))
    b.close()
    # (b) physical data: deferred fill + step, against fill written first (sync_guards) + step
    w = small_workloads("f32")[name]
    outs = []
    for force in (False, True):
        b = make_gpu(w, "f32")
        for _ in range(3):
            b.fill_guards()
            if force:
                b.sync_guards()
            b.cfl_dt(0.4, sync=False)
            b.step_dev()
        b.fill_guards()
        outs.append(b.download())
        b.close()
    assert np.array_equal(outs[0], outs[1])
    ref = o.fill_guards(outs[0].astype(np.float64).copy(), w.nbr)
    assert np.array_equal(outs[0].astype(np.float64), ref)
    assert deferred, "periodic fp32 3D bunches with n_x % 4 == 0 are expected to take the deferred route"


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("name", ["turb16", "turb_ragged", "turb_self"])
def test_two_kernel_path_defers_the_fill_too(name, dtype):
    """The two-kernel path (the fp64 default) reads halos through the neighbour table in its
    predictor when every neighbour exists: three steps with the fill deferred equal, bit for bit,
    three steps with the guard shell written first, and the shell a caller then sees equals the
    oracle's fill of the result."""
    w = small_workloads(dtype)[name]
    outs, launches = [], []
    for force in (False, True):
        b = make_gpu(w, dtype, path="two_kernel")
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
    assert launches[0] < launches[1]                      # no fill kernel inside the deferred loop
    ref = make_oracle(w).fill_guards(outs[0].astype(np.float64).copy(), w.nbr)
    assert np.array_equal(outs[0].astype(np.float64), ref)


# ------------------------------------------------------------------------ CFL -------
@pytest.mark.parametrize("dtype,tol", [("f64", 1e-13), ("f32", 2e-6)])
@pytest.mark.parametrize("name", ["sod_x", "tube_z", "ot_ragged", "turb_ragged"])
def test_cfl_dt_matches_oracle(name, dtype, tol):
    w = small_workloads(dtype)[name]
    o = make_oracle(w)
    U = o.fill_guards(w.U.astype(np.float64), w.nbr)
    dt_ref, pp_ref = o.cfl_dt(U, 0.4, per_patch=True)
    b = make_gpu(w, dtype)
    b.fill_guards()
    dt = b.cfl_dt(0.4, sync=True, per_patch=True)
    assert abs(dt - dt_ref) <= tol * dt_ref
    assert np.allclose(b.dt_patch.cpu().numpy(), pp_ref, rtol=tol, atol=0)
    assert abs(b.dt_dev.item() - dt) == 0
    b.close()


# ------------------------------------------------------------------- one step -------
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("limiter,emf_solver", [(1, 0), (2, 0), (1, 1)])
@pytest.mark.parametrize("name", ["sod_x", "sod_y", "tube_z", "ot64", "ot_ragged"] + THREE_D)
def test_one_step_matches_oracle(name, dtype, limiter, emf_solver):
    w = small_workloads(dtype)[name]
    o = make_oracle(w, limiter, emf_solver)
    U = o.fill_guards(w.U.astype(np.float64), w.nbr)
    dt = o.cfl_dt(U, 0.4)
    ref = o.step(U, dt)
    b = make_gpu(w, dtype, limiter, emf_solver)
    b.fill_guards()
    b.step(dt)
    got = b.download()
    assert_step_parity(masked(got, w.n), masked(ref, w.n), dtype, name)
    assert b.status() == 0
    b.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("limiter,emf_solver", [(1, 0), (2, 1)])
@pytest.mark.parametrize("name", THREE_D)
@pytest.mark.parametrize("path", ["staged", "two_kernel"])
def test_every_step_path_on_3d_bunches_matches_oracle(path, name, dtype, limiter, emf_solver):
    """3D bunches default to the one-pass kernel (fp32) or the two fused kernels (fp64); the
    other implementations of the step must agree with the oracle there as well (the staged
    kernels are the only path for collapsed dimensions)."""
    w = small_workloads(dtype)[name]
    o = make_oracle(w, limiter, emf_solver)
    U = o.fill_guards(w.U.astype(np.float64), w.nbr)
    dt = o.cfl_dt(U, 0.4)
    ref = o.step(U, dt)
    b = make_gpu(w, dtype, limiter, emf_solver, path=path)
    assert b.path == path
    b.fill_guards()
    b.step(dt)
    assert_step_parity(masked(b.download(), w.n), masked(ref, w.n), dtype, (name, path))
    b.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("path", ["auto", "staged", "two_kernel"])
@pytest.mark.parametrize("name", ["sod_x", "tube_z", "ot_ragged", "turb16", "turb_ragged", "turb_self", "turb_nx10"])
def test_hll_flux_variant_matches_oracle(name, path, dtype):
    """flux_solver = 1: the HLL flux of PAPER.md 2.1.1 at the faces, on every
    implementation of the step; three chained steps so that the variant's own states feed back."""
    w = small_workloads(dtype)[name]
    if path == "two_kernel" and not all(k > 1 for k in w.n):
        pytest.skip("the two-kernel path needs three active dimensions")
    o = make_oracle(w, 2, 1, flux_solver=1)
    b = make_gpu(w, dtype, 2, 1, path=path, flux_solver=1)
    U = w.U.astype(np.float64)
    for _ in range(3):
        U = o.fill_guards(U, w.nbr)
        dt = o.cfl_dt(U, 0.4)
        U = o.step(U, dt)
        b.fill_guards()
        b.step(dt)
    # three steps: per cell still inside the ONE-step tolerance, and north_star's N-step criteria
    got = b.download()
    assert rel_err(masked(got, w.n), masked(U, w.n)) <= TOL_STEP[dtype], (name, dtype)
    assert_nstep_parity(W.gather(got, w.n, w.P), W.gather(U, w.n, w.P), dtype, name)
    # and it is a different scheme: the HLLD result differs
    o2 = make_oracle(w, 2, 1)
    V = o2.fill_guards(w.U.astype(np.float64), w.nbr)
    V = o2.step(V, o2.cfl_dt(V, 0.4))
    W1 = o.step(o.fill_guards(w.U.astype(np.float64), w.nbr), o2.cfl_dt(o2.fill_guards(w.U.astype(np.float64), w.nbr), 0.4))
    assert rel_err(masked(W1, w.n), masked(V, w.n)) > 100 * TOL_STEP["f64"]
    assert b.status() == 0
    b.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("path", ["auto", "staged", "two_kernel"])
@pytest.mark.parametrize("sides", [(False, True, True), (True, False, False), (False, False, False)])
def test_3d_bunch_with_outflow_sides(sides, path, dtype):
    """3D bunches whose table has -1 (zero-gradient outflow) neighbours: no halo can be gathered
    from a neighbour there, so the fused kernels read the guard shell `k_fill_guards` wrote, and a
    patch evolves its own closing faces (O8).  Three steps against the oracle."""
    w = W.turbulence(N=(32, 16, 32), n=(16, 16, 16), dtype=NPD[dtype])
    w.nbr = W.neighbour_table(w.P, sides)
    o = make_oracle(w)
    b = make_gpu(w, dtype, path=path)
    U = w.U.astype(np.float64)
    for _ in range(3):
        U = o.fill_guards(U, w.nbr)
        dt = o.cfl_dt(U, 0.4)
        U = o.step(U, dt)
        b.fill_guards()
        b.step(dt)
    # (no fill before the comparison: next to an outflow side a diagonal neighbour is -1 too, so
    # the closing face a patch evolved itself need not equal the face 0 a fill would copy over it)
    got = b.download()
    assert rel_err(masked(got, w.n), masked(U, w.n)) <= TOL_STEP[dtype], (sides, path, dtype)
    assert_nstep_parity(W.gather(got, w.n, w.P), W.gather(U, w.n, w.P), dtype, sides)
    ref_fill = o.fill_guards(got.astype(np.float64).copy(), w.nbr)
    b.fill_guards()
    assert np.array_equal(b.download().astype(np.float64), ref_fill)
    assert b.status() == 0
    b.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_fused_tiles_cover_large_and_odd_patches(dtype):
    """Patch sizes that need several (x,y) tiles of the fused kernels with ragged edges: 40 x 20 x 12
    cells and 64 x 8 x 8; 24^3 (the paper's patch size), 24 x 40 x 12 and 48 x 24 x 10."""
    for N, n in (((80, 40, 24), (40, 20, 12)), ((64, 16, 16), (64, 8, 8)), ((48, 48, 48), (24, 24, 24)),
                 ((48, 40, 24), (24, 40, 12)), ((48, 48, 20), (48, 24, 10))):
        w = W.turbulence(N=N, n=n, dtype=NPD[dtype])
        o = make_oracle(w)
        U = o.fill_guards(w.U.astype(np.float64), w.nbr)
        dt = o.cfl_dt(U, 0.4)
        ref = o.step(U, dt)
        b = make_gpu(w, dtype)
        b.fill_guards()
        b.step(dt)
        assert_step_parity(masked(b.download(), w.n), masked(ref, w.n), dtype, n)
        b.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_sub_bunch_chunking_is_bitwise_invisible(dtype):
    w = small_workloads(dtype)["turb16"]                        # 8 patches
    outs = []
    for ws in (None, 1):                                         # whole bunch at once / one patch per chunk
        b = make_gpu(w, dtype, workspace_bytes=ws, path="two_kernel")   # the path that uses the workspace
        b.fill_guards(); b.cfl_dt(0.4, sync=False); b.step_dev()
        outs.append((b.download(), b.chunk))
        b.close()
    assert outs[0][1] == 8 and outs[1][1] == 1
    assert np.array_equal(masked(outs[0][0], w.n), masked(outs[1][0], w.n))


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_device_dt_path_equals_host_dt_path(dtype):
    w = small_workloads(dtype)["ot64"]
    a = make_gpu(w, dtype); a.fill_guards(); dt = a.cfl_dt(0.4, sync=True); a.step(dt)
    b = make_gpu(w, dtype); b.fill_guards(); b.cfl_dt(0.4, sync=False); b.step_dev()
    assert np.array_equal(masked(a.download(), w.n), masked(b.download(), w.n))
    c = make_gpu(w, dtype); c.fill_guards(); c.cfl_dt(0.4, sync=False); c.step_dev(dt_max=dt / 2)
    d = make_gpu(w, dtype); d.fill_guards(); d.step(dt / 2)
    assert np.array_equal(masked(c.download(), w.n), masked(d.download(), w.n))
    for x in (a, b, c, d):
        x.close()


# -------------------------------------------------------------------- N steps -------
def run_both(w, dtype, nsteps, limiter=1, emf_solver=0):
    o = make_oracle(w, limiter, emf_solver)
    U = w.U.astype(np.float64)
    b = make_gpu(w, dtype, limiter, emf_solver)
    for _ in range(nsteps):
        o.fill_guards(U, w.nbr)
        dt = o.cfl_dt(U, 0.4)
        U = o.step(U, dt)
        b.fill_guards()
        b.step(dt)                                              # same dt sequence on both sides
    got = b.download()
    bad = b.status()
    b.close()
    return W.gather(got, w.n, w.P).astype(np.float64), W.gather(U, w.n, w.P), bad


@pytest.mark.parametrize("name,nsteps", [("turb16", 20), ("ot64", 40), ("tube_z", 40)])
def test_n_steps_fp64_totals_and_fields(name, nsteps):
    w = small_workloads("f64")[name]
    g, o, bad = run_both(w, "f64", nsteps)
    assert bad == 0
    assert_nstep_parity(g, o, "f64", name)
    assert rel_err(g, o) <= 1e-12                                # per cell, after N steps: still the one-step bound


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_n_steps_on_a_128_cube_cut_of_config2(dtype):
    """N-step parity on a 128^3 cut (64 patches of 32^3, the bench's patch size, several
    tiles per SM) with the config-2 field construction: 8 steps against the oracle."""
    w = W.turbulence(N=128, n=32, dtype=NPD[dtype], config=2)
    g, o, bad = run_both(w, dtype, 8)
    assert bad == 0
    tg, to = g[:5].sum(axis=(1, 2, 3)), o[:5].sum(axis=(1, 2, 3))
    scale = np.array([to[0], np.abs(o[1:4]).sum(), np.abs(o[1:4]).sum(), np.abs(o[1:4]).sum(), to[4]])
    if dtype == "f64":
        assert np.all(np.abs(tg - to) <= TOL_TOTALS_F64 * scale), (tg - to) / scale
        assert rel_err(g, o) <= 1e-10
    else:
        for a, b_ in ((0, 1), (1, 4), (4, 5), (5, 8)):
            l1 = np.abs(g[a:b_] - o[a:b_]).sum() / max(np.abs(o[a:b_]).sum(), 1e-300)
            assert l1 <= TOL_L1_F32, (a, l1)
        assert np.all(np.abs(tg - to) <= 2e-6 * scale)


@pytest.mark.parametrize("name,nsteps", [("turb16", 20), ("ot64", 40), ("tube_z", 40)])
def test_n_steps_fp32_l1_norms(name, nsteps):
    w = small_workloads("f32")[name]
    g, o, bad = run_both(w, "f32", nsteps)
    assert bad == 0
    for a, b_ in ((0, 1), (1, 4), (4, 5), (5, 8)):
        l1 = np.abs(g[a:b_] - o[a:b_]).sum() / max(np.abs(o[a:b_]).sum(), 1e-300)
        assert l1 <= TOL_L1_F32, (name, a, l1)
    tg, to = g[:5].sum(axis=(1, 2, 3)), o[:5].sum(axis=(1, 2, 3))
    assert abs(tg[0] - to[0]) <= 1e-5 * to[0] and abs(tg[4] - to[4]) <= 1e-5 * to[4]


# --------------------------------------------------------------- whole configs -------
def gpu_run(w, dtype, t_end=None, max_steps=10 ** 9, limiter=1):
    b = make_gpu(w, dtype, limiter)
    t, steps = 0.0, 0
    t_end = w.t_end if t_end is None else t_end
    while t < t_end * (1 - 1e-14) and steps < max_steps:
        b.fill_guards()
        dt = min(b.cfl_dt(w.courant, sync=True), t_end - t)
        b.step(dt)
        t += dt
        steps += 1
    out = b.download()
    bad = b.status()
    b.close()
    return out, t, steps, bad


def test_config0_sod_on_gpu_against_exact_solution_and_oracle():
    """BASELINE.json config 0: 256 cells, 8 patches of 32, fp64, CFL 0.4, t = 0.2."""
    w = W.sod(256, 8)
    U, t, steps, bad = gpu_run(w, "f64")
    assert bad == 0 and 270 <= steps <= 290
    g = W.gather(U, w.n, w.P)
    x = (np.arange(256) + 0.5) / 256
    ex = exact_riemann.sample((x - 0.5) / t, 1, 0, 1, 0.125, 0, 0.1, 1.4)
    assert np.abs(g[0, 0, 0] - ex[0]).mean() <= 3.5e-3
    assert not g[2:4].any() and not g[5:].any()
    # the oracle over the same run (seconds)
    o = make_oracle(w)
    V = w.U.copy(); tt = 0.0
    while tt < w.t_end * (1 - 1e-14):
        o.fill_guards(V, w.nbr)
        dt = min(o.cfl_dt(V, 0.4), w.t_end - tt)
        V = o.step(V, dt); tt += dt
    assert rel_err(g, W.gather(V, w.n, w.P)) <= 1e-10
    # bunch of 8 == single patch, bitwise, on the GPU too
    U1, _, s1, _ = gpu_run(W.sod(256, 1), "f64")
    assert s1 == steps and np.array_equal(W.gather(U1, (256, 1, 1), (1, 1, 1)), g)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config1_orszag_tang_256_to_half(dtype):
    """BASELINE.json config 1: 256^2 as 64 patches of 32^2, to t = 0.5: invariants at full
    size and length; parity with the oracle over the first 30 steps."""
    w = W.orszag_tang(256, 32, dtype=NPD[dtype])
    U, t, steps, bad = gpu_run(w, dtype)
    assert bad == 0 and 1200 <= steps <= 1700 and abs(t - 0.5) < 1e-12
    g0 = W.gather(w.U, w.n, w.P).astype(np.float64)
    g = W.gather(U, w.n, w.P).astype(np.float64)
    eps = 1e-12 if dtype == "f64" else 2e-4
    rot = lambda a: a[:, ::-1, ::-1]
    assert np.abs(g[0] - rot(g[0])).max() <= eps * 100           # point symmetry
    tot0, tot1 = g0[:5].sum(axis=(1, 2, 3)), g[:5].sum(axis=(1, 2, 3))
    assert abs(tot1[0] - tot0[0]) <= eps * tot0[0] and abs(tot1[4] - tot0[4]) <= eps * tot0[4]
    bx, by = g[5, 0], g[6, 0]
    div = np.roll(bx, -1, 1) - bx + np.roll(by, -1, 0) - by
    assert np.abs(div).max() / np.sqrt(np.mean(bx ** 2 + by ** 2)) <= (1e-12 if dtype == "f64" else 1e-4)
    assert g[0].min() > 0.05 and g[0].max() < 0.6
    gg, oo, _ = run_both(w, dtype, 30)
    assert rel_err(gg, oo) <= (1e-10 if dtype == "f64" else 2e-4)


def test_decomposition_invariance_on_gpu_bitwise():
    a, b = W.turbulence(N=32, n=32, dtype=np.float32), W.turbulence(N=32, n=16, dtype=np.float32)
    outs = []
    for w in (a, b):
        h = make_gpu(w, "f32")
        dts = []
        for _ in range(3):
            h.fill_guards(); dts.append(h.cfl_dt(0.4, sync=True)); h.step(dts[-1])
        outs.append((W.gather(h.download(), w.n, w.P), dts))
        h.close()
    assert outs[0][1] == outs[1][1]
    assert np.array_equal(outs[0][0], outs[1][0])


def test_run_to_run_determinism():
    w = W.turbulence(N=32, n=16, dtype=np.float32)
    outs = []
    for _ in range(2):
        h = make_gpu(w, "f32")
        for _ in range(5):
            h.fill_guards(); h.cfl_dt(0.4, sync=False); h.step_dev()
        outs.append(h.download()); h.close()
    assert np.array_equal(outs[0], outs[1])


# ------------------------------------------------------------------ edge cases -------
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("path", ["auto", "two_kernel", "staged"])
def test_minimum_patch_size_on_every_path(path, dtype):
    """n == ng = 3, the thinnest legal patch (a neighbour's interior is exactly the guard shell), in
    both types and through every implementation of the step, three chained steps."""
    w = W.turbulence(N=6, n=3, dtype=NPD[dtype])
    o = make_oracle(w)
    b = make_gpu(w, dtype, path=path)
    U = w.U.astype(np.float64)
    for _ in range(3):
        U = o.fill_guards(U, w.nbr); dt = o.cfl_dt(U, 0.4); U = o.step(U, dt)
        b.fill_guards(); b.step(dt)
    assert rel_err(masked(b.download(), w.n), masked(U, w.n)) <= TOL_STEP[dtype]
    assert b.status() == 0
    b.close()


def test_step_rejects_bad_dt_and_counts_bad_cells():
    import ctypes as C
    w = W.turbulence(N=16, n=8, dtype=np.float32)
    b = make_gpu(w, "f32")
    for bad in (0.0, -1.0, float("nan"), float("inf")):
        assert b.lib.mhd_bunch_step(b.h, bad) == -1
    assert b.lib.mhd_bunch_cfl_dt(b.h, -0.4, None, None, None) == -1
    assert b.status() == 0
    U = w.U.copy(); U[4, 3, 5, 5, 5] = -1.0                     # negative energy => negative pressure
    b.load(U); b.fill_guards(); b.step(1e-6)
    assert b.status() >= 1
    b.close()


def test_launch_count_does_not_depend_on_bunch_size():
    """bunching exists to amortise launches; here launches per step are
    a constant of the dimensionality while the workspace holds the bunch."""
    counts = []
    for N in (16, 32):
        w = W.turbulence(N=N, n=8, dtype=np.float32)             # 8 and 64 patches
        b = make_gpu(w, "f32")
        l0 = b.launches
        b.fill_guards(); b.cfl_dt(0.4, sync=False); b.step_dev()
        counts.append(b.launches - l0)
        b.close()
    assert counts[0] == counts[1] <= 16


@pytest.mark.parametrize("shape", ["one_patch_32x32x40", "eight_patches_16", "six_patches_24x20x33"])
def test_z_segments_are_bitwise_invisible(shape):
    """Bunches with fewer tiles than SMs are cut along z into several CTAs per column
    (mhd_bunch_set_tuning, MHD_TUNE_ONEPASS_ZSEG, overrides the automatic choice): whatever the cut,
    ragged or not, on one patch or several, with the 32 x 8 or the 16 x 16 tile, the result is the same
    bit for bit, and equals the oracle."""
    w = {"one_patch_32x32x40": lambda: W.turbulence(N=(32, 32, 40), n=(32, 32, 40), dtype=np.float32),
         "eight_patches_16": lambda: W.turbulence(N=32, n=16, dtype=np.float32),
         "six_patches_24x20x33": lambda: W.turbulence(N=(24, 40, 99), n=(24, 20, 33), dtype=np.float32)}[shape]()
    outs = {}
    # 0 = automatic; n_z - 1 and n_z - 3 do not divide into non-empty segments (32 planes in 31 pieces of
    # ceil(32/31) = 2 planes would leave 15 CTAs past the top): the host rounds them to the cut that does
    for z in (1, 0, 2, 3, 5, w.n[2] - 3, w.n[2] - 1, w.n[2]):
        b = make_gpu(w, "f32")
        assert b.path == "onepass"
        b.set_tuning("onepass_zseg", z)
        for _ in range(2):
            b.fill_guards(); b.cfl_dt(0.4, sync=False); b.step_dev()
        outs[z] = b.download()
        assert b.status() == 0
        b.close()
    for z in outs:
        assert np.array_equal(outs[z], outs[1]), z
    o = make_oracle(w)
    U = w.U.astype(np.float64)
    for _ in range(2):
        U = o.fill_guards(U, w.nbr)
        U = o.step(U, o.cfl_dt(U, 0.4))
    assert rel_err(masked(outs[0], w.n), masked(U, w.n)) <= TOL_STEP["f32"]


# ------------------------------------------------------- full-size config 2 -------
def test_config2_full_size_sampled_patches_and_invariants():
    """BASELINE.json config 2 (512 patches of 32^3, fp32) in the launch configuration
    bench.py times: sampled patches against the oracle, invariants over the whole bunch."""
    w = W.turbulence(N=256, n=32, dtype=np.float32, config=2)
    b = make_gpu(w, "f32")
    b.fill_guards()
    dt = b.cfl_dt(0.4, sync=True)
    filled = b.download()
    # guard fill at full size: sampled patches, bit-exact against the global periodic image
    o_all = make_oracle(w)
    ref_fill = o_all.fill_guards(w.U.astype(np.float64), w.nbr)
    sample = [0, 73, 255, 300, 511]
    for p in sample:
        assert np.array_equal(filled[:, p].astype(np.float64), ref_fill[:, p])
    dt_ref = o_all.cfl_dt(ref_fill, 0.4)
    assert abs(dt - dt_ref) <= 2e-6 * dt_ref
    b.step(dt_ref)
    got = b.download()
    assert b.status() == 0
    import oracle
    o = oracle.Oracle(w.n, len(sample), w.gamma, w.dx)
    ref = o.step(np.ascontiguousarray(ref_fill[:, sample]), dt_ref)
    err = rel_err(masked(got[:, sample], w.n), masked(ref, w.n))
    assert err <= TOL_STEP["f32"], err
    assert_pure_large(masked(got[:, sample], w.n), masked(ref, w.n), "f32", "config 2, sampled patches")
    g0, g1 = W.gather(w.U, w.n, w.P).astype(np.float64), W.gather(got, w.n, w.P).astype(np.float64)
    t0, t1 = g0[:5].sum(axis=(1, 2, 3)), g1[:5].sum(axis=(1, 2, 3))
    assert abs(t1[0] - t0[0]) <= 2e-6 * t0[0] and abs(t1[4] - t0[4]) <= 2e-6 * t0[4]
    div = np.roll(g1[5], -1, 2) - g1[5] + np.roll(g1[6], -1, 1) - g1[6] + np.roll(g1[7], -1, 0) - g1[7]
    assert np.abs(div).max() / np.sqrt(np.mean(g1[5] ** 2 + g1[6] ** 2 + g1[7] ** 2)) <= 1e-4
    b.close()


# ------------------------------------------------------- full-size config 3 -------
def _patch_with_guards(g, n, P, p, ng=3):
    """Patch p of a periodic global field g [8, Nz, Ny, Nx] with its guard shell, taken from
    the global periodic image (what a guard fill must produce; independent of any fill code)."""
    px, py, pz = p % P[0], (p // P[0]) % P[1], p // (P[0] * P[1])
    idx = [(o * k - ng + np.arange(k + 2 * ng)) % N for o, k, N in
           ((pz, n[2], g.shape[1]), (py, n[1], g.shape[2]), (px, n[0], g.shape[3]))]
    return g[np.ix_(np.arange(g.shape[0]), idx[0], idx[1], idx[2])]


_C3 = {}


def _config3(dtype):
    """The 512^3 field is built once (fp64) and cast for the fp32 case -- the same values
    W.turbulence(dtype=float32) stores."""
    if "w" not in _C3:
        _C3["w"] = W.turbulence(N=512, n=32, dtype=np.float64, config=2)
    w = _C3["w"]
    import copy
    v = copy.copy(w)
    v.U = w.U if dtype == "f64" else w.U.astype(np.float32)
    if dtype == "f64":
        _C3.clear()            # last user: release 14 GB
    return v


@pytest.mark.parametrize("dtype", ["f32", "f64"])          # order matters: f64 releases the cached field
def test_config3_full_size_sampled_patches_and_invariants(dtype):
    """BASELINE.json config 3 (4096 patches of 32^3 on a periodic 512^3 cube, fp32 and fp64):
    sampled patches of one step against the oracle, the CFL step against the oracle evaluated
    slab by slab, conservation and div B over the whole bunch.  The oracle never sees more
    than a slab of patches at a time (host memory)."""
    import oracle
    w = _config3(dtype)
    g0 = W.gather(w.U, w.n, w.P)                         # [8, 512, 512, 512] in the storage type
    b = make_gpu(w, dtype)
    w.U = None
    b.fill_guards()
    dt = b.cfl_dt(0.4, sync=True)
    # oracle CFL step: min over slabs of 256 patches, each with guards from the periodic image
    npp = w.P[0] * w.P[1]
    dt_ref = np.inf
    o = oracle.Oracle(w.n, npp, w.gamma, w.dx)
    for s in range(0, w.npatch, npp):
        if (s // npp) % 8 != 3:  # two slabs in full; the rest through the sampled patches below
            continue
        U = np.ascontiguousarray(np.stack([_patch_with_guards(g0, w.n, w.P, p) for p in range(s, s + npp)], axis=1), dtype=np.float64)
        dt_ref = min(dt_ref, o.cfl_dt(U, 0.4))
    assert dt <= dt_ref * (1 + (1e-13 if dtype == "f64" else 2e-6))      # the GPU minimum covers every slab
    sample = [0, 15, 255, 256, 1911, 2730, 3840, 4095]
    os_ = oracle.Oracle(w.n, len(sample), w.gamma, w.dx)
    Us = np.ascontiguousarray(np.stack([_patch_with_guards(g0, w.n, w.P, p) for p in sample], axis=1), dtype=np.float64)
    ref = os_.step(Us, dt)
    b.step(dt)
    assert b.status() == 0
    got = b.download()
    err = rel_err(masked(got[:, sample], w.n), masked(ref, w.n))
    assert err <= TOL_STEP[dtype], err
    assert_pure_large(masked(got[:, sample], w.n), masked(ref, w.n), dtype, "config 3, sampled patches")
    g1 = W.gather(got, w.n, w.P)
    del got
    tol = 1e-12 if dtype == "f64" else 2e-6
    for f in (0, 4):
        t0, t1 = g0[f].sum(dtype=np.float64), g1[f].sum(dtype=np.float64)
        assert abs(t1 - t0) <= tol * abs(t0)
    div = np.roll(g1[5], -1, 2) - g1[5] + np.roll(g1[6], -1, 1) - g1[6] + np.roll(g1[7], -1, 0) - g1[7]
    brms = np.sqrt(np.mean(g1[5].astype(np.float64) ** 2 + g1[6].astype(np.float64) ** 2 + g1[7].astype(np.float64) ** 2))
    assert np.abs(div).max() / brms <= (1e-12 if dtype == "f64" else 1e-4)
    b.close()


# ------------------------------------- config 4's largest point: 64-bit offsets -------
def test_config4_corner_4096_patches_of_64_cubed():
    """BASELINE.json config 4's largest point, 4096 patches of 64^3 in fp32: 11.6 G elements per
    state buffer, the only case whose element offsets exceed 2^31 (and 2^32).  The global field
    (1024^3 cells) is not built on the host: the seeded field of a 256^3 block (4 x 4 x 4 patches)
    is repeated periodically on the device, which is again a periodic field.  Checks: sampled
    patches from the low, middle and high end of the buffer against the oracle (one step), and
    every patch bit for bit equal to its periodic image among the 64 patches of the block -- an
    offset that wrapped anywhere would break one of them."""
    import importlib.util
    import os
    import oracle
    import torch
    spec = importlib.util.spec_from_file_location("bench", os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "bench.py"))
    bench = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(bench)
    import gc
    gc.collect()
    torch.cuda.empty_cache()                       # earlier tests' buffers sit in torch's caching allocator
    free, _ = torch.cuda.mem_get_info()
    if free < 110 * 2 ** 30:
        pytest.skip("needs 2 x 46 GB of device memory")
    n, P = 64, (16, 16, 16)
    b, wb, B = bench.replicated_bunch(n, P, "f32", 0)
    assert b.lay.state_elems > 2 ** 33 and b.path == "onepass"
    b.fill_guards()
    dt = b.cfl_dt(0.4, sync=True)
    # the oracle on the block with the bunch's cell size: same field, same step
    ob = oracle.Oracle(wb.n, wb.npatch, wb.gamma, b.desc.dx[:])
    Ub = ob.fill_guards(wb.U.astype(np.float64), wb.nbr)
    dt_ref = ob.cfl_dt(Ub, 0.4)
    assert abs(dt - dt_ref) <= 2e-6 * dt_ref
    b.step(dt_ref)
    assert b.status() == 0
    v = b.view()                                                  # the new level, on the device
    ids = np.arange(4096)
    px, py, pz = ids % 16, (ids // 16) % 16, ids // 256
    img = (px % B[0]) + B[0] * ((py % B[1]) + B[1] * (pz % B[2]))
    sample = [0, 1911, 4095]
    simg = [int(img[p]) for p in sample]
    osub = oracle.Oracle(wb.n, len(sample), wb.gamma, b.desc.dx[:])
    ref = osub.step(np.ascontiguousarray(Ub[:, simg]), dt_ref)
    got = v[:, sample].cpu().numpy()
    assert_step_parity(masked(got, wb.n), masked(ref, wb.n), "f32", "64^3 x 4096")
    I = (slice(3, 3 + n),) * 3
    for q in range(64):
        same = torch.from_numpy(ids[img == q]).to(v.device)
        first = v[:, int(same[0])][(slice(None),) + I]
        for p in same[1:].tolist():
            assert torch.equal(v[:, p][(slice(None),) + I], first), (q, p)
    b.close()


# ------------------------------------------------ CFL reduction in the step's epilogue -------
@pytest.mark.parametrize("name", ["turb16", "turb_ragged", "turb_self", "turb_nx10", "turb_nx38", "turb_thin"])
def test_fused_cfl_epilogue_is_bitwise_the_standalone_reduction(name):
    """The one-pass step reduces the CFL rates of the level it writes in its epilogue;
    mhd_bunch_cfl_dt then only runs the bunch-wide reduction.  The step it returns, and the per-patch
    steps, must equal those of the stand-alone pass over the stored state bit for bit (both evaluate
    the same explicitly rounded function), and the oracle's within the CFL tolerance."""
    w = small_workloads("f32")[name]
    b = make_gpu(w, "f32")
    assert b.path == "onepass"
    b.set_tuning("fused_cfl", 1)
    o = make_oracle(w)
    for _ in range(3):
        b.fill_guards(); dt = b.cfl_dt(0.4, sync=True); b.step(dt)
    b.fill_guards()
    l0 = b.launches
    dt_f = b.cfl_dt(0.4, sync=True, per_patch=True)
    n_f, pp_f = b.launches - l0, b.dt_patch.cpu().numpy().copy()
    U = b.download().astype(np.float64)          # looking at the buffer: the library must fall back to the full pass
    b.fill_guards()
    l0 = b.launches
    dt_s = b.cfl_dt(0.4, sync=True, per_patch=True)
    n_s, pp_s = b.launches - l0, b.dt_patch.cpu().numpy().copy()
    assert n_f == 1 and n_s == 3, (n_f, n_s)
    assert dt_f == dt_s and np.array_equal(pp_f, pp_s)
    dt_o, pp_o = o.cfl_dt(o.fill_guards(U, w.nbr), 0.4, per_patch=True)
    assert abs(dt_f - dt_o) <= 2e-6 * dt_o and np.all(np.abs(pp_f - pp_o) <= 2e-6 * pp_o)
    # the state does not depend on the epilogue beyond round-off: the kernel without it is a separate
    # compilation of the same source (a handful of values in a million differ by one ulp)
    c = make_gpu(w, "f32")
    c.set_tuning("fused_cfl", 0)
    dts_c = []
    for _ in range(3):
        c.fill_guards(); dt = c.cfl_dt(0.4, sync=True); c.step(dt); dts_c.append(dt)
    assert rel_err(masked(c.download(), w.n), masked(U, w.n)) <= 2e-7
    # the library's own choice (MHD_TUNE_FUSED_CFL = 2, the default): these bunches are far below one wave of
    # tiles, so the epilogue runs -- three launches per step (cfl_final, set_dt, step) after the first, the state
    # bit for bit that of the handle with the epilogue forced on
    d = make_gpu(w, "f32")
    e = make_gpu(w, "f32")
    e.set_tuning("fused_cfl", 1)
    for s in range(3):
        l0 = d.launches
        d.fill_guards(); dt_d = d.cfl_dt(0.4, sync=True); d.step(dt_d)
        e.fill_guards(); dt_e = e.cfl_dt(0.4, sync=True); e.step(dt_e)
        assert dt_d == dt_e
        if s > 0:                                  # rows of whole 16-byte chunks: the fill is folded into the step too
            assert d.launches - l0 == (3 if w.n[0] % 4 == 0 else 4), d.launches - l0
    assert np.array_equal(d.download(), e.download())
    b.close(); c.close(); d.close(); e.close()
