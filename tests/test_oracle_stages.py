"""Pins of the oracle's stages O1-O5, O8, O9 against closed forms and invariants
(DESIGN.md "What pins each part").  Expected values are computed here from the paper's
printed equations or from the global-grid picture, never by calling the oracle twice."""
import numpy as np
import pytest

import oracle
from paper_2508_09568_b200 import workloads as W

NG = 3


def dense_patch_from_prims(rho, vel, p, bf, gamma):
    """Treat a padded patch as a little global grid: U[8,1,mz,my,mx] with every cell and
    lower face set (bf have one extra face in their normal direction)."""
    cons = W.conserved_from_primitive(rho, vel, p, bf, gamma)
    mz, my, mx = rho.shape
    U = np.zeros((8, 1, mz, my, mx))
    U[:5, 0] = cons
    U[5, 0] = bf[0][:, :, :mx]
    U[6, 0] = bf[1][:, :my, :]
    U[7, 0] = bf[2][:mz, :, :]
    return U


def smooth_patch(n, seed, gamma=5 / 3, linear=False):
    """Random smooth (or exactly linear) primitive data on a padded patch."""
    rng = np.random.default_rng(seed)
    mx, my, mz = W.padded(n)
    z, y, x = np.meshgrid(np.arange(mz + 1), np.arange(my + 1), np.arange(mx + 1), indexing="ij")
    def fld(base, amp, stag=(0, 0, 0)):
        a = rng.normal(size=3) * amp
        xs, ys, zs = x + 0.5 * (1 - stag[0]), y + 0.5 * (1 - stag[1]), z + 0.5 * (1 - stag[2])
        if linear:
            return base + a[0] * xs + a[1] * ys + a[2] * zs
        return base + amp * np.sin(0.3 * xs + a[0]) * np.cos(0.25 * ys + a[1]) * np.cos(0.2 * zs + a[2])
    C = (slice(0, mz), slice(0, my), slice(0, mx))
    rho = fld(2.0, 0.01 if linear else 0.3)[C]
    p = fld(1.5, 0.01 if linear else 0.2)[C]
    vel = [fld(0.3, 0.01 if linear else 0.4)[C] for _ in range(3)]
    bx = fld(0.5, 0.01 if linear else 0.3, (1, 0, 0))[:mz, :my, :mx + 1]
    by = fld(-0.2, 0.01 if linear else 0.3, (0, 1, 0))[:mz, :my + 1, :mx]
    bz = fld(0.1, 0.01 if linear else 0.3, (0, 0, 1))[:mz + 1, :my, :mx]
    if n[1] == 1:
        by = np.concatenate([by[:, :1], by[:, :1]], axis=1)
    if n[2] == 1:
        bz = np.concatenate([bz[:1], bz[:1]], axis=0)
    return rho, vel, p, (bx, by, bz)


def rng_cells(n, lo, hi):
    """index slices (z,y,x) of cells [-lo, n-1+hi] in active dims"""
    return tuple(slice(NG - lo, NG + k + hi) if k > 1 else slice(0, 1) for k in (n[2], n[1], n[0]))


# ------------------------------------------------------------------------- O1 -----
@pytest.mark.parametrize("n,P,periodic", [
    ((4, 5, 6), (2, 2, 2), (True, True, True)),
    ((4, 5, 6), (2, 1, 3), (False, True, True)),
    ((4, 3, 1), (3, 2, 1), (True, False, True)),
    ((5, 1, 1), (4, 1, 1), (False, True, True)),
    ((3, 3, 3), (1, 1, 1), (True, True, True)),      # a patch that is its own neighbour
])
def test_guard_fill_index_encoded(n, P, periodic):
    nbr = W.neighbour_table(P, periodic)
    npatch = P[0] * P[1] * P[2]
    o = oracle.Oracle(n, npatch, 5 / 3, (1, 1, 1))
    N = [n[d] * P[d] for d in range(3)]
    U = np.full(o.shape, -1.0)
    g = [NG if k > 1 else 0 for k in n]
    def gid(f, X, Y, Z):
        return f * 1e7 + (Z * N[1] + Y) * N[0] + X
    for p in range(npatch):
        px, py, pz = p % P[0], (p // P[0]) % P[1], p // (P[0] * P[1])
        for k in range(n[2]):
            for j in range(n[1]):
                for i in range(n[0]):
                    for f in range(8):
                        U[f, p, k + g[2], j + g[1], i + g[0]] = gid(f, px * n[0] + i, py * n[1] + j, pz * n[2] + k)
    sentinel = U.copy()
    o.fill_guards(U, nbr)
    for p in range(npatch):
        pc = (p % P[0], (p // P[0]) % P[1], p // (P[0] * P[1]))
        for k in range(-g[2], n[2] + g[2]):
            for j in range(-g[1], n[1] + g[1]):
                for i in range(-g[0], n[0] + g[0]):
                    loc = (i, j, k)
                    glob = [pc[d] * n[d] + loc[d] for d in range(3)]
                    inside = all(periodic[d] or 0 <= glob[d] < N[d] for d in range(3))
                    if inside:
                        src = [glob[d] % N[d] for d in range(3)]
                    else:   # zero-gradient: nearest interior cell of the patch itself
                        src = [pc[d] * n[d] + min(max(loc[d], 0), n[d] - 1) for d in range(3)]
                    for f in range(8):
                        got = U[f, p, k + g[2], j + g[1], i + g[0]]
                        exp = gid(f, *src)
                        if not inside and f >= 5:
                            a = f - 5
                            others = [d for d in range(3) if d != a]
                            if loc[a] == n[a] and n[a] > 1 and all(0 <= loc[d] < n[d] for d in others):
                                exp = sentinel[f, p, k + g[2], j + g[1], i + g[0]]   # closing face untouched
                        assert got == exp, (p, loc, f, got, exp)


# ------------------------------------------------------------------------- O2 -----
@pytest.mark.parametrize("n", [(6, 5, 4), (6, 5, 1), (7, 1, 1)])
def test_primitives_round_trip(n):
    gamma = 1.4
    rho, vel, p, bf = smooth_patch(n, 3, gamma)
    U = dense_patch_from_prims(rho, vel, p, bf, gamma)
    o = oracle.Oracle(n, 1, gamma, (0.1, 0.2, 0.3))
    st = o.stages(U, 0, 0.01)
    C = rng_cells(n, 2, 2)
    for f, ref in enumerate([rho, vel[0], vel[1], vel[2], p]):
        assert np.allclose(st["q"][f][C], ref[C], rtol=1e-13, atol=1e-13)
    bc = [0.5 * (bf[0][:, :, :-1] + bf[0][:, :, 1:]), 0.5 * (bf[1][:, :-1] + bf[1][:, 1:]), 0.5 * (bf[2][:-1] + bf[2][1:])]
    for a in range(3):
        assert np.array_equal(st["q"][5 + a][C], bc[a][C])


# ------------------------------------------------------------------------- O3 -----
@pytest.mark.parametrize("limiter", [1, 2])
@pytest.mark.parametrize("n", [(6, 5, 4), (6, 5, 1)])
def test_slopes_exact_for_linear_data(n, limiter):
    gamma = 1.4
    rho, vel, p, bf = smooth_patch(n, 4, gamma, linear=True)
    U = dense_patch_from_prims(rho, vel, p, bf, gamma)
    o = oracle.Oracle(n, 1, gamma, (0.1, 0.2, 0.3), limiter=limiter)
    st = o.stages(U, 0, 0.01)
    C = rng_cells(n, 1, 1)
    q = st["q"]
    dq = st["dq"].reshape(3, 8, *q.shape[1:])
    for d in range(3):
        if n[d] == 1:
            assert not dq[d].any()
            continue
        ax = 2 - d
        for f in range(8):
            if f == 5 + d:
                assert not dq[d][f].any()
                continue
            ref = np.roll(q[f], -1, axis=ax) - q[f]           # forward difference = the exact slope
            # p is not exactly linear (E is built from products), so allow curvature-level slack
            tol = 1e-3 if f == 4 else 1e-12
            assert np.allclose(dq[d][f][C], ref[C], rtol=tol, atol=tol * 1e-2), (d, f)
    # face-field transverse slopes: exact forward differences of the face values
    names = [(0, 1), (0, 2), (1, 0), (1, 2), (2, 0), (2, 1)]
    for idx, (a, t) in enumerate(names):
        if n[t] == 1:
            assert not st["dbf"][idx].any()
            continue
        b = U[5 + a, 0]
        ref = np.roll(b, -1, axis=2 - t) - b
        assert np.allclose(st["dbf"][idx][C], ref[C], rtol=1e-12, atol=1e-14)


def test_slopes_vanish_at_extrema():
    n = (8, 1, 1)
    mx = n[0] + 2 * NG
    rho = np.ones((1, 1, mx)); rho[0, 0, 6] = 3.0            # a spike
    vel = [np.zeros((1, 1, mx))] * 3
    p = np.ones((1, 1, mx))
    bf = (np.zeros((1, 1, mx + 1)), np.zeros((1, 2, mx)), np.zeros((2, 1, mx)))
    U = dense_patch_from_prims(rho, vel, p, bf, 1.4)
    st = oracle.Oracle(n, 1, 1.4, (1, 1, 1)).stages(U, 0, 0.0)
    assert not st["dq"][0].any()                              # spike and flat neighbours: all slopes 0


# ------------------------------------------------------------------ O4a, O4b -----
def test_predictor_emf_uniform_state_is_u_cross_b():
    n = (5, 4, 6)
    mx, my, mz = W.padded(n)
    u, v, w, bx, by, bz = 0.3, -0.7, 1.1, 0.5, 0.25, -0.8
    one = np.ones((mz, my, mx))
    bf = (bx * np.ones((mz, my, mx + 1)), by * np.ones((mz, my + 1, mx)), bz * np.ones((mz + 1, my, mx)))
    U = dense_patch_from_prims(2 * one, [u * one, v * one, w * one], one, bf, 1.4)
    st = oracle.Oracle(n, 1, 1.4, (1, 1, 1)).stages(U, 0, 0.1)
    C = rng_cells(n, 1, 2)
    ref = [v * bz - w * by, w * bx - u * bz, u * by - v * bx]      # (u x B), Eq. 7 sign
    for a in range(3):
        assert np.allclose(st["e0"][a][C], ref[a], rtol=1e-15, atol=0)
    # and the half-step faces do not move
    assert np.array_equal(st["bh"][0][rng_cells(n, 1, 1)], bx * one[rng_cells(n, 1, 1)])


def test_predictor_emf_eq7_to_11_literal():
    """Eq. 7-11 typed from the paper, on random data, z-edges."""
    n = (5, 4, 3)
    rho, vel, p, bf = smooth_patch(n, 5)
    U = dense_patch_from_prims(rho, vel, p, bf, 5 / 3)
    st = oracle.Oracle(n, 1, 5 / 3, (1, 1, 1)).stages(U, 0, 0.1)
    vx, vy = st["q"][1], st["q"][2]
    Bx, By = U[5, 0], U[6, 0]
    for (k, j, i) in [(3, 3, 3), (4, 5, 6), (2, 2, 2), (5, 7, 9)]:
        vxb = 0.25 * (vx[k, j, i] + vx[k, j - 1, i] + vx[k, j, i - 1] + vx[k, j - 1, i - 1])
        vyb = 0.25 * (vy[k, j, i] + vy[k, j - 1, i] + vy[k, j, i - 1] + vy[k, j - 1, i - 1])
        bxb = 0.5 * (Bx[k, j, i] + Bx[k, j - 1, i])
        byb = 0.5 * (By[k, j, i] + By[k, j, i - 1])
        assert np.isclose(st["e0"][2][k, j, i], vxb * byb - vyb * bxb, rtol=1e-14, atol=1e-16)


@pytest.mark.parametrize("n", [(6, 5, 4), (6, 5, 1)])
def test_half_step_faces_keep_divergence(n):
    rho, vel, p, bf = smooth_patch(n, 6)
    U = dense_patch_from_prims(rho, vel, p, bf, 5 / 3)
    dx = (0.1, 0.2, 0.3)
    st = oracle.Oracle(n, 1, 5 / 3, dx).stages(U, 0, 0.05)
    def div(b):
        d = 0
        for a in range(3):
            if n[a] > 1:
                d = d + (np.roll(b[a], -1, axis=2 - a) - b[a]) / dx[a]
        return d
    C = rng_cells(n, 1, 0)      # cells whose six faces all carry half-step values
    d0 = div([U[5, 0], U[6, 0], U[7, 0]])[C]
    d1 = div(st["bh"])[C]
    assert np.abs(d1 - d0).max() <= 1e-13 * np.abs(U[5:8]).max() / min(dx)
    assert np.abs(st["bh"][0] - U[5, 0])[C].max() > 1e-4   # the faces did move


def test_eq12_literal_for_half_step_bx():
    n = (5, 4, 3)
    rho, vel, p, bf = smooth_patch(n, 7)
    U = dense_patch_from_prims(rho, vel, p, bf, 5 / 3)
    dx = (0.1, 0.2, 0.3); dt = 0.04
    st = oracle.Oracle(n, 1, 5 / 3, dx).stages(U, 0, dt)
    ez, ey = st["e0"][2], st["e0"][1]
    for (k, j, i) in [(3, 3, 3), (4, 5, 6), (2, 2, 9)]:
        ref = U[5, 0, k, j, i] + (ez[k, j + 1, i] - ez[k, j, i]) / dx[1] * (dt / 2) \
            - (ey[k + 1, j, i] - ey[k, j, i]) / dx[2] * (dt / 2)           # Eq. 12 with dt/2
        assert np.isclose(st["bh"][0][k, j, i], ref, rtol=1e-14)


# ------------------------------------------------------------------------ O4c -----
def test_hydro_predictor_advects_smooth_density():
    """Uniform flow, uniform p, B=0: rho^h = rho - dt/2 u.grad(rho) + O(dx^2)."""
    errs = []
    for N in (32, 64):
        n = (N, N, 1)
        mx, my, mz = W.padded(n)
        h = 1.0 / N
        xc = (np.arange(mx) - NG + 0.5) * h
        yc = (np.arange(my) - NG + 0.5) * h
        Y, X = np.meshgrid(yc, xc, indexing="ij")
        rho = (1 + 0.2 * np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Y))[None]
        u0, v0 = 0.7, -0.4
        one = np.ones_like(rho)
        bf = (np.zeros((1, my, mx + 1)), np.zeros((1, my + 1, mx)), np.zeros((2, my, mx)))
        U = dense_patch_from_prims(rho, [u0 * one, v0 * one, 0 * one], one, bf, 1.4)
        dt = 0.2 * h
        st = oracle.Oracle(n, 1, 1.4, (h, h, 1.0), limiter=2).stages(U, 0, dt)
        gx = 0.2 * 2 * np.pi * np.cos(2 * np.pi * X) * np.cos(2 * np.pi * Y)
        gy = -0.2 * 2 * np.pi * np.sin(2 * np.pi * X) * np.sin(2 * np.pi * Y)
        ref = rho[0] - 0.5 * dt * (u0 * gx + v0 * gy)
        C = rng_cells(n, 1, 1)[1:]
        mask = (np.abs(np.cos(2 * np.pi * X)) > 0.3) & (np.abs(np.sin(2 * np.pi * Y)) > 0.3) & \
               (np.abs(np.sin(2 * np.pi * X)) > 0.3) & (np.abs(np.cos(2 * np.pi * Y)) > 0.3)
        err = np.abs(st["qh"][0][0] - ref)[C][mask[C]].max() / dt
        errs.append(err)
        # velocity and pressure untouched by a uniform flow without field
        assert np.allclose(st["qh"][1][0][C], u0, rtol=1e-13) and np.allclose(st["qh"][4][0][C], 1.0, rtol=1e-13)
    assert errs[1] < errs[0] / 3.0, errs             # second order in dx


def test_hydro_predictor_uniform_compression_closed_form():
    """rho, p uniform, u = a x, v = b y, w = c z (exactly linear => exact slopes), B = 0:
    rho^h = rho (1 - dt/2 (a+b+c)),  p^h = p (1 - dt/2 gamma (a+b+c)),
    u^h = u (1 - dt/2 a)   [Eq. 1-4 in primitive form, PAPER.md L110-114]."""
    n = (6, 5, 4)
    mx, my, mz = W.padded(n)
    dx = (0.1, 0.2, 0.3)
    a, b, c = 0.7, -0.3, 0.45
    z, y, x = np.meshgrid((np.arange(mz) - NG + 0.5) * dx[2], (np.arange(my) - NG + 0.5) * dx[1],
                          (np.arange(mx) - NG + 0.5) * dx[0], indexing="ij")
    one = np.ones((mz, my, mx))
    bf = (np.zeros((mz, my, mx + 1)), np.zeros((mz, my + 1, mx)), np.zeros((mz + 1, my, mx)))
    gamma, dt = 1.4, 0.02
    U = dense_patch_from_prims(2 * one, [a * x, b * y, c * z], 1.5 * one, bf, gamma)
    for lim in (1, 2):
        st = oracle.Oracle(n, 1, gamma, dx, limiter=lim).stages(U, 0, dt)
        C = rng_cells(n, 1, 1)
        assert np.allclose(st["qh"][0][C], 2 * (1 - 0.5 * dt * (a + b + c)), rtol=1e-13)
        assert np.allclose(st["qh"][4][C], 1.5 * (1 - 0.5 * dt * gamma * (a + b + c)), rtol=1e-12)
        assert np.allclose(st["qh"][1][C], (a * x * (1 - 0.5 * dt * a))[C], rtol=1e-12, atol=1e-14)
        assert np.allclose(st["qh"][2][C], (b * y * (1 - 0.5 * dt * b))[C], rtol=1e-12, atol=1e-14)
        assert np.allclose(st["qh"][3][C], (c * z * (1 - 0.5 * dt * c))[C], rtol=1e-12, atol=1e-14)


def test_hydro_predictor_magnetic_force_sign():
    """Static gas, p uniform, By(x) only: du/dt = -(1/rho) d/dx(By^2/2) (magnetic pressure
    pushes towards weaker field), dv/dt = 0; with Bx uniform added: dv/dt = +(Bx/rho) dBy/dx
    (tension)."""
    N = 64
    n = (N, 1, 1)
    mx = N + 2 * NG
    h = 1.0 / N
    xc = (np.arange(mx) - NG + 0.5) * h
    By = (1.0 + 0.3 * np.sin(2 * np.pi * xc)).reshape(1, 1, mx)
    dBy = (0.3 * 2 * np.pi * np.cos(2 * np.pi * xc)).reshape(1, 1, mx)
    one = np.ones((1, 1, mx))
    bxv = 0.6
    bf = (bxv * np.ones((1, 1, mx + 1)), np.concatenate([By, By], axis=1), np.zeros((2, 1, mx)))
    U = dense_patch_from_prims(2 * one, [0 * one] * 3, one, bf, 1.4)
    dt = 0.1 * h
    st = oracle.Oracle(n, 1, 1.4, (h, 1, 1), limiter=2).stages(U, 0, dt)
    C = (0, 0, slice(NG - 1, NG + N + 1))
    mask = np.abs(np.cos(2 * np.pi * xc[C[2]])) > 0.3
    du = st["qh"][1][C] / (0.5 * dt)
    dv = st["qh"][2][C] / (0.5 * dt)
    assert np.allclose(du[mask], (-(By * dBy) / 2.0)[C][mask], rtol=0, atol=0.02)
    assert np.allclose(dv[mask], (bxv * dBy / 2.0)[C][mask], rtol=0, atol=0.02)


# ------------------------------------------------------------------------- O5 -----
def test_face_states_feed_hlld_as_described():
    """The x-face flux of the step equals orc_hlld applied to q^h +- dq/2 typed here
    from O5, with the half-step face field as the normal component."""
    n = (5, 4, 3)
    rho, vel, p, bf = smooth_patch(n, 8)
    U = dense_patch_from_prims(rho, vel, p, bf, 5 / 3)
    o = oracle.Oracle(n, 1, 5 / 3, (0.1, 0.2, 0.3))
    st = o.stages(U, 0, 0.02)
    qh = st["qh"]; dq = st["dq"].reshape(3, 8, *qh.shape[1:]); fl = st["flux"].reshape(3, 5, *qh.shape[1:])
    for (k, j, i) in [(3, 3, 3), (4, 5, 6), (5, 6, 8)]:
        comp = [0, 1, 2, 3, 4, 6, 7]
        L = [qh[f][k, j, i - 1] + 0.5 * dq[0][f][k, j, i - 1] for f in comp]
        R = [qh[f][k, j, i] - 0.5 * dq[0][f][k, j, i] for f in comp]
        F = oracle.hlld(5 / 3, L, R, st["bh"][0][k, j, i])
        assert np.array_equal(fl[0][:, k, j, i], F[:5])
        # y-face: rotate (v,w,u) / (Bz,Bx); x must be interior for a y-face
        i = min(i, NG + n[0] - 1)
        comp = [0, 2, 3, 1, 4, 7, 5]
        L = [qh[f][k, j - 1, i] + 0.5 * dq[1][f][k, j - 1, i] for f in comp]
        R = [qh[f][k, j, i] - 0.5 * dq[1][f][k, j, i] for f in comp]
        F = oracle.hlld(5 / 3, L, R, st["bh"][1][k, j, i])
        assert np.array_equal(fl[1][[0, 2, 3, 1, 4], k, j, i], F[:5])
        # z-face: rotate (w,u,v) / (Bx,By)
        comp = [0, 3, 1, 2, 4, 5, 6]
        L = [qh[f][k - 1, j, i] + 0.5 * dq[2][f][k - 1, j, i] for f in comp]
        R = [qh[f][k, j, i] - 0.5 * dq[2][f][k, j, i] for f in comp]
        F = oracle.hlld(5 / 3, L, R, st["bh"][2][k, j, i])
        assert np.array_equal(fl[2][[0, 3, 1, 2, 4], k, j, i], F[:5])


def test_corner_states_feed_emf2d_as_described():
    n = (5, 4, 3)
    rho, vel, p, bf = smooth_patch(n, 9)
    U = dense_patch_from_prims(rho, vel, p, bf, 5 / 3)
    o = oracle.Oracle(n, 1, 5 / 3, (0.1, 0.2, 0.3))
    st = o.stages(U, 0, 0.02)
    qh = st["qh"]; dq = st["dq"].reshape(3, 8, *qh.shape[1:]); bh = st["bh"]; dbf = st["dbf"]
    comp = [0, 1, 2, 3, 4, 7]
    for (k, j, i) in [(3, 3, 3), (4, 5, 6), (5, 6, 8)]:
        cells = [(k, j - 1, i - 1, +1, +1), (k, j - 1, i, -1, +1), (k, j, i - 1, +1, -1), (k, j, i, -1, -1)]
        c = [[qh[f][kk, jj, ii] + sx * 0.5 * dq[0][f][kk, jj, ii] + sy * 0.5 * dq[1][f][kk, jj, ii] for f in comp]
             for (kk, jj, ii, sx, sy) in cells]
        AS = bh[0][k, j - 1, i] + 0.5 * dbf[0][k, j - 1, i]
        AN = bh[0][k, j, i] - 0.5 * dbf[0][k, j, i]
        BW = bh[1][k, j, i - 1] + 0.5 * dbf[2][k, j, i - 1]
        BE = bh[1][k, j, i] - 0.5 * dbf[2][k, j, i]
        assert st["emf"][2][k, j, i] == oracle.emf2d(5 / 3, 0, c, AS, AN, BW, BE)


# ------------------------------------------------------------------------- O8 -----
def _small_turb(N=16, n=8, seed=()):
    return W.turbulence(N=N, n=n, dtype=np.float64, config=2, seed_extra=seed)


def test_update_conserves_and_keeps_divb():
    w = _small_turb()
    o = oracle.Oracle(w.n, w.npatch, w.gamma, w.dx)
    U = w.U.copy()
    vol = np.prod(w.dx)
    tot0 = W.gather(U, w.n, w.P)[:5].sum(axis=(1, 2, 3))
    dx = w.dx[0]
    def maxdiv(U):
        g = W.gather(U, w.n, w.P)
        d = (np.roll(g[5], -1, 2) - g[5] + np.roll(g[6], -1, 1) - g[6] + np.roll(g[7], -1, 0) - g[7])
        return np.abs(d).max() / np.sqrt(np.mean(g[5] ** 2 + g[6] ** 2 + g[7] ** 2))
    assert maxdiv(U) < 1e-13
    for _ in range(5):
        o.fill_guards(U, w.nbr)
        dt = o.cfl_dt(U, 0.4)
        U = o.step(U, dt)
    g = W.gather(U, w.n, w.P)
    tot1 = g[:5].sum(axis=(1, 2, 3))
    scale = np.array([tot0[0], np.abs(g[1:4]).sum(), np.abs(g[1:4]).sum(), np.abs(g[1:4]).sum(), tot0[4]])
    assert np.all(np.abs(tot1 - tot0) <= 1e-13 * scale), (tot1 - tot0) / scale
    assert maxdiv(U) < 2e-13
    assert np.abs(g[0] - W.gather(w.U, w.n, w.P)[0]).max() > 1e-3      # something happened
    assert vol > 0


def test_closing_face_equals_neighbour_face_bitwise():
    w = _small_turb()
    o = oracle.Oracle(w.n, w.npatch, w.gamma, w.dx)
    U = w.U.copy()
    o.fill_guards(U, w.nbr)
    U1 = o.step(U, o.cfl_dt(U, 0.4))
    n = w.n[0]
    I = slice(NG, NG + n)
    for p in range(w.npatch):
        qx, qy, qz = w.nbr[p, 13 + 1], w.nbr[p, 13 + 3], w.nbr[p, 13 + 9]
        assert np.array_equal(U1[5, p, I, I, NG + n], U1[5, qx, I, I, NG])
        assert np.array_equal(U1[6, p, I, NG + n, I], U1[6, qy, I, NG, I])
        assert np.array_equal(U1[7, p, NG + n, I, I], U1[7, qz, NG, I, I])
    assert not np.array_equal(U1[5, 0, I, I, NG + n], U[5, 0, I, I, NG + n])


def test_uniform_moving_magnetised_state_is_preserved_bitwise():
    n = (6, 5, 4)
    mx, my, mz = W.padded(n)
    one = np.ones((mz, my, mx))
    bf = (0.5 * np.ones((mz, my, mx + 1)), 0.25 * np.ones((mz, my + 1, mx)), -0.8 * np.ones((mz + 1, my, mx)))
    U = dense_patch_from_prims(2 * one, [0.3 * one, -0.7 * one, 1.1 * one], 1.5 * one, bf, 1.4)
    o = oracle.Oracle(n, 1, 1.4, (0.1, 0.2, 0.3))
    U1 = o.step(U, 0.01)
    assert np.array_equal(U1, U)


# ------------------------------------------------------------------------- O9 -----
def test_cfl_uniform_closed_form_and_planted_cell():
    n = (6, 5, 4)
    mx, my, mz = W.padded(n)
    one = np.ones((mz, my, mx))
    rho0, p0, u, v, w_ = 2.0, 1.5, 0.3, -0.7, 1.1
    bx, by, bz = 0.5, 0.25, -0.8
    bf = (bx * np.ones((mz, my, mx + 1)), by * np.ones((mz, my + 1, mx)), bz * np.ones((mz + 1, my, mx)))
    gamma = 1.4
    dx = (0.1, 0.2, 0.3)
    U1 = dense_patch_from_prims(rho0 * one, [u * one, v * one, w_ * one], p0 * one, bf, gamma)
    U = np.concatenate([U1, U1, U1], axis=1)
    def cf(bn):
        b2 = bx * bx + by * by + bz * bz
        s = gamma * p0 + b2
        return np.sqrt((s + np.sqrt(s * s - 4 * gamma * p0 * bn * bn)) / (2 * rho0))
    rate = (abs(u) + cf(bx)) / dx[0] + (abs(v) + cf(by)) / dx[1] + (abs(w_) + cf(bz)) / dx[2]
    o = oracle.Oracle(n, 3, gamma, dx)
    dt, pp = o.cfl_dt(U, 0.4, per_patch=True)
    assert np.isclose(dt, 0.4 / rate, rtol=1e-14) and np.allclose(pp, 0.4 / rate, rtol=1e-14)
    # plant one fast interior cell in patch 1 (momentum x10); guards must not matter
    U[1, 1, NG + 2, NG + 1, NG + 3] *= 10
    U[4, 1, NG + 2, NG + 1, NG + 3] += 0.5 * rho0 * (100 - 1) * u * u
    U[1, 2, 0, 0, 0] *= 1000                                   # a guard cell: ignored
    dt2, pp2 = o.cfl_dt(U, 0.4, per_patch=True)
    rate2 = rate + (10 * abs(u) - abs(u)) / dx[0]
    assert np.isclose(pp2[1], 0.4 / rate2, rtol=1e-12) and dt2 == pp2[1]
    assert pp2[0] == pp[0] and pp2[2] == pp[2]


def test_cfl_skips_collapsed_dimensions():
    w = W.sod(64, 2)
    o = oracle.Oracle(w.n, w.npatch, w.gamma, w.dx)
    dt = o.cfl_dt(w.U, 0.4)
    assert np.isclose(dt, 0.4 * (1 / 64) / np.sqrt(1.4), rtol=1e-14)   # c = sqrt(gamma p/rho) = sqrt(1.4) on the left


def test_openmp_build_of_the_oracle_is_bitwise_the_plain_build():
    """bench.py's all-cores leg uses the same source built with -fopenmp: same bits."""
    w = W.turbulence(N=16, n=8, dtype=np.float64)
    res = {}
    for key in ("f64", "f64_omp"):
        o = oracle.Oracle(w.n, w.npatch, w.gamma, w.dx, dtype=key)
        U = o.fill_guards(w.U.copy(), w.nbr)
        dt, pp = o.cfl_dt(U, 0.4, per_patch=True)
        res[key] = (dt, pp, o.step(U, dt))
    assert res["f64"][0] == res["f64_omp"][0]
    assert np.array_equal(res["f64"][1], res["f64_omp"][1])
    assert np.array_equal(res["f64"][2], res["f64_omp"][2])
    assert oracle.threads(0, "f64") == 1 and oracle.threads(0) >= 1
