"""Seeded synthetic workloads shaped like BASELINE.json's configs (numpy only).

This module serves BOTH the CPU oracle's tests and the CUDA path (it imports neither).
It holds the decomposition of a global grid into a bunch of patches, the neighbour
table, and the initial conditions; it holds none of the scheme's arithmetic (the only
physics here is the definition of the initial state: E from rho, u, p, B by the EOS of
PAPER.md L68, and face fields as the discrete curl of a vector potential).

The paper's own runs (Sod L186, Orszag-Tang L188, 3D turbulence L212) need DISPATCH
drivers and initial data that are not available; these are the stand-ins (DESIGN.md,
"Input recipe").  Nothing here is copied from a benchmark suite: the set-ups are the
closed forms written in BASELINE.json.

Dense bunch layout: U[field][patch][k][j][i], guards included (width ng in active
dimensions, none in collapsed ones), field order rho, mx, my, mz, E, Bx, By, Bz with
B on LOWER faces.  Patch id p = px + Px*(py + Py*pz).
"""
from dataclasses import dataclass, field

import numpy as np

NG = 3


# ------------------------------------------------------------------ decomposition --
def padded(n, ng=NG):
    """(mx, my, mz) for interior sizes n = (nx, ny, nz)."""
    return tuple(k + 2 * ng if k > 1 else 1 for k in n)


def neighbour_table(P, periodic):
    """nbr[npatch][27]: class (oz+1)*9+(oy+1)*3+(ox+1) -> patch id or -1 (outflow)."""
    Px, Py, Pz = P
    nbr = np.full((Px * Py * Pz, 27), -1, dtype=np.int32)
    for pz in range(Pz):
        for py in range(Py):
            for px in range(Px):
                p = px + Px * (py + Py * pz)
                for oz in (-1, 0, 1):
                    for oy in (-1, 0, 1):
                        for ox in (-1, 0, 1):
                            q = [px + ox, py + oy, pz + oz]
                            ok = True
                            for d in range(3):
                                if 0 <= q[d] < P[d]:
                                    continue
                                if periodic[d]:
                                    q[d] %= P[d]
                                else:
                                    ok = False
                            cls = (oz + 1) * 9 + (oy + 1) * 3 + (ox + 1)
                            nbr[p, cls] = q[0] + Px * (q[1] + Py * q[2]) if ok else -1
    return nbr


def scatter(cons5, bfaces, n, P, ng=NG, dtype=np.float64):
    """Global fields -> dense bunch array.

    cons5  : [5, Nz, Ny, Nx] rho, mx, my, mz, E at cell centres
    bfaces : (bx [Nz,Ny,Nx+1], by [Nz,Ny+1,Nx], bz [Nz+1,Ny,Nx]) on faces; in a
             collapsed dimension the extra face is ignored.
    Interior cells and the closing faces (face n in the first high guard slot) are set;
    all other guard cells are zero until a guard fill.
    """
    nx, ny, nz = n
    Px, Py, Pz = P
    mx, my, mz = padded(n, ng)
    g = [ng if k > 1 else 0 for k in n]
    U = np.zeros((8, Px * Py * Pz, mz, my, mx), dtype=dtype)
    for pz in range(Pz):
        for py in range(Py):
            for px in range(Px):
                p = px + Px * (py + Py * pz)
                X = slice(px * nx, (px + 1) * nx); Y = slice(py * ny, (py + 1) * ny); Z = slice(pz * nz, (pz + 1) * nz)
                I = (slice(g[2], g[2] + nz), slice(g[1], g[1] + ny), slice(g[0], g[0] + nx))
                U[:5, p][(slice(None),) + I] = cons5[:, Z, Y, X]
                ex = 1 if nx > 1 else 0; ey = 1 if ny > 1 else 0; ez = 1 if nz > 1 else 0
                U[5, p, I[0], I[1], g[0]:g[0] + nx + ex] = bfaces[0][Z, Y, px * nx:(px + 1) * nx + ex]
                U[6, p, I[0], g[1]:g[1] + ny + ey, I[2]] = bfaces[1][Z, py * ny:(py + 1) * ny + ey, X]
                U[7, p, g[2]:g[2] + nz + ez, I[1], I[2]] = bfaces[2][pz * nz:(pz + 1) * nz + ez, Y, X]
    return U


def gather(U, n, P, ng=NG):
    """Dense bunch array -> global interior fields [8, Nz, Ny, Nx] (lower-face B)."""
    nx, ny, nz = n
    Px, Py, Pz = P
    g = [ng if k > 1 else 0 for k in n]
    out = np.zeros((8, Pz * nz, Py * ny, Px * nx), dtype=U.dtype)
    for pz in range(Pz):
        for py in range(Py):
            for px in range(Px):
                p = px + Px * (py + Py * pz)
                out[:, pz * nz:(pz + 1) * nz, py * ny:(py + 1) * ny, px * nx:(px + 1) * nx] = \
                    U[:, p, g[2]:g[2] + nz, g[1]:g[1] + ny, g[0]:g[0] + nx]
    return out


def to_compact(U, n, ng=NG):
    """Dense bunch array [8, npatch, mz, my, mx] -> compact host layout [8, npatch, nz, ny, nx]
    (interior cells only; include/mhd_bunch.h, host-streaming path)."""
    g = [ng if k > 1 else 0 for k in n]
    return np.ascontiguousarray(U[:, :, g[2]:g[2] + n[2], g[1]:g[1] + n[1], g[0]:g[0] + n[0]])


def from_compact(Uc, n, ng=NG):
    """Compact host layout -> dense bunch array with every guard cell zero."""
    mx, my, mz = padded(n, ng)
    g = [ng if k > 1 else 0 for k in n]
    U = np.zeros(Uc.shape[:2] + (mz, my, mx), dtype=Uc.dtype)
    U[:, :, g[2]:g[2] + n[2], g[1]:g[1] + n[1], g[0]:g[0] + n[0]] = Uc
    return U


def conserved_from_primitive(rho, vel, p, bfaces, gamma):
    """Definition of the initial state (EOS): returns cons5 [5,Nz,Ny,Nx].
    Cell-centred B is the mean of the two faces (reading O2/Q5)."""
    bc = [0.5 * (bfaces[0][:, :, :-1] + bfaces[0][:, :, 1:]),
          0.5 * (bfaces[1][:, :-1, :] + bfaces[1][:, 1:, :]),
          0.5 * (bfaces[2][:-1, :, :] + bfaces[2][1:, :, :])]
    ekin = 0.5 * rho * (vel[0] ** 2 + vel[1] ** 2 + vel[2] ** 2)
    emag = 0.5 * (bc[0] ** 2 + bc[1] ** 2 + bc[2] ** 2)
    E = p / (gamma - 1.0) + ekin + emag
    return np.stack([rho, rho * vel[0], rho * vel[1], rho * vel[2], E])


@dataclass
class Workload:
    name: str
    n: tuple            # interior cells per patch (nx, ny, nz)
    P: tuple            # patches per side (Px, Py, Pz)
    gamma: float
    dx: tuple
    periodic: tuple
    U: np.ndarray       # dense [8, npatch, mz, my, mx]; guards unfilled
    nbr: np.ndarray     # [npatch, 27] int32
    courant: float = 0.4
    t_end: float = 0.0
    ng: int = NG
    meta: dict = field(default_factory=dict)

    @property
    def npatch(self):
        return self.P[0] * self.P[1] * self.P[2]

    @property
    def cells(self):
        return self.npatch * self.n[0] * self.n[1] * self.n[2]


def _finish(name, n, P, gamma, dx, periodic, cons5, bfaces, dtype, **kw):
    U = scatter(cons5, bfaces, n, P, NG, dtype=np.float64).astype(dtype)
    return Workload(name=name, n=tuple(n), P=tuple(P), gamma=gamma, dx=tuple(dx), periodic=tuple(periodic),
                    U=U, nbr=neighbour_table(P, periodic), **kw)


# ------------------------------------------------------------------------ config 0 --
def sod(ncell=256, npatch=8, dtype=np.float64, axis=0):
    """BASELINE.json config 0: 1D Sod tube, B=0, gamma=1.4, [0,1], outflow ends.
    `axis` orients the tube along x (0), y (1) or z (2) for the permutation tests."""
    N = [1, 1, 1]; N[axis] = ncell
    n = [1, 1, 1]; n[axis] = ncell // npatch
    P = [1, 1, 1]; P[axis] = npatch
    x = (np.arange(ncell) + 0.5) / ncell
    shp = [1, 1, 1]; shp[2 - axis] = ncell        # arrays are [z, y, x]
    left = (x < 0.5).reshape(shp)
    rho = np.where(left, 1.0, 0.125) * np.ones((N[2], N[1], N[0]))
    p = np.where(left, 1.0, 0.1) * np.ones_like(rho)
    vel = [np.zeros_like(rho) for _ in range(3)]
    bf = (np.zeros((N[2], N[1], N[0] + 1)), np.zeros((N[2], N[1] + 1, N[0])), np.zeros((N[2] + 1, N[1], N[0])))
    dx = [1.0, 1.0, 1.0]; dx[axis] = 1.0 / ncell
    per = [True, True, True]; per[axis] = False
    cons = conserved_from_primitive(rho, vel, p, bf, 1.4)
    return _finish("sod", n, P, 1.4, dx, per, cons, bf, dtype, courant=0.4, t_end=0.2,
                   meta={"ncell": ncell, "axis": axis})


def mhd_tube(left, right, bn, gamma, ncell=128, npatch=4, axis=0, dtype=np.float64, t_end=0.1):
    """Generic 1D MHD Riemann problem along `axis` with outflow ends.  left/right =
    (rho, un, ut1, ut2, p, Bt1, Bt2) in the tube's own (normal, t1, t2) frame, which is
    the cyclic image of (x, y, z); `bn` is the uniform normal field."""
    N = [1, 1, 1]; N[axis] = ncell
    n = [1, 1, 1]; n[axis] = ncell // npatch
    P = [1, 1, 1]; P[axis] = npatch
    t1, t2 = (axis + 1) % 3, (axis + 2) % 3
    x = (np.arange(ncell) + 0.5) / ncell
    shp = [1, 1, 1]; shp[2 - axis] = ncell
    isl = (x < 0.5).reshape(shp)
    one = np.ones((N[2], N[1], N[0]))
    pick = lambda k: np.where(isl, left[k], right[k]) * one
    rho, p = pick(0), pick(4)
    vel = [None] * 3
    vel[axis], vel[t1], vel[t2] = pick(1), pick(2), pick(3)
    fs = [(N[2], N[1], N[0] + 1), (N[2], N[1] + 1, N[0]), (N[2] + 1, N[1], N[0])]
    bf = [None] * 3
    bf[axis] = bn * np.ones(fs[axis])
    for t, k in ((t1, 5), (t2, 6)):
        b = pick(k)
        bf[t] = np.concatenate([b, b], axis=2 - t)
    dx = [1.0, 1.0, 1.0]; dx[axis] = 1.0 / ncell
    per = [True, True, True]; per[axis] = False
    cons = conserved_from_primitive(rho, vel, p, tuple(bf), gamma)
    return _finish("mhd_tube", n, P, gamma, dx, per, cons, tuple(bf), dtype, courant=0.4, t_end=t_end,
                   meta={"ncell": ncell, "axis": axis})


# ------------------------------------------------------------------------ config 1 --
def orszag_tang(N=256, n=32, dtype=np.float64):
    """BASELINE.json config 1: Orszag-Tang vortex on periodic [0,1]^2, gamma=5/3."""
    gamma = 5.0 / 3.0
    B0 = 1.0 / np.sqrt(4.0 * np.pi)
    dx = 1.0 / N
    xc = (np.arange(N) + 0.5) * dx
    xf = np.arange(N + 1) * dx
    rho = np.full((1, N, N), 25.0 / (36.0 * np.pi))
    p = np.full((1, N, N), 5.0 / (12.0 * np.pi))
    Y, X = np.meshgrid(xc, xc, indexing="ij")
    vel = [(-np.sin(2 * np.pi * Y))[None], (np.sin(2 * np.pi * X))[None], np.zeros((1, N, N))]
    # corner vector potential A_z(x_i, y_j); B = curl A by differencing => div B = 0 to round-off
    Yf, Xf = np.meshgrid(xf, xf, indexing="ij")
    Az = B0 * (np.cos(2 * np.pi * Yf) / (2 * np.pi) + np.cos(4 * np.pi * Xf) / (4 * np.pi))
    bx = ((Az[1:, :] - Az[:-1, :]) / dx)[None]          # [1, N, N+1]
    by = (-(Az[:, 1:] - Az[:, :-1]) / dx)[None]         # [1, N+1, N]
    bz = np.zeros((2, N, N))
    cons = conserved_from_primitive(rho, vel, p, (bx, by, bz), gamma)
    P = (N // n, N // n, 1)
    return _finish("orszag_tang", (n, n, 1), P, gamma, (dx, dx, 1.0), (True, True, True), cons, (bx, by, bz),
                   dtype, courant=0.4, t_end=0.5, meta={"N": N})


# -------------------------------------------------------------------- configs 2 - 4 --
def _band_limited(rng, N, power, kmin=1, kmax=8, base=32):
    """Band-limited Gaussian random field on a periodic N^3 grid: white N(0,1) noise on
    a base^3 grid, filtered with a(k) = |k|^-power for kmin <= |k| <= kmax (integer
    wavenumbers), zero elsewhere, interpolated spectrally to N^3.  The field depends on
    the seed only, not on N (so it can be refined).  Mean zero, unit variance."""
    white = rng.standard_normal((base, base, base))
    spec = np.fft.rfftn(white)
    k1 = np.fft.fftfreq(base, 1.0 / base)
    kz, ky, kx = np.meshgrid(k1, k1, np.fft.rfftfreq(base, 1.0 / base), indexing="ij")
    kk = np.sqrt(kx ** 2 + ky ** 2 + kz ** 2)
    amp = np.where((kk >= kmin) & (kk <= kmax), np.maximum(kk, 1e-30) ** (-power), 0.0)
    spec = spec * amp
    Nz, Ny, Nx = (N, N, N) if np.isscalar(N) else N
    kmax = max(1, min(kmax, min(Nz, Ny, Nx) // 2 - 1))        # tiny test grids: stay below Nyquist
    amp = np.where(kk <= kmax, amp, 0.0)
    spec = spec * (amp > 0)
    big = np.zeros((Nz, Ny, Nx // 2 + 1), dtype=np.complex128)
    h = kmax + 1
    for sz, dz_ in ((slice(0, h), slice(0, h)), (slice(base - h + 1, base), slice(Nz - h + 1, Nz))):
        for sy, dy_ in ((slice(0, h), slice(0, h)), (slice(base - h + 1, base), slice(Ny - h + 1, Ny))):
            big[dz_, dy_, :h] = spec[sz, sy, :h]
    try:                       # the same pocketfft transform on all cores (bitwise the numpy result)
        from scipy import fft as _sfft
        f = _sfft.irfftn(big, s=(Nz, Ny, Nx), axes=(0, 1, 2), workers=-1)
    except ImportError:
        f = np.fft.irfftn(big, s=(Nz, Ny, Nx), axes=(0, 1, 2))
    f *= (Nz * Ny * Nx / base ** 3)
    f -= f.mean()
    f /= f.std()
    return f


def turbulence(N=256, n=32, dtype=np.float32, config=2, patches=None, seed_extra=()):
    """BASELINE.json configs 2-4: driven-turbulence-like periodic cube, gamma=5/3.
    rho lognormal (sigma_ln 0.5, mean 1) from a smooth band-limited field, p = 1, v a
    k^-2 Gaussian field with rms Mach 1, B = (0.1,0,0) + curl of a Gaussian potential
    (rms 0.05).  `N` may be a 3-tuple (Nx,Ny,Nz) for non-cubic patch arrangements."""
    gamma = 5.0 / 3.0
    if np.isscalar(N):
        N = (N, N, N)
    n3 = (n, n, n) if np.isscalar(n) else tuple(n)
    Nx, Ny, Nz = N
    shape = (Nz, Ny, Nx)
    L = max(N)
    dx = 1.0 / L

    def rng(fld):
        return np.random.default_rng(np.random.SeedSequence([2508, 9568, config, fld, *seed_extra]))

    lnrho = 0.5 * _band_limited(rng(0), shape, 2.0)
    rho = np.exp(lnrho)
    rho /= rho.mean()
    p = np.ones(shape)
    vel = [_band_limited(rng(1 + a), shape, 2.0) for a in range(3)]
    v2 = np.mean(vel[0] ** 2 + vel[1] ** 2 + vel[2] ** 2)
    cs = np.sqrt(gamma * 1.0 / 1.0)
    vel = [v * (cs / np.sqrt(v2)) for v in vel]
    A = [_band_limited(rng(4 + a), shape, 3.0) for a in range(3)]   # Ax, Ay, Az on edges

    def d(f, axis):  # forward periodic difference along array axis
        return np.roll(f, -1, axis=axis) - f
    # arrays are [z, y, x]: axis 2 = x, 1 = y, 0 = z
    bx = d(A[2], 1) / dx - d(A[1], 0) / dx
    by = d(A[0], 0) / dx - d(A[2], 2) / dx
    bz = d(A[1], 2) / dx - d(A[0], 1) / dx
    rms = np.sqrt(np.mean(bx ** 2 + by ** 2 + bz ** 2))
    s = 0.05 / rms
    bx = 0.1 + s * bx; by = s * by; bz = s * bz
    # append the periodic closing faces
    bxf = np.concatenate([bx, bx[:, :, :1]], axis=2)
    byf = np.concatenate([by, by[:, :1, :]], axis=1)
    bzf = np.concatenate([bz, bz[:1, :, :]], axis=0)
    cons = conserved_from_primitive(rho, vel, p, (bxf, byf, bzf), gamma)
    P = patches if patches is not None else (Nx // n3[0], Ny // n3[1], Nz // n3[2])
    assert (P[0] * n3[0], P[1] * n3[1], P[2] * n3[2]) == (Nx, Ny, Nz)
    return _finish(f"turbulence_c{config}", n3, P, gamma, (dx, dx, dx), (True, True, True), cons,
                   (bxf, byf, bzf), dtype, courant=0.4, meta={"N": N})


def alfven_wave(N=32, n=None, dtype=np.float64, axis=0, amp=0.1):
    """Circularly polarised Alfven wave along `axis` on a periodic 1D grid (an exact
    nonlinear solution of ideal MHD): rho=1, p=0.1, Bn=1, Bt = amp*(cos, sin)(2 pi x),
    v_t = -Bt/sqrt(rho); moves with the Alfven speed 1, period 1."""
    gamma = 5.0 / 3.0
    n = n or N
    Ns = [1, 1, 1]; Ns[axis] = N
    ns = [1, 1, 1]; ns[axis] = n
    P = [1, 1, 1]; P[axis] = N // n
    xc = (np.arange(N) + 0.5) / N
    shp = [1, 1, 1]; shp[2 - axis] = N
    ph = (2 * np.pi * xc).reshape(shp)
    one = np.ones((Ns[2], Ns[1], Ns[0]))
    t1, t2 = (axis + 1) % 3, (axis + 2) % 3
    bt1 = amp * np.cos(ph) * one; bt2 = amp * np.sin(ph) * one
    vel = [None] * 3
    vel[axis] = 0 * one; vel[t1] = -bt1; vel[t2] = -bt2
    fs = [(Ns[2], Ns[1], Ns[0] + 1), (Ns[2], Ns[1] + 1, Ns[0]), (Ns[2] + 1, Ns[1], Ns[0])]
    bf = [None] * 3
    bf[axis] = np.ones(fs[axis])
    for t, b in ((t1, bt1), (t2, bt2)):   # collapsed dimensions: duplicate the cell value
        bf[t] = np.concatenate([b, b], axis=2 - t)
    cons = conserved_from_primitive(one.copy(), vel, 0.1 * one, tuple(bf), gamma)
    dx = [1.0, 1.0, 1.0]; dx[axis] = 1.0 / N
    return _finish("alfven", ns, P, gamma, dx, (True, True, True), cons, tuple(bf), dtype,
                   courant=0.4, t_end=1.0, meta={"N": N, "axis": axis, "amp": amp})


def alfven_wave_2d(N=32, n=None, dtype=np.float64, amp=0.1):
    """Circularly polarised Alfven wave running along the diagonal of the periodic unit
    square (x,y), z collapsed: phase = 2 pi (x + y), B_par = 1 along (1,1)/sqrt2, rho = 1,
    p = 0.1; period 1/sqrt(2).  In-plane faces are the discrete curl of A_z at corners."""
    gamma = 5.0 / 3.0
    n = n or N
    h = 1.0 / N
    xc = (np.arange(N) + 0.5) * h
    xf = np.arange(N + 1) * h
    Y, X = np.meshgrid(xc, xc, indexing="ij")
    ph = 2 * np.pi * (X + Y)
    r2 = np.sqrt(2.0)
    Yf, Xf = np.meshgrid(xf, xf, indexing="ij")
    Az = -amp * np.sin(2 * np.pi * (Xf + Yf)) / (2 * np.pi * r2)
    bx = (1.0 / r2 + (Az[1:, :] - Az[:-1, :]) / h)[None]
    by = (1.0 / r2 - (Az[:, 1:] - Az[:, :-1]) / h)[None]
    bzc = (amp * np.sin(ph))[None]
    bz = np.concatenate([bzc, bzc], axis=0)
    one = np.ones((1, N, N))
    vperp = -amp * np.cos(ph)[None]          # along e_perp = (-1,1)/sqrt2
    vel = [-vperp / r2, vperp / r2, -bzc]
    cons = conserved_from_primitive(one, vel, 0.1 * one, (bx, by, bz), gamma)
    P = (N // n, N // n, 1)
    return _finish("alfven2d", (n, n, 1), P, gamma, (h, h, 1.0), (True, True, True), cons, (bx, by, bz), dtype,
                   courant=0.4, t_end=1.0 / r2, meta={"N": N})


def from_global_periodic(g, n, gamma, dx, dtype=np.float64, name="global"):
    """Bunch from global periodic fields g[8, Nz, Ny, Nx] (lower-face B)."""
    Nz, Ny, Nx = g.shape[1:]
    bf = (np.concatenate([g[5], g[5][:, :, :1]], axis=2), np.concatenate([g[6], g[6][:, :1, :]], axis=1),
          np.concatenate([g[7], g[7][:1, :, :]], axis=0))
    P = (Nx // n[0], Ny // n[1], Nz // n[2])
    return _finish(name, n, P, gamma, dx, (True, True, True), g[:5], bf, dtype)
