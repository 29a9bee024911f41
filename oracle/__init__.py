"""ctypes binding of the CPU oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It never imports paper_2508_09568_b200.

    o = oracle.Oracle(n=(32, 1, 1), npatch=8, gamma=1.4, dx=(1/256, 1, 1))
    o.fill_guards(U, nbr); dt = o.cfl_dt(U, 0.4); U1 = o.step(U, dt)

Arrays are numpy, dense, shape [8, npatch, mz, my, mx] (guards included), dtype
float64 (or float32 with dtype="f32", a diagnostic build of the same source).
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

NSTAGE = 70
STAGE_SLICES = {
    "q": (0, 8), "dq": (8, 32), "dbf": (32, 38), "e0": (38, 41), "bh": (41, 44),
    "qh": (44, 52), "flux": (52, 67), "emf": (67, 70),
}


class _Desc(C.Structure):
    _fields_ = [("n", C.c_int32 * 3), ("ng", C.c_int32), ("npatch", C.c_int32),
                ("limiter", C.c_int32), ("emf_solver", C.c_int32), ("flux_solver", C.c_int32),
                ("gamma", C.c_double), ("dx", C.c_double * 3)]


_LIBS = {}


def _lib(key):
    if key not in _LIBS:
        # MHD_ORACLE_LIBDIR: load liboracle_<key>.so from there instead of building the committed
        # source -- how tests/test_oracle_mutations.py points the pins at a deliberately broken
        # copy of the oracle.  "f64_omp" is the OpenMP build of the same source (bench.py).
        alt = os.environ.get("MHD_ORACLE_LIBDIR")
        if key == "f64_omp":
            path = _build.build_omp()
        elif alt:
            path = os.path.join(alt, "liboracle_%s.so" % key)
        else:
            path = _build.build()[key]
        lib = C.CDLL(path)
        rp = C.c_void_p
        lib.orc_sizeof_real.restype = C.c_int
        lib.orc_threads.restype = C.c_int
        lib.orc_threads.argtypes = [C.c_int]
        lib.orc_patch_cells.restype = C.c_int64
        lib.orc_patch_cells.argtypes = [C.POINTER(_Desc)]
        lib.orc_state_elems.restype = C.c_int64
        lib.orc_state_elems.argtypes = [C.POINTER(_Desc)]
        lib.orc_fill_guards.restype = None
        lib.orc_fill_guards.argtypes = [C.POINTER(_Desc), rp, rp]
        lib.orc_cfl_dt.restype = C.c_double
        lib.orc_cfl_dt.argtypes = [C.POINTER(_Desc), rp, C.c_double, rp]
        lib.orc_step.restype = None
        lib.orc_step.argtypes = [C.POINTER(_Desc), rp, rp, C.c_double]
        lib.orc_stages.restype = None
        lib.orc_stages.argtypes = [C.POINTER(_Desc), rp, C.c_int32, C.c_double, rp]
        lib.orc_local_ready.restype = C.c_int
        lib.orc_local_ready.argtypes = [C.POINTER(_Desc), rp, rp, rp, rp, C.c_int32]
        lib.orc_fill_guards_local.restype = None
        lib.orc_fill_guards_local.argtypes = [C.POINTER(_Desc), rp, rp, rp, rp, rp, rp, C.c_int32]
        lib.orc_step_local.restype = C.c_int
        lib.orc_step_local.argtypes = [C.POINTER(_Desc), rp, rp, rp, rp, rp, rp, rp, C.c_int32, rp]
        real = C.c_float if key == "f32" else C.c_double
        lib.orc_limiter.restype = real
        lib.orc_limiter.argtypes = [C.c_int32, real, real]
        lib.orc_hlld.restype = None
        lib.orc_hlld.argtypes = [C.c_double, rp, rp, real, rp]
        lib.orc_hll.restype = None
        lib.orc_hll.argtypes = [C.c_double, rp, rp, real, rp]
        lib.orc_emf2d.restype = real
        lib.orc_emf2d.argtypes = [C.c_double, C.c_int32, rp, real, real, real, real]
        lib.orc_fast_speed.restype = real
        lib.orc_fast_speed.argtypes = [C.c_double, real, real, real, real, real]
        _LIBS[key] = lib
    return _LIBS[key]


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


class Oracle:
    def __init__(self, n, npatch, gamma, dx, ng=3, limiter=1, emf_solver=0, dtype="f64", flux_solver=0):
        self.key = dtype
        self.np_dtype = np.float32 if dtype == "f32" else np.float64
        self.lib = _lib(dtype)
        d = _Desc()
        d.n[:] = list(n)
        d.ng, d.npatch, d.limiter, d.emf_solver, d.flux_solver = ng, npatch, limiter, emf_solver, flux_solver
        d.gamma = gamma
        d.dx[:] = list(dx)
        self.desc = d
        self.n = tuple(n)
        self.ng = ng
        self.npatch = npatch
        self.m = tuple(k + 2 * ng if k > 1 else 1 for k in n)   # (mx, my, mz)
        self.shape = (8, npatch, self.m[2], self.m[1], self.m[0])
        assert self.lib.orc_state_elems(C.byref(d)) == int(np.prod(self.shape))

    def _chk(self, U):
        assert U.dtype == self.np_dtype and U.shape == self.shape and U.flags["C_CONTIGUOUS"], \
            (U.dtype, U.shape, self.shape)

    def fill_guards(self, U, nbr):
        self._chk(U)
        nbr = np.ascontiguousarray(nbr, dtype=np.int32)
        assert nbr.shape == (self.npatch, 27)
        self.lib.orc_fill_guards(C.byref(self.desc), _ptr(nbr), _ptr(U))
        return U

    def cfl_dt(self, U, courant, per_patch=False):
        self._chk(U)
        pp = np.zeros(self.npatch, dtype=np.float64)
        dt = self.lib.orc_cfl_dt(C.byref(self.desc), _ptr(U), courant, _ptr(pp))
        return (dt, pp) if per_patch else dt

    def step(self, U, dt):
        self._chk(U)
        out = np.empty_like(U)
        self.lib.orc_step(C.byref(self.desc), _ptr(U), _ptr(out), dt)
        return out

    def stages(self, U, patch, dt):
        """All scratch arrays of one patch: dict name -> array [count, mz, my, mx]."""
        self._chk(U)
        out = np.zeros((NSTAGE,) + self.shape[2:], dtype=self.np_dtype)
        self.lib.orc_stages(C.byref(self.desc), _ptr(U), patch, dt, _ptr(out))
        return {k: out[a:b] for k, (a, b) in STAGE_SLICES.items()}

    # ---- O10: local time steps (two slices per patch) -------------------------------------
    def local_state(self, U, t0=0.0):
        """Both slices = U at time t0: dict(S=[S0, S1], cur, t_old, t_new)."""
        self._chk(U)
        return {"S": [U.copy(), U.copy()], "cur": np.zeros(self.npatch, dtype=np.int32),
                "t_old": np.full(self.npatch, t0), "t_new": np.full(self.npatch, t0)}

    def local_ready(self, st, nbr, patches):
        nbr = np.ascontiguousarray(nbr, dtype=np.int32)
        lst = np.ascontiguousarray(patches, dtype=np.int32)
        return bool(self.lib.orc_local_ready(C.byref(self.desc), _ptr(nbr), _ptr(st["t_old"]), _ptr(st["t_new"]), _ptr(lst), len(lst)))

    def fill_guards_local(self, st, nbr, p):
        nbr = np.ascontiguousarray(nbr, dtype=np.int32)
        self.lib.orc_fill_guards_local(C.byref(self.desc), _ptr(nbr), _ptr(st["S"][0]), _ptr(st["S"][1]), _ptr(st["cur"]),
                                       _ptr(st["t_old"]), _ptr(st["t_new"]), int(p))

    def step_local(self, st, nbr, patches, dt):
        """Advance the listed patches by their own dt (in place); False if one is not ready."""
        nbr = np.ascontiguousarray(nbr, dtype=np.int32)
        lst = np.ascontiguousarray(patches, dtype=np.int32)
        dts = np.ascontiguousarray(np.broadcast_to(np.asarray(dt, dtype=np.float64), lst.shape))
        rc = self.lib.orc_step_local(C.byref(self.desc), _ptr(nbr), _ptr(st["S"][0]), _ptr(st["S"][1]), _ptr(st["cur"]),
                                     _ptr(st["t_old"]), _ptr(st["t_new"]), _ptr(lst), len(lst), _ptr(dts))
        return rc == 0

    def local_newest(self, st):
        """[8, npatch, ...]: the newer slice of every patch."""
        out = np.empty_like(st["S"][0])
        for p in range(self.npatch):
            out[:, p] = st["S"][st["cur"][p]][:, p]
        return out

    # interior view helper: [8, npatch, nz, ny, nx]
    def interior(self, U):
        sl = [slice(self.ng, self.ng + k) if k > 1 else slice(0, 1) for k in self.n]
        return U[:, :, sl[2], sl[1], sl[0]]


def threads(want=0, dtype="f64_omp"):
    """Threads the per-patch loops of the OpenMP build use (set if want > 0); 1 for the plain builds."""
    return _lib(dtype).orc_threads(want)


def limiter(kind, a, b, dtype="f64"):
    return _lib(dtype).orc_limiter(kind, a, b)


def hlld(gamma, L, R, bn, dtype="f64"):
    """L, R = (rho,u,v,w,p,By,Bz); returns fluxes of (rho,mu,mv,mw,E,By,Bz)."""
    t = np.float64 if dtype == "f64" else np.float32
    L = np.ascontiguousarray(L, dtype=t); R = np.ascontiguousarray(R, dtype=t)
    F = np.zeros(7, dtype=t)
    _lib(dtype).orc_hlld(gamma, _ptr(L), _ptr(R), float(bn), _ptr(F))
    return F


def hll(gamma, L, R, bn, dtype="f64"):
    """HLL flux (PAPER.md 2.1.1); same arguments and layout as hlld."""
    t = np.float64 if dtype == "f64" else np.float32
    L = np.ascontiguousarray(L, dtype=t); R = np.ascontiguousarray(R, dtype=t)
    F = np.zeros(7, dtype=t)
    _lib(dtype).orc_hll(gamma, _ptr(L), _ptr(R), float(bn), _ptr(F))
    return F


def emf2d(gamma, solver, corners, AS, AN, BW, BE, dtype="f64"):
    """corners[4][6]: SW,SE,NW,NE x (rho,ua,ub,ue,p,Be)."""
    t = np.float64 if dtype == "f64" else np.float32
    c = np.ascontiguousarray(corners, dtype=t)
    assert c.shape == (4, 6)
    return _lib(dtype).orc_emf2d(gamma, solver, _ptr(c), float(AS), float(AN), float(BW), float(BE))


def fast_speed(gamma, rho, p, bn, bt1, bt2, dtype="f64"):
    return _lib(dtype).orc_fast_speed(gamma, rho, p, bn, bt1, bt2)
