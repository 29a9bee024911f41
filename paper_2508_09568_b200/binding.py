"""Thin ctypes binding of include/mhd_bunch.h -- argument marshalling only.

Every step of the path runs in the hand-written sm_100a kernels of libmhd_bunch.so.
PyTorch is used for device memory and streams only.  There is no CPU fallback: if the
library cannot be loaded or no CUDA device is present, construction raises.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

MHD_F32, MHD_F64 = 0, 1
PATHS = {"auto": 0, "staged": 1, "two_kernel": 2, "onepass": 3, "tile2d": 4}
TUNE = {"onepass_zseg": 1, "predict_ty": 2, "fused_cfl": 3, "host_bands": 4, "host_max_pitch": 5}
_ERR = {0: "ok", -1: "MHD_EINVAL", -2: "MHD_ENOMEM", -3: "MHD_ECUDA", -4: "MHD_ESTATE"}

ABI_SYMBOLS = [
    "mhd_bunch_query", "mhd_bunch_create", "mhd_bunch_fill_guards", "mhd_bunch_cfl_dt", "mhd_bunch_step",
    "mhd_bunch_step_dev", "mhd_bunch_upload", "mhd_bunch_download", "mhd_bunch_set_timing",
    "mhd_bunch_kernel_times", "mhd_bunch_current", "mhd_bunch_status", "mhd_bunch_launch_count",
    "mhd_bunch_chunk", "mhd_bunch_sync_guards", "mhd_bunch_set_path", "mhd_bunch_get_path", "mhd_bunch_set_tuning", "mhd_bunch_measure_alu_peak", "mhd_bunch_destroy", "mhd_bunch_strerror", "mhd_bunch_last_cuda_error",
    "mhd_bunch_host_query", "mhd_bunch_host_attach", "mhd_bunch_step_host", "mhd_bunch_host_detach",
    "mhd_bunch_host_schedule",
    "mhd_bunch_ring_plan", "mhd_bunch_ring_attach", "mhd_bunch_step_ring", "mhd_bunch_ring_detach",
    "mhd_bunch_local_begin", "mhd_bunch_step_local", "mhd_bunch_cfl_local", "mhd_bunch_local_state", "mhd_bunch_local_end",
    "mhd_bunch_cfl_dt_static",
]
CFL_STATIC_MAX_PATCHES = 32768   # MHD_CFL_STATIC_MAX_PATCHES of include/mhd_bunch.h


class Desc(C.Structure):
    _fields_ = [("n", C.c_int32 * 3), ("ng", C.c_int32), ("npatch", C.c_int32), ("dtype", C.c_int32),
                ("limiter", C.c_int32), ("emf_solver", C.c_int32), ("device", C.c_int32), ("flux_solver", C.c_int32),
                ("gamma", C.c_double), ("dx", C.c_double * 3), ("stream", C.c_void_p)]


class Layout(C.Structure):
    _fields_ = [("stride", C.c_int64 * 5), ("origin", C.c_int64), ("state_elems", C.c_int64),
                ("state_bytes", C.c_size_t), ("workspace_min", C.c_size_t), ("workspace_best", C.c_size_t),
                ("m", C.c_int32 * 3), ("reserved", C.c_int32)]


class HostLayout(C.Structure):
    _fields_ = [("host_bytes", C.c_size_t), ("staging_bytes", C.c_size_t), ("chunk_patches", C.c_int32),
                ("nchunk", C.c_int32), ("pipelined", C.c_int32), ("bands", C.c_int32)]


_lib = None


def load_library(build_if_missing=True):
    """Load libmhd_bunch.so (building it with nvcc if absent or stale).  Raises on failure."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.TARGET
    if build_if_missing and _build.stale():
        _build.build()
    if not os.path.exists(path):
        raise RuntimeError(f"{path} is missing: the CUDA extension must be built (no CPU fallback)")
    lib = C.CDLL(path)
    vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    lib.mhd_bunch_query.argtypes = [C.POINTER(Desc), C.POINTER(Layout)]
    lib.mhd_bunch_create.argtypes = [C.POINTER(Desc), vp, vp, vp, vp, C.c_size_t, C.POINTER(vp)]
    lib.mhd_bunch_fill_guards.argtypes = [vp]
    lib.mhd_bunch_sync_guards.argtypes = [vp]
    lib.mhd_bunch_cfl_dt.argtypes = [vp, dbl, C.POINTER(dbl), vp, vp]
    lib.mhd_bunch_step.argtypes = [vp, dbl]
    lib.mhd_bunch_step_dev.argtypes = [vp, vp, dbl]
    lib.mhd_bunch_upload.argtypes = [vp, vp]
    lib.mhd_bunch_download.argtypes = [vp, vp]
    lib.mhd_bunch_set_timing.argtypes = [vp, i32]
    lib.mhd_bunch_kernel_times.argtypes = [vp, i32, C.POINTER(C.c_char_p), C.POINTER(dbl), C.POINTER(i64), C.POINTER(i32)]
    lib.mhd_bunch_current.argtypes = [vp, C.POINTER(vp)]
    lib.mhd_bunch_status.argtypes = [vp, C.POINTER(i64)]
    lib.mhd_bunch_launch_count.argtypes = [vp, C.POINTER(i64)]
    lib.mhd_bunch_chunk.argtypes = [vp, C.POINTER(i32)]
    lib.mhd_bunch_set_path.argtypes = [vp, i32]
    lib.mhd_bunch_get_path.argtypes = [vp, C.POINTER(i32)]
    lib.mhd_bunch_measure_alu_peak.argtypes = [i32, i32, vp, C.c_size_t, C.POINTER(dbl)]
    lib.mhd_bunch_set_tuning.argtypes = [vp, i32, i32]
    lib.mhd_bunch_destroy.argtypes = [vp]
    lib.mhd_bunch_host_query.argtypes = [vp, i32, C.POINTER(HostLayout)]
    lib.mhd_bunch_host_attach.argtypes = [vp, vp, C.c_size_t, i32]
    lib.mhd_bunch_step_host.argtypes = [vp, vp, vp, dbl, dbl, C.POINTER(dbl), C.POINTER(dbl)]
    lib.mhd_bunch_host_detach.argtypes = [vp]
    lib.mhd_bunch_host_schedule.argtypes = [vp, i32, i32, i32, i32, i32, C.POINTER(i32), C.POINTER(i32), C.POINTER(i32), vp, vp, vp,
                                            C.POINTER(i32), vp, vp, vp, vp, i32, C.POINTER(dbl)]
    lib.mhd_bunch_ring_plan.argtypes = [vp, i32, i32, i32, C.POINTER(i32), C.POINTER(i32), vp, vp, vp, vp, i32]
    lib.mhd_bunch_ring_attach.argtypes = [vp, vp, i32, i32, vp, C.c_size_t]
    lib.mhd_bunch_step_ring.argtypes = [vp, vp, vp, dbl, dbl, C.POINTER(dbl)]
    lib.mhd_bunch_ring_detach.argtypes = [vp]
    lib.mhd_bunch_local_begin.argtypes = [vp, dbl]
    lib.mhd_bunch_step_local.argtypes = [vp, vp, i32, vp]
    lib.mhd_bunch_cfl_local.argtypes = [vp, dbl, vp]
    lib.mhd_bunch_local_state.argtypes = [vp, vp, vp, vp]
    lib.mhd_bunch_local_end.argtypes = [vp]
    lib.mhd_bunch_cfl_dt_static.argtypes = [C.POINTER(Desc), vp, dbl, vp, vp]
    lib.mhd_bunch_strerror.argtypes = [C.c_int]
    lib.mhd_bunch_strerror.restype = C.c_char_p
    lib.mhd_bunch_last_cuda_error.restype = C.c_char_p
    for name in ABI_SYMBOLS:
        getattr(lib, name)
    _lib = lib
    return lib


def _check(rc, what):
    if rc != 0:
        lib = load_library()
        msg = lib.mhd_bunch_strerror(rc).decode()
        cu = lib.mhd_bunch_last_cuda_error().decode()
        raise RuntimeError(f"{what}: {_ERR.get(rc, rc)} ({msg}) {cu}")


def make_desc(n, npatch, gamma, dx, dtype=MHD_F32, limiter=1, emf_solver=0, device=0, stream=0, ng=3, flux_solver=0):
    d = Desc()
    d.n[:] = list(n)
    d.ng, d.npatch, d.dtype, d.limiter, d.emf_solver, d.device = ng, npatch, dtype, limiter, emf_solver, device
    d.flux_solver = flux_solver
    d.gamma = gamma
    d.dx[:] = list(dx)
    d.stream = stream
    return d


def query(desc):
    lay = Layout()
    _check(load_library().mhd_bunch_query(C.byref(desc), C.byref(lay)), "mhd_bunch_query")
    return lay


def measure_alu_peak(dtype="f32", device=0):
    """Measured FMA-chain peak in TFLOP/s (FMA = 2 flops) of the fp32 or fp64 pipe."""
    import torch
    v = C.c_double(0.0)
    scratch = torch.empty(4 << 20, dtype=torch.uint8, device=torch.device("cuda", device))
    _check(load_library().mhd_bunch_measure_alu_peak(MHD_F32 if dtype == "f32" else MHD_F64, device, scratch.data_ptr(),
                                                     scratch.numel(), C.byref(v)), "mhd_bunch_measure_alu_peak")
    return v.value


def cfl_dt_static(desc, state, courant, dt_dev, dt_patch=None):
    """mhd_bunch_cfl_dt_static: the CFL step of a state buffer for callers that own no handle and no
    workspace and cannot allocate one where they stand (a framework's task hook running under other
    streams' work, an application whose pool holds all of HBM).  The reduction's scratch is an array
    inside libmhd_bunch.so, good for CFL_STATIC_MAX_PATCHES patches and shared by every call on the
    device, so calls that may overlap on the GPU must be ordered by the caller.

    desc: make_desc(...); state: torch CUDA tensor in the layout query(desc) gives, closing faces up to
    date; dt_dev: torch CUDA float64[1]; dt_patch: torch CUDA float64[npatch] or None.  Only enqueues
    on desc.stream.  Raises RuntimeError (MHD_ENOMEM) beyond the limit."""
    _check(load_library().mhd_bunch_cfl_dt_static(C.byref(desc), state.data_ptr(), courant, dt_dev.data_ptr(),
                                                   dt_patch.data_ptr() if dt_patch is not None else None),
           "mhd_bunch_cfl_dt_static")


def host_schedule(nbr, chunk_patches=0, nz=32, guard=3, bands=0):
    """Schedule of the host-streaming step for a neighbour table (host only, no device): dict with
    chunk, bands, the upload pieces (piece_chunk, piece_k0, piece_k1: planes [k0, k1) of a chunk), the
    step units in order (unit_chunk, unit_za, unit_zb), ready[u] (last piece unit u needs) and the
    simulated makespan."""
    nbr = np.ascontiguousarray(nbr, dtype=np.int32)
    npatch = nbr.shape[0]
    chunk, bnd, npiece, nunit, span = C.c_int32(0), C.c_int32(0), C.c_int32(0), C.c_int32(0), C.c_double(0.0)
    cap = 4 * npatch + 64
    pc, k0, k1, uc, za, zb, ready = (np.zeros(cap, dtype=np.int32) for _ in range(7))
    ptr = lambda a: a.ctypes.data_as(C.c_void_p)
    _check(load_library().mhd_bunch_host_schedule(ptr(nbr), npatch, nz, guard, chunk_patches, bands, C.byref(chunk), C.byref(bnd),
                                                  C.byref(npiece), ptr(pc), ptr(k0), ptr(k1), C.byref(nunit), ptr(uc), ptr(za),
                                                  ptr(zb), ptr(ready), cap, C.byref(span)), "mhd_bunch_host_schedule")
    n, m = nunit.value, npiece.value
    return {"chunk": chunk.value, "nchunk": -(-npatch // chunk.value), "bands": bnd.value, "npiece": m, "nunit": n,
            "piece_chunk": pc[:m].copy(), "piece_k0": k0[:m].copy(), "piece_k1": k1[:m].copy(),
            "unit_chunk": uc[:n].copy(), "unit_za": za[:n].copy(), "unit_zb": zb[:n].copy(), "ready": ready[:n].copy(),
            "makespan": span.value}


def ring_plan(nbr, chunk_patches, ring_chunks):
    """Schedule of a ring step (host only): dict(nchunk, up_chunk, up_slot, up_step, step_slot) or
    None if a chunk's neighbourhood does not fit in `ring_chunks` slots."""
    nbr = np.ascontiguousarray(nbr, dtype=np.int32)
    npatch = nbr.shape[0]
    nchunk, nup = C.c_int32(0), C.c_int32(0)
    cap = 4 * npatch + 8
    a, b_, c_, d_ = (np.zeros(cap, dtype=np.int32) for _ in range(4))
    rc = load_library().mhd_bunch_ring_plan(nbr.ctypes.data_as(C.c_void_p), npatch, chunk_patches, ring_chunks, C.byref(nchunk),
                                            C.byref(nup), a.ctypes.data_as(C.c_void_p), b_.ctypes.data_as(C.c_void_p),
                                            c_.ctypes.data_as(C.c_void_p), d_.ctypes.data_as(C.c_void_p), cap)
    if rc == -2:
        return None
    _check(rc, "mhd_bunch_ring_plan")
    n = nup.value
    return {"nchunk": nchunk.value, "up_chunk": a[:n].copy(), "up_slot": b_[:n].copy(), "up_step": c_[:n].copy(),
            "step_slot": d_[:nchunk.value].copy()}


class MhdBunch:
    """A bunch of patches resident in HBM.

        b = MhdBunch(n=(32,32,32), npatch=512, nbr=nbr, gamma=5/3, dx=(h,h,h), dtype="f32")
        b.load(U_dense_numpy); b.fill_guards(); b.cfl_dt(0.4, sync=False); b.step_dev()
    """

    def __init__(self, n, npatch, nbr, gamma, dx, dtype="f32", limiter=1, emf_solver=0, device=0,
                 workspace_bytes=None, stream=None, flux_solver=0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("MhdBunch needs a CUDA device: there is no CPU fallback")
        self.torch = torch
        self.lib = load_library()
        self.device = torch.device("cuda", device)
        self.tdtype = torch.float32 if dtype == "f32" else torch.float64
        self.npdtype = np.float32 if dtype == "f32" else np.float64
        self.n, self.npatch = tuple(n), npatch
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.current_stream()
        self.desc = make_desc(n, npatch, gamma, dx, MHD_F32 if dtype == "f32" else MHD_F64, limiter, emf_solver,
                              device, self.stream.cuda_stream, flux_solver=flux_solver)
        self.lay = query(self.desc)
        self.m = tuple(self.lay.m)
        ws = self.lay.workspace_best if workspace_bytes is None else max(int(workspace_bytes), self.lay.workspace_min)
        self.state = [torch.zeros(self.lay.state_elems, dtype=self.tdtype, device=self.device) for _ in range(2)]
        self.workspace = torch.empty(ws, dtype=torch.uint8, device=self.device)
        self.dt_dev = torch.zeros(1, dtype=torch.float64, device=self.device)
        self.dt_patch = torch.zeros(npatch, dtype=torch.float64, device=self.device)
        nbr = np.ascontiguousarray(nbr, dtype=np.int32)
        assert nbr.shape == (npatch, 27)
        h = C.c_void_p()
        _check(self.lib.mhd_bunch_create(C.byref(self.desc), nbr.ctypes.data_as(C.c_void_p), self.state[0].data_ptr(),
                                         self.state[1].data_ptr(), self.workspace.data_ptr(), ws, C.byref(h)),
               "mhd_bunch_create")
        self.h = h

    # ---- plumbing -----------------------------------------------------------------
    def _cur_index(self):
        p = C.c_void_p()
        _check(self.lib.mhd_bunch_current(self.h, C.byref(p)), "mhd_bunch_current")
        return 0 if p.value == self.state[0].data_ptr() else 1

    def view(self, which=None):
        """Strided torch view [8, npatch, mz, my, mx] of the current (or given) buffer."""
        idx = self._cur_index() if which is None else which
        shape = (8, self.npatch, self.m[2], self.m[1], self.m[0])
        return self.state[idx].as_strided(shape, tuple(self.lay.stride), int(self.lay.origin))

    def load(self, U):
        """Dense numpy [8, npatch, mz, my, mx] -> current buffer."""
        t = self.torch.from_numpy(np.ascontiguousarray(U, dtype=self.npdtype))
        with self.torch.cuda.stream(self.stream):
            self.view().copy_(t.to(self.device, non_blocking=False))
        self.stream.synchronize()

    def download(self):
        with self.torch.cuda.stream(self.stream):
            out = self.view().contiguous().cpu().numpy()
        return out

    # ---- the path -------------------------------------------------------------------
    def fill_guards(self):
        _check(self.lib.mhd_bunch_fill_guards(self.h), "mhd_bunch_fill_guards")

    def sync_guards(self):
        """Write a deferred guard fill to HBM now (include/mhd_bunch.h)."""
        _check(self.lib.mhd_bunch_sync_guards(self.h), "mhd_bunch_sync_guards")

    def cfl_dt(self, courant, sync=True, per_patch=False):
        dt = C.c_double(0.0)
        _check(self.lib.mhd_bunch_cfl_dt(self.h, courant, C.byref(dt) if sync else None, self.dt_dev.data_ptr(),
                                         self.dt_patch.data_ptr() if per_patch else None), "mhd_bunch_cfl_dt")
        return dt.value if sync else None

    def step(self, dt):
        _check(self.lib.mhd_bunch_step(self.h, dt), "mhd_bunch_step")

    def step_dev(self, dt_max=0.0):
        _check(self.lib.mhd_bunch_step_dev(self.h, self.dt_dev.data_ptr(), dt_max), "mhd_bunch_step_dev")

    def upload_host(self, host_tensor):
        _check(self.lib.mhd_bunch_upload(self.h, host_tensor.data_ptr()), "mhd_bunch_upload")

    def download_host(self, host_tensor):
        _check(self.lib.mhd_bunch_download(self.h, host_tensor.data_ptr()), "mhd_bunch_download")

    # ---- host-streaming path (include/mhd_bunch.h: mhd_bunch_host_*) -------------------
    def host_attach(self, chunk_patches=0):
        """Allocate the device staging (a torch tensor) and attach it; returns the layout."""
        lay = HostLayout()
        _check(self.lib.mhd_bunch_host_query(self.h, chunk_patches, C.byref(lay)), "mhd_bunch_host_query")
        self.host_staging = self.torch.empty(lay.staging_bytes, dtype=self.torch.uint8, device=self.device)
        _check(self.lib.mhd_bunch_host_attach(self.h, self.host_staging.data_ptr(), lay.staging_bytes,
                                              lay.chunk_patches), "mhd_bunch_host_attach")
        self.host_lay = lay
        return lay

    def step_host(self, host_in, host_out, dt=0.0, courant=0.4):
        """host_in/host_out: pinned torch CPU tensors in the compact layout [8, npatch, nz, ny, nx].
        Returns (dt_used, dt_next)."""
        used, nxt = C.c_double(0.0), C.c_double(0.0)
        _check(self.lib.mhd_bunch_step_host(self.h, host_in.data_ptr(), host_out.data_ptr(), dt, courant,
                                            C.byref(used), C.byref(nxt)), "mhd_bunch_step_host")
        return used.value, nxt.value

    # ---- ring mode: a host bunch larger than the device buffers (mhd_bunch_ring_*) ------------
    def ring_attach(self, nbr_big, chunk_patches):
        nbr_big = np.ascontiguousarray(nbr_big, dtype=np.int32)
        esz = 4 if self.tdtype == self.torch.float32 else 8
        nbytes = 2 * ((8 * chunk_patches * self.n[0] * self.n[1] * self.n[2] * esz + 255) // 256 * 256)
        self.ring_staging = self.torch.empty(nbytes, dtype=self.torch.uint8, device=self.device)
        _check(self.lib.mhd_bunch_ring_attach(self.h, nbr_big.ctypes.data_as(C.c_void_p), nbr_big.shape[0], chunk_patches,
                                              self.ring_staging.data_ptr(), nbytes), "mhd_bunch_ring_attach")

    def step_ring(self, host_in, host_out, dt, courant=0.4):
        nxt = C.c_double(0.0)
        _check(self.lib.mhd_bunch_step_ring(self.h, host_in.data_ptr(), host_out.data_ptr(), dt, courant, C.byref(nxt)),
               "mhd_bunch_step_ring")
        return nxt.value

    def ring_detach(self):
        _check(self.lib.mhd_bunch_ring_detach(self.h), "mhd_bunch_ring_detach")

    # ---- local time steps (include/mhd_bunch.h: mhd_bunch_local_*) --------------------------
    def local_begin(self, t0=0.0):
        _check(self.lib.mhd_bunch_local_begin(self.h, t0), "mhd_bunch_local_begin")

    def step_local(self, patches, dt):
        """Advance the listed patches by their own dt; returns False if one of them is not ready."""
        lst = np.ascontiguousarray(patches, dtype=np.int32)
        dts = np.ascontiguousarray(np.broadcast_to(np.asarray(dt, dtype=np.float64), lst.shape))
        rc = self.lib.mhd_bunch_step_local(self.h, lst.ctypes.data_as(C.c_void_p), len(lst), dts.ctypes.data_as(C.c_void_p))
        if rc == -4:
            return False
        _check(rc, "mhd_bunch_step_local")
        return True

    def cfl_local(self, courant):
        out = np.zeros(self.npatch, dtype=np.float64)
        _check(self.lib.mhd_bunch_cfl_local(self.h, courant, out.ctypes.data_as(C.c_void_p)), "mhd_bunch_cfl_local")
        return out

    def local_state(self):
        t0, t1 = np.zeros(self.npatch), np.zeros(self.npatch)
        slot = np.zeros(self.npatch, dtype=np.int32)
        _check(self.lib.mhd_bunch_local_state(self.h, t0.ctypes.data_as(C.c_void_p), t1.ctypes.data_as(C.c_void_p),
                                              slot.ctypes.data_as(C.c_void_p)), "mhd_bunch_local_state")
        return t0, t1, slot

    def local_newest(self):
        """Dense numpy [8, npatch, mz, my, mx]: the newer slice of every patch."""
        _, _, slot = self.local_state()
        self.stream.synchronize()
        both = [self.view(i).contiguous().cpu().numpy() for i in (0, 1)]
        out = both[0].copy()
        for p in np.nonzero(slot == 1)[0]:
            out[:, p] = both[1][:, p]
        return out

    def local_end(self):
        _check(self.lib.mhd_bunch_local_end(self.h), "mhd_bunch_local_end")

    def status(self):
        v = C.c_int64(0)
        _check(self.lib.mhd_bunch_status(self.h, C.byref(v)), "mhd_bunch_status")
        return v.value

    @property
    def launches(self):
        v = C.c_int64(0)
        _check(self.lib.mhd_bunch_launch_count(self.h, C.byref(v)), "mhd_bunch_launch_count")
        return v.value

    @property
    def chunk(self):
        v = C.c_int32(0)
        _check(self.lib.mhd_bunch_chunk(self.h, C.byref(v)), "mhd_bunch_chunk")
        return v.value

    def set_path(self, path):
        """'auto' | 'staged' | 'two_kernel' | 'onepass' (include/mhd_bunch.h, MHD_PATH_*)."""
        _check(self.lib.mhd_bunch_set_path(self.h, PATHS[path]), "mhd_bunch_set_path")

    @property
    def path(self):
        v = C.c_int32(0)
        _check(self.lib.mhd_bunch_get_path(self.h, C.byref(v)), "mhd_bunch_get_path")
        return {k: n for n, k in PATHS.items()}[v.value]

    def set_tuning(self, key, value):
        """key: 'onepass_zseg' | 'predict_ty' | 'fused_cfl' | 'host_bands' | 'host_max_pitch' (include/mhd_bunch.h, MHD_TUNE_*)."""
        _check(self.lib.mhd_bunch_set_tuning(self.h, TUNE[key], int(value)), "mhd_bunch_set_tuning")

    def set_timing(self, on):
        _check(self.lib.mhd_bunch_set_timing(self.h, 1 if on else 0), "mhd_bunch_set_timing")

    def kernel_times(self):
        cap = 16
        names = (C.c_char_p * cap)()
        ms = (C.c_double * cap)()
        cnt = (C.c_int64 * cap)()
        n = C.c_int32(0)
        _check(self.lib.mhd_bunch_kernel_times(self.h, cap, names, ms, cnt, C.byref(n)), "mhd_bunch_kernel_times")
        return {names[i].decode(): (ms[i], cnt[i]) for i in range(n.value)}

    def close(self):
        if getattr(self, "h", None) is not None and self.h.value:
            self.lib.mhd_bunch_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
