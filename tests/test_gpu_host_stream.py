"""GPU parity of the host-streaming path (include/mhd_bunch.h, mhd_bunch_host_*; SURVEY 8f
NEXT-1): a host-resident bunch in the compact layout goes
through upload -> guard exchange -> step -> download in chunks.  The result is compared with
the CPU oracle (same tolerances as the resident path) and, bit for bit, with the resident
path of the same library."""
import numpy as np
import pytest

from parity_util import TOL_STEP, make_gpu, make_oracle, rel_err
from paper_2508_09568_b200 import workloads as W

pytestmark = pytest.mark.gpu
NPD = {"f32": np.float32, "f64": np.float64}


def workloads(dtype):
    t = NPD[dtype]
    return {
        "turb16": W.turbulence(N=32, n=16, dtype=t),                          # 8 patches, 3D periodic
        "turb_slabs": W.turbulence(N=(16, 16, 64), n=(16, 16, 8), dtype=t),   # 8 slabs stacked along z
        "turb_ragged": W.turbulence(N=(24, 20, 36), n=(12, 10, 9), dtype=t),
        "turb_self": W.turbulence(N=16, n=16, dtype=t),
        "ot64": W.orszag_tang(64, 32, dtype=t),                               # 2D: tile kernel, whole-chunk units
        "alfven1d": W.alfven_wave(N=64, n=16, dtype=t),                       # 1D along x: line kernel
    }


def pinned(a):
    import torch
    t = torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    return t


def oracle_step(w, dt=None, courant=0.4):
    o = make_oracle(w)
    U = o.fill_guards(w.U.astype(np.float64), w.nbr)
    dt_ref = o.cfl_dt(U, courant)
    new = o.step(U, dt_ref if dt is None else dt)
    new_f = o.fill_guards(new.copy(), w.nbr)
    return dt_ref, new, o.cfl_dt(new_f, courant)


@pytest.mark.parametrize("path", ["two_kernel", "staged"])
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_step_host_on_the_other_step_paths(dtype, path):
    """fp32 3D bunches default to the one-pass kernel; the same call through the two-kernel path
    (overlapped schedule, predictor gathers halos) and the staged path (whole-bunch step)."""
    import torch
    w = workloads(dtype)["turb_slabs"]
    dt_ref, ref, dt_next_ref = oracle_step(w)
    b = make_gpu(w, dtype, path=path)
    b.host_attach(2)
    hin = pinned(W.to_compact(w.U, w.n))
    hout = torch.zeros_like(hin).pin_memory()
    used, nxt = b.step_host(hin, hout, dt=dt_ref, courant=0.4)
    assert rel_err(hout.numpy().astype(np.float64), W.to_compact(ref, w.n)) <= TOL_STEP[dtype]
    assert abs(nxt - dt_next_ref) <= 10 * TOL_STEP[dtype] * dt_next_ref
    b.close()


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("chunk", [1, 3, 0])
@pytest.mark.parametrize("given_dt", [True, False])
@pytest.mark.parametrize("name", ["turb16", "turb_slabs", "turb_ragged", "turb_self", "ot64", "alfven1d"])
def test_step_host_matches_oracle(name, given_dt, chunk, dtype):
    import torch
    w = workloads(dtype)[name]
    dt_ref, ref, dt_next_ref = oracle_step(w)
    b = make_gpu(w, dtype)
    b.load(np.zeros_like(w.U))                       # nothing of the input may come from the device
    lay = b.host_attach(chunk)
    assert lay.host_bytes == 8 * w.npatch * int(np.prod(w.n)) * np.dtype(NPD[dtype]).itemsize
    hin = pinned(W.to_compact(w.U, w.n))
    hout = torch.zeros_like(hin).pin_memory()
    used, nxt = b.step_host(hin, hout, dt=dt_ref if given_dt else 0.0, courant=0.4)
    tol_dt = 1e-13 if dtype == "f64" else 2e-6
    assert abs(used - dt_ref) <= tol_dt * dt_ref
    assert abs(nxt - dt_next_ref) <= max(tol_dt, 10 * TOL_STEP[dtype]) * dt_next_ref
    got = hout.numpy().astype(np.float64)
    err = rel_err(got, W.to_compact(ref, w.n))
    assert err <= TOL_STEP[dtype], err
    assert np.array_equal(hin.numpy(), W.to_compact(w.U, w.n))     # the input is read-only
    assert b.status() == 0
    b.close()


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("name", ["turb16", "turb_slabs", "ot64", "alfven1d"])
def test_host_stream_equals_resident_path_bitwise_over_several_steps(name, dtype):
    """Three chained steps (dt_next of one call is the dt of the next) through host buffers
    against the resident loop fill_guards -> cfl_dt -> step of the same library."""
    import torch
    w = workloads(dtype)[name]
    r = make_gpu(w, dtype)
    res_dts = []
    for _ in range(3):
        r.fill_guards()
        dt = r.cfl_dt(0.4, sync=True)
        res_dts.append(dt)
        r.step(dt)
    want = W.to_compact(r.download(), w.n)
    r.close()

    b = make_gpu(w, dtype)
    b.host_attach(2)
    bufs = [pinned(W.to_compact(w.U, w.n)), None]
    bufs[1] = torch.zeros_like(bufs[0]).pin_memory()
    dt, dts = 0.0, []
    for s in range(3):
        used, dt = b.step_host(bufs[s % 2], bufs[(s + 1) % 2], dt=dt, courant=0.4)
        dts.append(used)
    assert dts == res_dts
    assert np.array_equal(bufs[1].numpy(), want)
    # the device holds the same level: resident calls may follow
    assert np.array_equal(W.to_compact(b.download(), w.n), want)
    b.close()


@pytest.mark.parametrize("chunk,bands", [(2, 4), (4, 2), (8, 4), (3, 3)])
def test_banded_host_stream_equals_resident_path_bitwise(chunk, bands):
    """The first chunk and the last two are stepped band by band (MHD_TUNE_HOST_BANDS): the one-pass
    kernel and the closing-face sync run on plane ranges, uploads arrive as plane ranges, downloads
    leave as plane ranges -- the result is the resident step's, bit for bit, over chained steps."""
    import torch
    w = W.turbulence(N=(32, 32, 64), n=(16, 16, 32), dtype=np.float32)      # 2 x 2 x 2 patches of 32 planes
    r = make_gpu(w, "f32")
    res_dts = []
    for _ in range(3):
        r.fill_guards()
        dt = r.cfl_dt(0.4, sync=True)
        res_dts.append(dt)
        r.step(dt)
    want = W.to_compact(r.download(), w.n)
    r.close()
    b = make_gpu(w, "f32")
    b.load(np.zeros_like(w.U))
    b.set_tuning("host_bands", bands)
    lay = b.host_attach(chunk)
    assert (lay.chunk_patches, lay.bands, lay.pipelined) == (chunk, bands, 1)
    bufs = [pinned(W.to_compact(w.U, w.n)), None]
    bufs[1] = torch.zeros_like(bufs[0]).pin_memory()
    dt, dts = 0.0, []
    for s in range(3):
        used, dt = b.step_host(bufs[s % 2], bufs[(s + 1) % 2], dt=dt, courant=0.4)
        dts.append(used)
    assert dts == res_dts
    assert np.array_equal(bufs[1].numpy(), want)
    assert np.array_equal(W.to_compact(b.download(), w.n), want)
    b.close()


def test_host_stream_schedule_and_rejections():
    from paper_2508_09568_b200.binding import HostLayout, _check
    import ctypes as C
    w = W.turbulence(N=(16, 16, 64), n=(16, 16, 8), dtype=np.float32)
    b = make_gpu(w, "f32")
    lay = b.host_attach(1)
    assert (lay.chunk_patches, lay.nchunk, lay.pipelined) == (1, 8, 1)
    lay2 = HostLayout()
    b.set_path("two_kernel")            # its predictor gathers halos too: same overlapped schedule
    _check(b.lib.mhd_bunch_host_query(b.h, 3, C.byref(lay2)), "q")
    assert (lay2.chunk_patches, lay2.nchunk, lay2.pipelined) == (3, 3, 1)
    b.set_path("staged")                # reads the guard shell from HBM: whole-bunch step between the copies
    _check(b.lib.mhd_bunch_host_query(b.h, 3, C.byref(lay2)), "q")
    assert (lay2.chunk_patches, lay2.nchunk, lay2.pipelined) == (3, 3, 0)
    b.close()
    # outflow neighbours: the compact layout cannot carry the evolved closing faces
    s = W.sod(256, 8, dtype=np.float64)
    b = make_gpu(s, "f64")
    with pytest.raises(RuntimeError):
        b.host_attach(0)
    # not attached -> state error
    import torch
    t = torch.zeros(8, dtype=torch.float64).pin_memory()
    with pytest.raises(RuntimeError):
        b.step_host(t, t, dt=0.1)
    b.close()


# ------------------------------------------------- ring mode: bunch larger than the buffers ----
@pytest.mark.parametrize("shape", ["slabs16_R3", "slabs16_R5", "cube64_R3", "ragged_chunks"])
def test_ring_step_equals_resident_step_bitwise(shape):
    """a host-resident bunch streams through device
    buffers that hold only a WINDOW of it (a ring of chunk slots deliberately smaller than the bunch;
    halos are read through a neighbour table rewritten in slot numbers, the first chunks are uploaded
    a second time for the last ones).  Three chained steps, each bit for bit the resident step of the
    same kernel (the ring always runs the variant with the CFL epilogue, so the resident handle is
    switched to it too), with the same dt sequence from that epilogue."""
    import torch
    from paper_2508_09568_b200.binding import MhdBunch
    w, chunk, R = {"slabs16_R3": (lambda: W.turbulence(N=(32, 32, 128), n=16, dtype=np.float32), 4, 3),
                   "slabs16_R5": (lambda: W.turbulence(N=(32, 32, 128), n=16, dtype=np.float32), 4, 5),
                   "cube64_R3": (lambda: W.turbulence(N=128, n=32, dtype=np.float32, config=2), 16, 3),
                   "ragged_chunks": (lambda: W.turbulence(N=(48, 32, 160), n=16, dtype=np.float32), 7, 6)}[shape]
    w = w()
    assert R * chunk < w.npatch
    ref = make_gpu(w, "f32")                                   # the whole bunch resident
    ref.set_tuning("fused_cfl", 1)
    win = MhdBunch(w.n, R * chunk, W.neighbour_table((R * chunk, 1, 1), (True, True, True)), w.gamma, w.dx, dtype="f32")
    win.ring_attach(w.nbr, chunk)
    hin = pinned(W.to_compact(w.U, w.n))
    hout = torch.empty_like(hin).pin_memory()
    ref.fill_guards()
    dt = ref.cfl_dt(0.4, sync=True)
    for _ in range(3):
        ref.fill_guards()
        ref.step(dt)
        dt_next = win.step_ring(hin, hout, dt, 0.4)
        want = W.to_compact(ref.download(), w.n)
        assert np.array_equal(hout.numpy(), want)
        ref.fill_guards()
        dt = ref.cfl_dt(0.4, sync=True)
        assert dt_next == dt
        hin, hout = hout, hin
    assert win.status() == 0
    win.ring_detach()
    ref.close(); win.close()


def test_ring_attach_rejections():
    from paper_2508_09568_b200.binding import MhdBunch
    w = W.turbulence(N=(32, 32, 64), n=16, dtype=np.float32)
    win = MhdBunch(w.n, 8, W.neighbour_table((8, 1, 1), (True, True, True)), w.gamma, w.dx, dtype="f32")
    with pytest.raises(RuntimeError):
        win.ring_attach(w.nbr, 4)                              # two slots cannot hold a slab and both neighbours
    bad = w.nbr.copy(); bad[3, 0] = -1
    with pytest.raises(RuntimeError):
        win.ring_attach(bad, 2)
    w64 = MhdBunch(w.n, 12, W.neighbour_table((12, 1, 1), (True, True, True)), w.gamma, w.dx, dtype="f64")
    with pytest.raises(RuntimeError):
        w64.ring_attach(w.nbr, 4)                              # needs the one-pass step
    assert win.lib.mhd_bunch_step_ring(win.h, None, None, 1e-3, 0.4, None) == -4
    win.close(); w64.close()
