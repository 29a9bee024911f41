"""GPU parity of the host-streaming path (include/mhd_bunch.h, mhd_bunch_host_*; SURVEY 8f
NEXT-1): a host-resident bunch in the compact layout goes
through upload -> guard exchange -> step -> download in chunks.  The result is compared with
the CPU oracle (same tolerances as the resident path) and, bit for bit, with the resident
path of the same library."""
import numpy as np
import pytest

from parity_util import TOL_STEP, assert_pure_large, make_gpu, make_oracle, rel_err
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
    assert_pure_large(hout.numpy().astype(np.float64), W.to_compact(ref, w.n), dtype, path)
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
    assert_pure_large(got, W.to_compact(ref, w.n), dtype, name)
    assert np.array_equal(hin.numpy(), W.to_compact(w.U, w.n))     # the input is read-only
    assert b.status() == 0
    b.close()


# host_max_pitch = 1 forces the field-by-field copies that a host bunch with 2 GiB or more per field
# takes (CUDA refuses the bunch-wide pitch of the single strided copy there); 0 = the device's limit
@pytest.mark.parametrize("max_pitch", [0, 1])
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("name", ["turb16", "turb_slabs", "ot64", "alfven1d"])
def test_host_stream_equals_resident_path_bitwise_over_several_steps(name, dtype, max_pitch):
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
    b.set_tuning("host_max_pitch", max_pitch)
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


@pytest.mark.parametrize("max_pitch", [0, 1])
@pytest.mark.parametrize("chunk,bands", [(2, 4), (4, 2), (8, 4), (3, 3)])
def test_banded_host_stream_equals_resident_path_bitwise(chunk, bands, max_pitch):
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
    b.set_tuning("host_max_pitch", max_pitch)        # 1: plane ranges cross as eight 2D copies, not one 3D copy
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
@pytest.mark.parametrize("shape,max_pitch", [("slabs16_R3", 0), ("slabs16_R5", 0), ("cube64_R3", 0), ("ragged_chunks", 0),
                                             ("slabs16_R3", 1), ("ragged_chunks", 1)])
def test_ring_step_equals_resident_step_bitwise(shape, max_pitch):
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
    win.set_tuning("host_max_pitch", max_pitch)      # 1: the copies a bunch with >= 2 GiB per field takes
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


def test_attached_ring_fences_off_the_other_modes():
    """While a ring is attached the device neighbour table holds slot-space rows of the big bunch: the
    resident, host-streaming and local-time-step calls would silently run with it, so they return
    MHD_ESTATE (-4) until ring_detach, after which the window is an ordinary bunch again."""
    import torch
    from paper_2508_09568_b200.binding import MhdBunch
    w = W.turbulence(N=(32, 32, 128), n=16, dtype=np.float32)
    wn = W.neighbour_table((12, 1, 1), (True, True, True))
    win = MhdBunch(w.n, 12, wn, w.gamma, w.dx, dtype="f32")
    win.view()[:] = torch.from_numpy(w.U[:, :12]).to(win.device)
    win.fill_guards()
    dt0 = win.cfl_dt(0.4, sync=True)
    win.ring_attach(w.nbr, 4)
    lib, h = win.lib, win.h
    stage = torch.empty(1 << 20, dtype=torch.uint8, device=win.device)
    dt = __import__("ctypes").c_double(0.0)
    assert lib.mhd_bunch_fill_guards(h) == -4
    assert lib.mhd_bunch_sync_guards(h) == -4
    assert lib.mhd_bunch_cfl_dt(h, 0.4, __import__("ctypes").byref(dt), None, None) == -4
    assert lib.mhd_bunch_step(h, 1e-4) == -4
    assert lib.mhd_bunch_step_dev(h, win.dt_dev.data_ptr(), 0.0) == -4
    assert lib.mhd_bunch_host_attach(h, stage.data_ptr(), stage.numel(), 4) == -4
    assert lib.mhd_bunch_step_host(h, None, None, 1e-4, 0.4, None, None) == -4
    assert lib.mhd_bunch_local_begin(h, 0.0) == -4
    win.ring_detach()
    win.fill_guards()                                          # the window's own table is back on the device
    assert win.cfl_dt(0.4, sync=True) == dt0
    win.local_begin(0.0)
    assert lib.mhd_bunch_ring_attach(h, w.nbr.ctypes.data_as(__import__("ctypes").c_void_p), w.npatch, 4, stage.data_ptr(), stage.numel()) == -4
    assert lib.mhd_bunch_step_ring(h, None, None, 1e-4, 0.4, None) == -4
    win.local_end()
    win.close()


def _mem_available_gib():
    try:
        with open("/proc/meminfo") as fh:
            for line in fh:
                if line.startswith("MemAvailable:"):
                    return int(line.split()[1]) / 2 ** 20
    except OSError:
        pass
    return 0.0


@pytest.mark.skipif(__import__("os").environ.get("MHD_BIG_HOST_TEST", "1") != "1" or _mem_available_gib() < 96,
                    reason="needs 32 GiB of host memory (runs where 96 GiB are available; MHD_BIG_HOST_TEST=0 turns it off)")
def test_ring_step_on_a_host_bunch_with_2gib_per_field():
    """The case the field-by-field copies exist for: 16384 patches of 32^3 in fp32 are exactly 2 GiB per
    field, so the stride between fields of the host bunch is above cudaDevAttrMaxPitch (2^31 - 1) and a
    single strided copy is refused with cudaErrorInvalidPitchValue.  The bunch is a periodic block of
    2 x 2 x 4 patches repeated 1024 times along z (again a periodic field), streamed through a window of
    192 patches from pageable memory; every repetition must come back as the block's own resident step,
    bit for bit.  About 12 s on the B200 box."""
    import torch
    from paper_2508_09568_b200.binding import MhdBunch
    reps, chunk, R = 1024, 64, 3
    wb = W.turbulence(N=(64, 64, 128), n=32, dtype=np.float32, config=2)
    nb = wb.npatch
    assert nb == 16
    ref = make_gpu(wb, "f32")
    ref.set_tuning("fused_cfl", 1)
    ref.fill_guards()
    dt = ref.cfl_dt(0.4, sync=True)
    ref.step(dt)
    want = W.to_compact(ref.download(), wb.n)                   # [8, 16, 32, 32, 32]
    ref.close()
    P = (2, 2, 4 * reps)
    nbr = W.neighbour_table(P, (True, True, True))
    npatch = nb * reps
    block = W.to_compact(wb.U, wb.n)
    hin = np.empty((8, npatch) + block.shape[2:], dtype=np.float32)
    assert hin[0].nbytes == 2 ** 31                             # one field: 2 GiB, one past the largest legal pitch
    hin.reshape(8, reps, nb, *block.shape[2:])[:] = block[:, None]
    hout = np.empty_like(hin)
    win = MhdBunch(wb.n, R * chunk, W.neighbour_table((R * chunk, 1, 1), (True, True, True)), wb.gamma, wb.dx, dtype="f32")
    win.ring_attach(nbr, chunk)
    win.step_ring(torch.from_numpy(hin), torch.from_numpy(hout), dt, 0.4)
    out = hout.reshape(8, reps, nb, *block.shape[2:])
    for r in range(reps):
        assert np.array_equal(out[:, r], want), r
    assert win.status() == 0
    win.ring_detach()
    win.close()
