"""Small runs of every step path for compute-sanitizer (SURVEY.md section 4 tier 4, section 5;
PAPER.md L150-152: GPU memory errors and a device leak were the paper's own pain points).

    compute-sanitizer --tool racecheck --error-exitcode 3 python tests/sanitizer_cases.py [case ...]

Each case drives the library through the Python binding on bunches small enough for the
sanitizer's slowdown: 2 x 2 x 2 patches of 8^3 and one patch of 32^3 for the 3D paths.  Results are
not compared with the oracle here (the parity tests do that); a case only checks that the run
finished with finite numbers and no bad cells, so that the sanitizer's verdict is about a run that
did the work.  tests/test_gpu_sanitizer.py runs the smallest one-pass case under racecheck;
profiles/r3_sanitizer.md records the full sweep.  Not collected by pytest (no test_ prefix)."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2508_09568_b200 import workloads as W            # noqa: E402
from paper_2508_09568_b200.binding import MhdBunch          # noqa: E402

F = {"f32": np.float32, "f64": np.float64}


def _bunch(w, dtype, path="auto", **tune):
    b = MhdBunch(w.n, w.npatch, w.nbr, w.gamma, w.dx, dtype=dtype)
    b.set_path(path)
    for k, v in tune.items():
        b.set_tuning(k, v)
    b.load(w.U)
    return b


def _resident(w, dtype, path="auto", steps=2, want=None, **tune):
    b = _bunch(w, dtype, path, **tune)
    assert want is None or b.path == want, (b.path, want)
    for _ in range(steps):
        b.fill_guards()
        b.cfl_dt(0.4, sync=False)
        b.step_dev()
    out = b.download()
    assert np.isfinite(out).all() and b.status() == 0
    b.close()


def small3d(dtype):
    return W.turbulence(N=16, n=8, dtype=F[dtype])             # 2 x 2 x 2 patches of 8^3: the 16 x 16 tile


def one32(dtype):
    return W.turbulence(N=32, n=32, dtype=F[dtype])            # one patch of 32^3, its own neighbour: the 32 x 8 tile


def case_onepass_small():
    _resident(small3d("f32"), "f32", want="onepass")


def case_onepass_zseg_cfl():
    for w in (small3d("f32"), one32("f32")):
        for zseg in (1, 3):
            for cfl in (0, 1):
                _resident(w, "f32", want="onepass", onepass_zseg=zseg, fused_cfl=cfl)


def case_onepass_variants():
    w = small3d("f32")
    for lim, emf, flux in ((2, 0, 0), (1, 1, 0), (1, 0, 1)):
        b = MhdBunch(w.n, w.npatch, w.nbr, w.gamma, w.dx, dtype="f32", limiter=lim, emf_solver=emf, flux_solver=flux)
        b.load(w.U)
        b.fill_guards(); b.cfl_dt(0.4, sync=False); b.step_dev()
        assert np.isfinite(b.download()).all() and b.status() == 0
        b.close()
    s = W.turbulence(N=(20, 24, 18), n=(10, 12, 9), dtype=np.float32)   # ragged rows: no gather, ragged tiles
    _resident(s, "f32", want="onepass")


def case_two_kernel():
    for dtype in ("f32", "f64"):
        for w in (small3d(dtype), one32(dtype)):
            _resident(w, dtype, path="two_kernel", want="two_kernel")


def case_staged():
    for dtype in ("f32", "f64"):
        _resident(small3d(dtype), dtype, path="staged", want="staged")
    _resident(W.sod(64, 4, dtype=np.float64), "f64", steps=2)              # outflow sides, cell-by-cell fill


def case_tile2d():
    for dtype in ("f32", "f64"):
        _resident(W.orszag_tang(64, 32, dtype=F[dtype]), dtype, want="tile2d")
        _resident(W.orszag_tang(60, 20, dtype=F[dtype]), dtype, want="tile2d")


def case_line1d():
    for dtype in ("f32", "f64"):
        _resident(W.alfven_wave(N=64, n=16, dtype=F[dtype]), dtype, want="tile2d")


def case_step_host():
    import torch
    for w, chunk, tune in ((W.turbulence(N=(16, 16, 64), n=(16, 16, 8), dtype=np.float32), 2, {}),
                           (W.turbulence(N=(32, 32, 64), n=(16, 16, 32), dtype=np.float32), 2, {"host_bands": 2}),
                           (W.turbulence(N=(16, 16, 64), n=(16, 16, 8), dtype=np.float32), 3, {"host_max_pitch": 1})):
        b = _bunch(w, "f32", **tune)
        b.host_attach(chunk)
        hin = torch.from_numpy(np.ascontiguousarray(W.to_compact(w.U, w.n))).pin_memory()
        hout = torch.zeros_like(hin).pin_memory()
        dt = 0.0
        for _ in range(2):
            _, dt = b.step_host(hin, hout, dt=dt, courant=0.4)
            hin, hout = hout, hin
        assert np.isfinite(hin.numpy()).all() and b.status() == 0
        b.close()


def case_step_ring():
    import torch
    w = W.turbulence(N=(32, 32, 128), n=16, dtype=np.float32)              # 32 patches through a window of 12
    win = MhdBunch(w.n, 12, W.neighbour_table((12, 1, 1), (True, True, True)), w.gamma, w.dx, dtype="f32")
    win.ring_attach(w.nbr, 4)
    hin = torch.from_numpy(np.ascontiguousarray(W.to_compact(w.U, w.n))).pin_memory()
    hout = torch.empty_like(hin).pin_memory()
    dt = 1e-3
    for _ in range(2):
        dt = min(dt, win.step_ring(hin, hout, dt, 0.4))
        hin, hout = hout, hin
    assert np.isfinite(hin.numpy()).all() and win.status() == 0
    win.ring_detach()
    win.close()


def case_step_local():
    for dtype, path in (("f32", "auto"), ("f64", "two_kernel"), ("f64", "staged")):
        w = small3d(dtype)
        b = _bunch(w, dtype, path)
        b.local_begin(0.0)
        dt = 0.5 * float(b.cfl_local(0.4).min())
        assert b.step_local(np.arange(8), [dt / 2 if p in (0, 3, 5) else dt for p in range(8)])
        assert b.step_local([0, 3, 5], dt / 2)
        b.local_end()
        assert np.isfinite(b.download()).all() and b.status() == 0
        b.close()


def case_cfl_static():
    import torch
    from paper_2508_09568_b200 import binding
    for dtype in ("f32", "f64"):
        w = small3d(dtype)
        b = _bunch(w, dtype)
        b.fill_guards()
        state = b.state[b._cur_index()]
        dt = torch.zeros(1, dtype=torch.float64, device=state.device)
        pp = torch.zeros(w.npatch, dtype=torch.float64, device=state.device)
        for _ in range(2):
            binding.cfl_dt_static(b.desc, state, 0.4, dt, pp)
        b.stream.synchronize()
        assert dt.item() == b.cfl_dt(0.4, sync=True)
        b.close()


CASES = {k[5:]: v for k, v in list(globals().items()) if k.startswith("case_")}

if __name__ == "__main__":
    names = sys.argv[1:] or list(CASES)
    for name in names:
        CASES[name]()
        print("ran", name, flush=True)
