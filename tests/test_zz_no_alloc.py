"""mhd_bunch_cfl_dt_static: the CFL step for callers that cannot allocate device memory.

Every other entry point borrows a workspace that somebody had to cudaMalloc.  A framework's
task-update hook that runs while other streams are busy (an allocation there serialises the whole
device), an application whose own pool already holds all of HBM, or a module that is handed nothing
but a state pointer has no such workspace and cannot get one where it stands.  For them the library
carries the reduction's scratch inside its own image (MHD_CFL_STATIC_MAX_PATCHES slots, one array per
GPU, shared by every call and never cleared between calls).

What is checked: the new entry point against the handle path (mhd_bunch_cfl_dt), whose kernels it
launches -- the repository's dt tests hold paths that evaluate the same rate function to equality,
bit for bit, and so does this one -- on TWO CALLS IN A ROW that share the array: first a "hot" state
with large rates, then a calm one of the same shape, so that maxima left behind by the first call
would make the second step too small if the call forgot to clear its slots.  Then a bunch of fewer
patches, and the refusal beyond the limit.

This file sorts last on purpose (pytest -x stops at the first failure; a failure here must not hide
the parity tests) and passes alone in a fresh process as well as after the rest of the suite: it
builds its own bunches and depends on nothing another test leaves on the device.
"""
import numpy as np
import pytest

from parity_util import make_gpu
from paper_2508_09568_b200 import workloads as W

pytestmark = pytest.mark.gpu
NPD = {"f32": np.float32, "f64": np.float64}


def _handle_dt(w, U, dtype):
    """(handle, dt, per-patch dt, current state tensor) of the existing path on state U."""
    b = make_gpu(w, dtype)
    b.load(U)
    b.fill_guards()
    dt = b.cfl_dt(0.4, sync=True, per_patch=True)
    pp = b.dt_patch.cpu().numpy().copy()
    state = b.state[b._cur_index()]        # mhd_bunch_current: guard shell and closing faces are in HBM now
    return b, dt, pp, state


def _static_dt(b, state, npatch):
    import torch
    from paper_2508_09568_b200 import binding
    dt = torch.full((1,), -1.0, dtype=torch.float64, device=state.device)
    pp = torch.full((npatch,), -1.0, dtype=torch.float64, device=state.device)
    binding.cfl_dt_static(b.desc, state, 0.4, dt, pp)      # enqueues on the handle's stream; no allocation inside
    b.stream.synchronize()
    return dt.item(), pp.cpu().numpy()


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_static_cfl_matches_handle_path_on_two_calls_in_a_row(dtype):
    w = W.turbulence(N=32, n=16, dtype=NPD[dtype])           # 8 patches of 16^3
    hot = w.U.copy()
    hot[4] *= 25.0                                           # 25 x the energy: faster waves, larger rates
    b_hot, dt_hot, pp_hot, s_hot = _handle_dt(w, hot, dtype)
    b_cal, dt_cal, pp_cal, s_cal = _handle_dt(w, w.U, dtype)
    assert dt_hot < 0.5 * dt_cal                             # the order of the two calls below matters
    got_hot = _static_dt(b_hot, s_hot, w.npatch)             # call 1 leaves the hot maxima in the shared array
    got_cal = _static_dt(b_cal, s_cal, w.npatch)             # call 2 must not see them
    assert got_hot[0] == dt_hot and np.array_equal(got_hot[1], pp_hot)
    assert got_cal[0] == dt_cal and np.array_equal(got_cal[1], pp_cal)
    # the input was not touched: the handle path still gives the same answer
    assert b_cal.cfl_dt(0.4, sync=True) == dt_cal
    # a smaller bunch afterwards uses only the first slots of the array
    w1 = W.turbulence(N=16, n=16, dtype=NPD[dtype])          # one patch, its own neighbour
    b1, dt1, pp1, s1 = _handle_dt(w1, w1.U, dtype)
    got1 = _static_dt(b1, s1, w1.npatch)
    assert got1[0] == dt1 and np.array_equal(got1[1], pp1)
    for b in (b_hot, b_cal, b1):
        b.close()


def test_static_cfl_refuses_bunches_beyond_its_scratch():
    import torch
    from paper_2508_09568_b200 import binding
    w = W.turbulence(N=16, n=16, dtype=np.float32)
    b = make_gpu(w, "f32")
    b.fill_guards()
    state = b.state[b._cur_index()]
    dt = torch.full((1,), -1.0, dtype=torch.float64, device=state.device)
    big = binding.make_desc(w.n, binding.CFL_STATIC_MAX_PATCHES + 1, w.gamma, w.dx, binding.MHD_F32)
    with pytest.raises(RuntimeError, match="MHD_ENOMEM.*MHD_CFL_STATIC_MAX_PATCHES"):
        binding.cfl_dt_static(big, state, 0.4, dt)           # rejected on the host: nothing is launched
    torch.cuda.synchronize()
    assert dt.item() == -1.0
    with pytest.raises(RuntimeError, match="MHD_EINVAL"):
        binding.cfl_dt_static(b.desc, state, 0.0, dt)        # courant must be positive
    b.close()
