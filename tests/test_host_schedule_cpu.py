"""Host logic of the host-streaming path (include/mhd_bunch.h, mhd_bunch_host_schedule): the
chunk schedule is computed from the neighbour table alone, so it is checked here without a
GPU -- safety (no chunk steps before every chunk holding one of its neighbours has been
uploaded), tightness, the permutations, the simulated makespan against a pipeline simulation
typed in this file, and the library's choice of chunk size."""
import ctypes as C

import numpy as np
import pytest

from paper_2508_09568_b200 import binding as B
from paper_2508_09568_b200 import workloads as W

TABLES = {
    "cube8": W.neighbour_table((8, 8, 8), (True, True, True)),          # config 2
    "slabs": W.neighbour_table((1, 1, 8), (True, True, True)),
    "paper300": W.neighbour_table((5, 6, 10), (True, True, True)),      # bunch of 300
    "single": W.neighbour_table((1, 1, 1), (True, True, True)),
}


def simulate(npatch, chunk, up_order, ready, step_order, alpha=0.3, eps=1.5):
    """Three in-order queues: uploads back to back, a step after its last needed upload and
    after the previous step, a download after its step and after the previous download."""
    size = lambda c: min(chunk, npatch - c * chunk)
    t, t_up = 0.0, []
    for c in up_order:
        t += size(c) + eps
        t_up.append(t)
    t_step = t_dn = 0.0
    for c in step_order:
        t_step = max(t_step, t_up[ready[c]]) + alpha * size(c) + eps
        t_dn = max(t_dn, t_step) + size(c) + eps
    return t_dn


@pytest.mark.parametrize("chunk", [0, 1, 7, 37, 64, 10 ** 6])
@pytest.mark.parametrize("name", sorted(TABLES))
def test_schedule_is_safe_tight_and_complete(name, chunk):
    nbr = TABLES[name]
    npatch = nbr.shape[0]
    s = B.host_schedule(nbr, chunk)
    ck, n = s["chunk"], s["nchunk"]
    assert 1 <= ck <= npatch and n == -(-npatch // ck)
    if 0 < chunk <= npatch:
        assert ck == chunk
    assert sorted(s["up_order"]) == list(range(n)) and sorted(s["step_order"]) == list(range(n))
    upos = np.empty(n, dtype=int)
    upos[s["up_order"]] = np.arange(n)
    need = np.zeros(n, dtype=int)
    for p in range(npatch):
        c = p // ck
        qs = nbr[p][nbr[p] >= 0]
        need[c] = max(need[c], upos[c], upos[qs // ck].max())
    assert np.array_equal(s["ready"], need)                      # safe (>=) and tight (==)
    r = s["ready"][s["step_order"]]
    assert np.all(np.diff(r) >= 0)                               # chunks step in order of readiness
    assert abs(s["makespan"] - simulate(npatch, ck, s["up_order"], s["ready"], s["step_order"])) < 1e-9


def test_periodic_stack_starts_after_three_uploads_and_default_chunk_is_the_best_candidate():
    s = B.host_schedule(TABLES["cube8"], 64)                     # one z-slab of patches per chunk
    assert list(s["up_order"]) == [7, 0, 1, 2, 3, 4, 5, 6]       # last slab first: slab 0 needs it
    assert list(s["ready"]) == [2, 3, 4, 5, 6, 7, 7, 7]          # slab c waits for slab c+1; three slabs wait for the last upload
    assert s["step_order"][0] == 0
    best = B.host_schedule(TABLES["cube8"], 0)
    assert best["chunk"] == 64
    for k in (1, 2, 3, 4, 6, 8, 12, 16, 24, 32, 48, 64):
        ck = -(-512 // k)
        assert best["makespan"] <= B.host_schedule(TABLES["cube8"], ck)["makespan"] + 1e-9
    assert B.host_schedule(W.neighbour_table((16, 16, 16), (True,) * 3), 0)["chunk"] == 256     # config 3: a slab again


def test_schedule_rejects_bad_tables():
    lib = B.load_library()
    nbr = TABLES["slabs"].copy()
    a, b_ = C.c_int32(0), C.c_int32(0)
    args = lambda t, cap=8: (t.ctypes.data_as(C.c_void_p), t.shape[0], 0, C.byref(a), C.byref(b_), None, None, None, cap, None)
    assert lib.mhd_bunch_host_schedule(*args(nbr)) == 0 and b_.value >= 1
    bad = nbr.copy(); bad[3, 5] = 8
    assert lib.mhd_bunch_host_schedule(*args(bad)) == -1
    up = np.zeros(1, dtype=np.int32)
    assert lib.mhd_bunch_host_schedule(nbr.ctypes.data_as(C.c_void_p), 8, 1, C.byref(a), C.byref(b_),
                                       up.ctypes.data_as(C.c_void_p), None, None, 1, None) == -2       # capacity too small
    assert lib.mhd_bunch_host_schedule(None, 8, 1, C.byref(a), C.byref(b_), None, None, None, 0, None) == -1


# ---------------------------------------------------------------- ring mode: the planner ----
def _need(nbr, chunk):
    C = (len(nbr) + chunk - 1) // chunk
    return [sorted({q // chunk for p in range(c * chunk, min(len(nbr), (c + 1) * chunk)) for q in nbr[p] if q >= 0} | {c})
            for c in range(C)]


@pytest.mark.parametrize("P,chunk,R", [((2, 2, 8), 4, 3), ((2, 2, 8), 4, 5), ((4, 4, 4), 16, 3), ((4, 4, 4), 8, 6), ((8, 8, 8), 64, 4),
                                       ((3, 2, 5), 6, 3), ((2, 2, 2), 8, 1), ((4, 4, 4), 5, 13)])
def test_ring_plan_keeps_every_needed_chunk_resident_and_never_overfills(P, chunk, R):
    """mhd_bunch_ring_plan replayed on the host: before step c every chunk holding a neighbour of chunk
    c sits in a slot, no slot holds two chunks, a chunk is only evicted when the step at hand does not
    need it, and a periodic stack of slabs costs exactly two uploads more than it has slabs."""
    nbr = W.neighbour_table(P, (True, True, True))
    pl = B.ring_plan(nbr, chunk, R)
    need = _need(nbr, chunk)
    assert pl is not None and pl["nchunk"] == len(need)
    slot_chunk, u = {}, 0
    for c in range(pl["nchunk"]):
        while u < len(pl["up_chunk"]) and pl["up_step"][u] == c:
            s, x = int(pl["up_slot"][u]), int(pl["up_chunk"][u])
            assert 0 <= s < R and x in need[c] and x not in slot_chunk.values()
            assert slot_chunk.get(s) not in need[c]               # never evicts what the step needs
            slot_chunk[s] = x
            u += 1
        resident = set(slot_chunk.values())
        assert set(need[c]) <= resident and len(slot_chunk) <= R
        assert slot_chunk[int(pl["step_slot"][c])] == c
    assert u == len(pl["up_chunk"])
    if P == (2, 2, 8) and R == 3:
        assert len(pl["up_chunk"]) == 8 + 2                        # slabs 7 and 0 come twice
    if R >= pl["nchunk"]:
        assert len(pl["up_chunk"]) == pl["nchunk"]                 # everything fits: one upload each


def test_ring_plan_refuses_a_window_that_cannot_hold_a_neighbourhood():
    nbr = W.neighbour_table((2, 2, 8), (True, True, True))
    assert B.ring_plan(nbr, 4, 2) is None                          # a slab needs itself and both neighbours
    assert B.ring_plan(nbr, 4, 3) is not None
