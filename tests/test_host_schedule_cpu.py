"""Host logic of the host-streaming path (include/mhd_bunch.h, mhd_bunch_host_schedule): the
upload schedule is computed from the neighbour table alone, so it is checked here without a
GPU -- safety (no chunk steps before every plane its kernels read has been uploaded: its own
patches, its in-plane neighbours whole, the guard-width layers of its z-neighbours), tightness,
completeness (every plane of every patch crosses PCIe exactly once), the simulated makespan
against a pipeline simulation typed in this file, and the library's choice of chunk size."""
import ctypes as C

import numpy as np
import pytest

from paper_2508_09568_b200 import binding as B
from paper_2508_09568_b200 import workloads as W

TABLES = {
    "cube8": W.neighbour_table((8, 8, 8), (True, True, True)),          # config 2
    "slabs": W.neighbour_table((1, 1, 8), (True, True, True)),
    "pair": W.neighbour_table((2, 2, 2), (True, True, True)),           # the same patch is the +z and the -z neighbour
    "paper300": W.neighbour_table((5, 6, 10), (True, True, True)),      # bunch of 300
    "single": W.neighbour_table((1, 1, 1), (True, True, True)),
}


def simulate(npatch, chunk, nz, s, alpha=0.33, eps_up=2.0, eps_step=0.5, eps_dn=0.7):
    """Three in-order queues: uploads back to back, a step after the last piece it needs and
    after the previous step, a download after its step and after the previous download."""
    size = lambda c: min(chunk, npatch - c * chunk)
    t, t_up = 0.0, []
    for q, k0, k1 in zip(s["piece_chunk"], s["piece_k0"], s["piece_k1"]):
        t += size(q) * (k1 - k0) / nz + eps_up
        t_up.append(t)
    t_step = t_dn = 0.0
    for u in range(s["nunit"]):
        sz = size(s["unit_chunk"][u]) * (s["unit_zb"][u] - s["unit_za"][u]) / nz
        t_step = max(t_step, t_up[s["ready"][u]]) + alpha * sz + eps_step
        t_dn = max(t_dn, t_step) + sz + eps_dn
    return t_dn


def planes_read(nbr, ck, c, za, zb, nz, g):
    """What the step of planes [za, zb) of chunk c reads, as a set of (patch, plane): O1 -- guard zones
    come from the neighbours' interiors, at most g cells deep (plane k of an o_z = +1 neighbour is the
    patch's plane nz + k, plane k of an o_z = -1 neighbour its plane k - nz)."""
    need = set()
    layered = g >= 1 and 2 * g + 1 <= nz <= 64
    for p in range(c * ck, min(len(nbr), (c + 1) * ck)):
        for cls in range(27):
            q = nbr[p][cls]
            if q < 0:
                continue
            oz = cls // 9 - 1
            if not layered:
                need |= {(q, k) for k in range(nz)}
            else:
                need |= {(q, k) for k in range(nz) if za - g <= k + oz * nz < zb + g}
    return need


@pytest.mark.parametrize("nz,g,bands", [(32, 3, 1), (32, 3, 4), (6, 3, 2), (1, 0, 1), (16, 3, 2), (64, 3, 0)])
@pytest.mark.parametrize("chunk", [0, 1, 7, 37, 64, 10 ** 6])
@pytest.mark.parametrize("name", sorted(TABLES))
def test_schedule_is_safe_tight_and_complete(name, chunk, nz, g, bands):
    nbr = TABLES[name]
    npatch = nbr.shape[0]
    if npatch * nz > 9000 and chunk in (1, 7):
        pytest.skip("set arithmetic over every plane: covered by the smaller tables")
    s = B.host_schedule(nbr, chunk, nz=nz, guard=g, bands=bands)
    ck, n = s["chunk"], s["nchunk"]
    assert 1 <= ck <= npatch and n == -(-npatch // ck) and s["bands"] >= 1
    if 0 < chunk <= npatch:
        assert ck == chunk
    # completeness: the pieces of a chunk partition its planes, and so do the units (in chunk order, bands ascending)
    seen, landed_after = {}, {}             # (patch, plane) -> index of the piece that carries it
    for i, (q, k0, k1) in enumerate(zip(s["piece_chunk"], s["piece_k0"], s["piece_k1"])):
        assert 0 <= q < n and 0 <= k0 < k1 <= nz
        for k in range(k0, k1):
            assert (q, k) not in seen, "plane uploaded twice"
            seen[(q, k)] = i
        for p in range(q * ck, min(npatch, (q + 1) * ck)):
            for k in range(k0, k1):
                landed_after[(p, k)] = i
    assert len(seen) == n * nz
    units = list(zip(s["unit_chunk"], s["unit_za"], s["unit_zb"]))
    assert units == sorted(units) and [u[0] for u in units if u[1] == 0] == list(range(n))
    for c in range(n):
        mine = [(za, zb) for q, za, zb in units if q == c]
        assert mine[0][0] == 0 and mine[-1][1] == nz and all(a[1] == b_[0] for a, b_ in zip(mine, mine[1:]))
        assert len(mine) == 1 or (c in (0, n - 2, n - 1) and all(zb - za >= 8 for za, zb in mine))
    # safety (>=) and tightness (==): ready[u] is the last piece that carries something unit u reads;
    # units step in order, so ready does not decrease
    for u, (c, za, zb) in enumerate(units):
        last = max(landed_after[x] for x in planes_read(nbr, ck, c, za, zb, nz, g))
        assert s["ready"][u] == max(last, s["ready"][u - 1] if u else -1)
    assert abs(s["makespan"] - simulate(npatch, ck, nz, s)) < 1e-9


@pytest.mark.parametrize("seed", range(12))
def test_schedule_on_arbitrary_tables(seed):
    """The planner assumes nothing about the arrangement: random tables (any patch may be anybody's neighbour in
    any class, some entries -1), random chunk sizes, plane counts, guard widths and band counts -- the same three
    properties must hold (every plane uploaded once, ready[] safe and tight, units partition their chunks)."""
    rng = np.random.default_rng(1000 + seed)
    npatch = int(rng.integers(1, 40))
    nbr = rng.integers(-1, npatch, size=(npatch, 27)).astype(np.int32)
    nbr[:, 13] = np.arange(npatch)
    nz = int(rng.choice([1, 5, 7, 16, 33, 64, 70]))
    g = int(rng.choice([0, 1, 3]))
    chunk = int(rng.integers(1, npatch + 1))
    bands = int(rng.integers(1, 6))
    s = B.host_schedule(nbr, chunk, nz=nz, guard=g, bands=bands)
    ck, n = s["chunk"], s["nchunk"]
    landed_after, seen = {}, set()
    for i, (q, k0, k1) in enumerate(zip(s["piece_chunk"], s["piece_k0"], s["piece_k1"])):
        for k in range(k0, k1):
            assert (q, k) not in seen
            seen.add((q, k))
            for p in range(q * ck, min(npatch, (q + 1) * ck)):
                landed_after[(p, k)] = i
    assert len(seen) == n * nz
    units = list(zip(s["unit_chunk"], s["unit_za"], s["unit_zb"]))
    assert units == sorted(units)
    for c in range(n):
        mine = [(za, zb) for q, za, zb in units if q == c]
        assert mine[0][0] == 0 and mine[-1][1] == nz and all(a[1] == b_[0] for a, b_ in zip(mine, mine[1:]))
    for u, (c, za, zb) in enumerate(units):
        last = max(landed_after[x] for x in planes_read(nbr, ck, c, za, zb, nz, g))
        assert s["ready"][u] == max(last, s["ready"][u - 1] if u else -1)
    assert abs(s["makespan"] - simulate(npatch, ck, nz, s)) < 1e-9


def test_periodic_stack_never_waits_for_the_bulk_of_a_z_neighbour():
    s = B.host_schedule(TABLES["cube8"], 64, bands=1)             # one z-slab of patches per chunk, stepped whole
    pieces = list(zip(s["piece_chunk"], s["piece_k0"], s["piece_k1"]))
    # slab 0 whole, then the bottom layer of slab 1 and the top layer of slab 7: slab 0 steps after ONE slab
    assert pieces[:3] == [(0, 0, 32), (1, 0, 3), (7, 29, 32)] and s["ready"][0] == 2
    # every later slab waits for the rest of itself and the bottom layer of the next one only
    assert pieces[3:5] == [(1, 3, 32), (2, 0, 3)] and s["ready"][1] == 4
    assert pieces[-1] == (7, 3, 29) and s["ready"][7] == len(pieces) - 1 and s["ready"][6] == len(pieces) - 2
    # the last upload releases ONE slab (the whole-chunk schedule released three, 1.45 of the transfer time)
    assert s["makespan"] < 512 * 1.26
    # bands: the first slab starts stepping after a quarter of it (+ guard planes) is up, the last upload
    # releases a quarter of the last slab
    t = B.host_schedule(TABLES["cube8"], 64, bands=4)
    pieces = list(zip(t["piece_chunk"], t["piece_k0"], t["piece_k1"]))
    units = list(zip(t["unit_chunk"], t["unit_za"], t["unit_zb"]))
    assert pieces[:2] == [(0, 0, 11), (7, 29, 32)] and t["ready"][0] == 1
    assert units[:4] == [(0, 0, 8), (0, 8, 16), (0, 16, 24), (0, 24, 32)] and units[-1] == (7, 24, 32) and t["nunit"] == 17
    assert pieces[-1] == (7, 27, 29) and t["makespan"] < 512 * 1.28      # every extra H2D copy costs 2 patch-times of start-up
    best = B.host_schedule(TABLES["cube8"], 0)
    for k in (1, 2, 3, 4, 6, 8, 12, 16, 24, 32, 48, 64, 96, 128):
        for bands in (1, 2, 4):
            assert best["makespan"] <= B.host_schedule(TABLES["cube8"], -(-512 // k), bands=bands)["makespan"] * 1.002
    assert best["makespan"] < 512 * 1.26 and (best["chunk"], best["bands"]) == (64, 2)
    # thin patches: no layers, no bands, every need is a whole chunk
    t = B.host_schedule(TABLES["cube8"], 64, nz=6, guard=3, bands=4)
    assert all(k0 == 0 and k1 == 6 for k0, k1 in zip(t["piece_k0"], t["piece_k1"])) and t["npiece"] == 8 and t["nunit"] == 8


def test_schedule_rejects_bad_tables():
    lib = B.load_library()
    nbr = TABLES["slabs"].copy()
    o = [C.c_int32(0) for _ in range(4)]
    ptr = lambda t: t.ctypes.data_as(C.c_void_p)
    def call(t, npatch=8, nz=32, chunk=0, arr=None, cap=64):
        return lib.mhd_bunch_host_schedule(ptr(t) if t is not None else None, npatch, nz, 3, chunk, 0, C.byref(o[0]), C.byref(o[1]),
                                           C.byref(o[2]), arr, None, None, C.byref(o[3]), None, None, None, None, cap, None)
    assert call(nbr) == 0 and o[0].value >= 1 and o[2].value >= 1 and o[3].value >= 1
    bad = nbr.copy(); bad[3, 5] = 8
    assert call(bad) == -1
    up = np.zeros(1, dtype=np.int32)
    assert call(nbr, chunk=1, arr=ptr(up), cap=1) == -2          # capacity too small
    assert call(None) == -1
    assert call(nbr, nz=0) == -1


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
