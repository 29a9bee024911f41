#!/usr/bin/env python
"""bench.py -- throughput of the bunch MHD update on B200 (cell-updates/s).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c2|c3|c3f64|c2f64|small|c4]
                    [--sub c2f64,c3,c3f64 | --sub none]
    python bench.py --impl reference ...      # the CPU oracle on a bounded sample

A step = one pass of the whole hot path over the bunch: fill_guards -> cfl_dt (dt stays
on the device) -> step.  The headline workload is BASELINE.json config 2 (512 patches of
32^3, fp32, seeded turbulence-like field); the metric is quoted "(fp32/fp64)", so the same
JSON line carries sub-records for the config-2 shape in fp64 and for config 3 (4096 patches)
in fp32 and fp64, each with its own value, roofline fraction and end-to-end number.
`--workload c4` runs BASELINE.json's bunching sweep instead.  Prints ONE JSON line (see
DESIGN.md, "Measurement").  Multi-GPU: the path does not shard (north_star: one GPU) --
under torchrun every rank runs an independent replica ("replicas only").
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2508_09568_b200 import workloads as W  # noqa: E402

METRIC = "mhd_cell_updates_per_sec"
UNIT = "cell-updates/s"

WORKLOADS = {
    # name: (N, n, dtype, description)
    "c2": (256, 32, "f32", "config2: 512 patches x 32^3, fp32, periodic 256^3 turbulence-like field"),
    "c3": (512, 32, "f32", "config3: 4096 patches x 32^3, fp32, periodic 512^3"),
    "c3f64": (512, 32, "f64", "config3: 4096 patches x 32^3, fp64, periodic 512^3"),
    "c2f64": (256, 32, "f64", "config2 shape in fp64: 512 patches x 32^3"),
    "small": (64, 32, "f32", "8 patches x 32^3, fp32 (smoke size)"),
}
# the CPU oracle's bounded samples: the same seeded field construction on a cut of the cube
SAMPLE_1 = (64, 64, 64)          # 8 patches of 32^3, single thread
SAMPLE_ALL = (128, 128, 64)      # 32 patches of 32^3, OpenMP over patches on all host cores
TRAFFIC_FILE = os.path.join("profiles", "r3_ncu_traffic.txt")


def peaks():
    """Measured roofline denominators (driver-written), else the profiling guide's fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)), "source": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback"}


# Algorithmic work per interior cell-update of each kernel class.
# bytes: compulsory HBM reads + writes of that pass with perfect on-chip reuse, in units of
#        sizeof(real); r(a,b) = volume ratio of a pass that covers cells [-a, n-1+b].
# flops: counted on the oracle's source by oracle/opcount.cpp at 32^3 (add+mul+div+sqrt,
#        FMA = 2): whole step 3625.4, cfl 86; HLLD solve 392, HLLD-2D edge solve 453.
STEP_FLOPS_32 = 3625.4
CFL_FLOPS = 86.0
STEP_FLOPS_2D, CFL_FLOPS_2D = 3088.2, 66.0     # `oracle/opcount 32 2d`: patches of 32 x 32 x 1 cells (no z face, three edges)
# configs 0 and 1 of BASELINE.json: small bunches (256 and 65 536 cells) -- a step is a handful of launches and
# the rate is set by launch latency, so these records carry the per-step time and the launch count, and an ALU
# fraction only for the 2D tile kernel
SMALL = {
    "c0": ("sod", "f64", "config0: 1D Sod tube, 8 patches x 32 cells, fp64, outflow ends"),
    "c1": ("ot", "f64", "config1: Orszag-Tang 256^2, 64 patches x 32^2, fp64, periodic"),
    "c1f32": ("ot", "f32", "config1: Orszag-Tang 256^2, 64 patches x 32^2, fp32, periodic"),
    "ot2048f64": ("ot2048", "f64", "Orszag-Tang 2048^2, 4096 patches x 32^2, fp64 (a 2D bunch large enough to fill the GPU)"),
    "ot2048": ("ot2048", "f32", "Orszag-Tang 2048^2, 4096 patches x 32^2, fp32 (a 2D bunch large enough to fill the GPU)"),
}


def algorithmic_work(cls, n, ng=3):
    r = lambda a, b: ((n + a + b) / n) ** 3
    f1 = (n + 1) / n
    riemann_flops = 3 * f1 * (28 + 392) + 3 * f1 * f1 * (104 + 453) + 81     # face + edge states, solves, update
    table = {
        # class: (values per cell, flops per cell, bound)
        "fill_guards": (2 * 8 * (r(ng, ng) - 1.0), 0.0, "hbm"),
        "sync_closing_faces": (2 * 3 / n, 0.0, "hbm"),
        "cfl": (8 + 3 / n, CFL_FLOPS, "hbm"),
        "predict": (8 * r(2, 3) + 38 * r(1, 1), STEP_FLOPS_32 - riemann_flops, "hbm"),
        "riemann_update": (38 * r(1, 1) + 8 + 8, riemann_flops, "alu"),
        "step_onepass": (8 * r(2, 3) + 8, STEP_FLOPS_32, "alu"),
        "step_onepass_cfl": (8 * r(2, 3) + 8, STEP_FLOPS_32 + CFL_FLOPS, "alu"),
        # staged path (general, collapsed dimensions)
        "prim": (8 * r(2, 3) + 8 * r(2, 2), 40.0, "hbm"),
        "emf0": ((3 + 3) * r(2, 2) + 3 * r(1, 2), 70.0, "hbm"),
        "hlld_flux": (3 * ((5 + 7) * r(1, 1) + 3 * r(1, 2) + 5 * r(0, 1)), 3 * f1 * 420, "alu"),
        "emf_2d": (3 * ((5 + 12 + 2) * r(1, 1) + 3 * r(1, 2) + 1 * r(0, 1)), 3 * f1 * f1 * 557, "alu"),
        "update": (8 + 15 * r(0, 1) + 3 * r(0, 1) + 8, 81.0, "hbm"),
    }
    return table.get(cls)


def ncu_traffic(workload, cls):
    """DRAM bytes per launch of a kernel class from the committed ncu capture of this round
    (a cross-reference, not something this run measured), or None."""
    try:
        return json.load(open(os.path.join(ROOT, TRAFFIC_FILE))).get(workload, {}).get(cls)
    except Exception:
        return None


def aggregate_over_ranks(ms, cells_per_rank, steps, world, device=None):
    """Whole-job throughput of N independent replicas: every rank processed cells_per_rank
    cells per step; the job's time is the MAX over ranks (all_reduce), the value their sum
    over that time.  Returns (value, ms_max).  world == 1 needs no process group."""
    if world > 1:
        import torch
        import torch.distributed as dist
        t = torch.tensor([ms], dtype=torch.float64, device=device or "cpu")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    return world * cells_per_rank * steps / (ms * 1e-3), ms


class ClockSampler(threading.Thread):
    """nvidia-smi clocks and throttle reasons during the timed region."""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.stop_flag = index, [], False

    def run(self):
        while not self.stop_flag:
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                p = [x.strip() for x in out.strip().split(",")]
                if len(p) >= 7:
                    self.rows.append(p)
            except Exception:
                pass
            time.sleep(0.1)

    def summary(self):
        self.stop_flag = True
        self.join(timeout=6)
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        mhz = sorted(float(r[0]) for r in self.rows if r[0].replace(".", "").isdigit())
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(r[3 + k].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": mhz[len(mhz) // 2] if mhz else None, "sm_max_mhz": float(self.rows[0][1]),
                "reasons": reasons, "samples": len(self.rows)}


def run_oracle_sample(steps, warmup, all_cores=False):
    """The oracle as it stands on a bounded sample; returns dict(value, seconds, cores, sample).
    all_cores: the same source built with -fopenmp (`parallel for` over patches, patches being
    independent between guard fills) on every host core."""
    import oracle
    N = SAMPLE_ALL if all_cores else SAMPLE_1
    w = W.turbulence(N=N, n=32, dtype=np.float32, config=2)
    key = "f64_omp" if all_cores else "f64"
    cores = oracle.threads(os.cpu_count() or 1) if all_cores else 1
    o = oracle.Oracle(w.n, w.npatch, w.gamma, w.dx, dtype=key)
    U = w.U.astype(np.float64)

    def one(U):
        o.fill_guards(U, w.nbr)
        dt = o.cfl_dt(U, 0.4)
        return o.step(U, dt)
    for _ in range(warmup):
        U = one(U)
    t0 = time.perf_counter()
    for _ in range(steps):
        U = one(U)
    el = time.perf_counter() - t0
    assert np.isfinite(U).all()
    desc = (f"config-2 field construction on {N[0]}x{N[1]}x{N[2]} cells = {w.npatch} patches x 32^3, fp64 oracle, "
            f"fill+cfl+step, {steps} steps after {warmup} warm-up, " +
            (f"OpenMP over patches on {cores} threads (nproc = {os.cpu_count()})" if all_cores else "single thread"))
    return {"value": w.cells * steps / el, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc, "seconds": el}


# ------------------------------------------------------------------- one workload ----
def measure(name, args, local, world, rank, field_cache, headline):
    """Resident loop, per-class times with rooflines, and the end-to-end host-buffer loop of one
    workload.  Returns the record (dict)."""
    import torch
    import torch.distributed as dist
    from paper_2508_09568_b200.binding import MhdBunch, measure_alu_peak
    N, n, dtype, wdesc = WORKLOADS[name]
    npd = np.float32 if dtype == "f32" else np.float64
    if N not in field_cache:                       # the fp64 field serves both types (same values as a direct build)
        field_cache.clear()
        field_cache[N] = W.turbulence(N=N, n=n, dtype=np.float64, config=2)
    w = field_cache[N]
    b = MhdBunch(w.n, w.npatch, w.nbr, w.gamma, w.dx, dtype=dtype, device=local)
    b.load(w.U if dtype == "f64" else w.U.astype(np.float32))
    b.set_path(args.path)
    if args.fused_cfl != 2 and b.path == "onepass":
        b.set_tuning("fused_cfl", args.fused_cfl)
    stream = b.stream
    courant = 0.4
    steps = args.steps if headline else max(3, min(args.steps, args.sub_steps))

    def one_step():
        b.fill_guards()
        if args.explicit_fill:
            b.sync_guards()        # write the guard shell to HBM every step (k_fill_guards), as a caller that reads it would
        b.cfl_dt(courant, sync=False)
        b.step_dev()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def totals():
        """mass and total energy over the interior cells (fp64 sums on the device, outside the timed region)"""
        v = b.view()
        g = [3 if k > 1 else 0 for k in w.n]
        I = v[:, :, g[2]:g[2] + w.n[2], g[1]:g[1] + w.n[1], g[0]:g[0] + w.n[0]]
        return float(I[0].sum(dtype=torch.float64)), float(I[4].sum(dtype=torch.float64))

    warm = max(3, args.warmup)
    for _ in range(warm):
        one_step()
    barrier()
    tot0 = totals()
    b.fill_guards()            # looking at the buffer made the library re-validate the closing faces: do it here, untimed
    barrier()
    l0 = b.launches
    sampler = ClockSampler(local)
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    with torch.cuda.stream(stream):
        ev0.record(stream)
        for _ in range(steps):
            one_step()
        ev1.record(stream)
    barrier()
    ms = ev0.elapsed_time(ev1)
    clocks = sampler.summary()
    launches = b.launches - l0
    bad = b.status()
    tot1 = totals()
    conservation = {"mass_rel_drift": abs(tot1[0] - tot0[0]) / abs(tot0[0]), "energy_rel_drift": abs(tot1[1] - tot0[1]) / abs(tot0[1]),
                    "note": "interior totals before/after the timed steps (periodic bunch: conserved up to round-off)"}
    value, ms = aggregate_over_ranks(ms, w.cells, steps, world, device="cuda")

    # ---- per-kernel-class device times (separate pass, events around every launch) ----
    b.fill_guards()
    b.set_timing(True)
    tsteps = min(steps, 10)
    for _ in range(tsteps):
        one_step()
    kt = b.kernel_times()
    b.set_timing(False)
    pk = peaks()
    esz = 4 if dtype == "f32" else 8
    alu_peak = measure_alu_peak(dtype, local)               # TFLOP/s, FMA-chain, measured now
    alu_nominal = 148 * (128 if dtype == "f32" else 64) * 2 * pk["sm_max_mhz"] * 1e6 / 1e12
    classes = {k: {"ms_per_step": v[0] / tsteps, "launches_per_step": v[1] / tsteps} for k, v in kt.items()}
    tot = sum(c["ms_per_step"] for c in classes.values())
    for k, c in classes.items():
        c["share"] = c["ms_per_step"] / tot
        a = algorithmic_work(k, n)
        # a class that does not run every step (e.g. the closing-face sync after the caller looked at the
        # buffer) has no per-step rate: no fraction is printed for it
        if a and c["launches_per_step"] >= 1.0:
            c["bound"] = a[2]
            c["alg_bytes_per_cell"] = a[0] * esz
            c["alg_flops_per_cell"] = a[1]
            c["alg_gbs"] = a[0] * esz * w.cells / (c["ms_per_step"] * 1e-3) / 1e9
            c["alg_tflops"] = a[1] * w.cells / (c["ms_per_step"] * 1e-3) / 1e12
            c["hbm_frac"] = c["alg_gbs"] / pk["hbm_gbs"]
            c["alu_frac"] = c["alg_tflops"] / alu_peak
    dom = max((k for k in classes if k != "misc"), key=lambda k: classes[k]["ms_per_step"])
    dc = classes[dom]
    per_launch_ms = dc["ms_per_step"] / dc["launches_per_step"]
    if dc.get("bound") == "alu":
        roofline = {"kernel": dom, "bound": "alu", "achieved": dc["alg_tflops"], "peak": alu_peak, "unit": "TFLOP/s",
                    "frac": dc["alu_frac"], "peak_source": "measured FMA chain (mhd_bunch_measure_alu_peak), FMA = 2 flops",
                    "peak_nominal": alu_nominal,
                    "alg_flops_per_launch": dc["alg_flops_per_cell"] * w.cells / dc["launches_per_step"]}
    else:
        roofline = {"kernel": dom, "bound": "hbm", "achieved": dc.get("alg_gbs"), "peak": pk["hbm_gbs"], "unit": "GB/s",
                    "frac": dc.get("hbm_frac"), "peak_source": pk["source"],
                    "alg_bytes_per_launch": dc.get("alg_bytes_per_cell", 0) * w.cells / dc["launches_per_step"]}
    roofline.update({"traffic": ncu_traffic(name, dom), "traffic_source": TRAFFIC_FILE, "avg_launch_ms": per_launch_ms,
                     "share_of_step": dc["share"], "hbm_frac": dc.get("hbm_frac"), "alu_frac": dc.get("alu_frac")})
    # whole-pass view: counted flops of step + cfl, compulsory traffic of a fully fused step
    pass_flops = STEP_FLOPS_32 + CFL_FLOPS
    step_view = {"alg_flops_per_cell": pass_flops, "alg_tflops": pass_flops * value / world / 1e12,
                 "alu_frac": pass_flops * value / world / 1e12 / alu_peak, "alu_peak_tflops": alu_peak,
                 "compulsory_bytes_per_cell": 16 * esz,
                 "hbm_frac_at_compulsory_bytes": 16 * esz * value / world / 1e9 / pk["hbm_gbs"]}

    # ---- end to end through the host-buffer path of the C ABI -------------------------
    # mhd_bunch_step_host: the bunch lives in pinned HOST memory (compact layout, interiors
    # only); every step uploads it, exchanges guards and steps on the GPU, and downloads the
    # new level, chunk by chunk on separate copy streams (include/mhd_bunch.h).  dt of a step
    # is the CFL step the previous call returned, so uploads, kernels and downloads overlap.
    e2e = None
    if not args.no_e2e:
        hl = b.host_attach(args.host_chunk)
        cur = b.download()
        hin = torch.from_numpy(W.to_compact(cur, w.n)).pin_memory()
        hout = torch.empty_like(hin).pin_memory()
        del cur
        esteps = max(2, min(steps, 10))
        _, dt_next = b.step_host(hin, hout, dt=0.0, courant=courant)      # warm-up, and the first dt
        hin, hout = hout, hin
        barrier()
        t0 = time.perf_counter()
        for _ in range(esteps):
            _, dt_next = b.step_host(hin, hout, dt=dt_next, courant=courant)   # synchronises
            hin, hout = hout, hin
        el = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([el], device="cuda", dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            el = float(t.item())
        assert bool(torch.isfinite(hin).all())
        e2e = {"value": world * w.cells * esteps / el, "unit": UNIT, "h2d_bytes_per_step": int(hl.host_bytes),
               "d2h_bytes_per_step": int(hl.host_bytes), "steps": esteps, "ms_per_step": 1e3 * el / esteps,
               "chunk_patches": int(hl.chunk_patches), "chunks": int(hl.nchunk), "bands": int(hl.bands), "overlapped": bool(hl.pipelined),
               "note": "mhd_bunch_step_host: compact host state (interiors only) uploaded from pinned memory, "
                       "stepped and downloaded every step in chunks (thin z-layers of the next chunk ahead of its bulk, first chunk and last two in z-bands) on library copy streams; wall clock"}
        del hin, hout
    rec = {"workload": name, "value": value, "unit": UNIT, "steps": steps, "warmup": warm, "ms_per_step": ms / steps,
           "dtype": dtype,
           "config": {"workload": wdesc, "patches": w.npatch, "patch": [n, n, n], "guard": 3, "courant": courant,
                      "chunk_patches": b.chunk, "step_path": b.path,
                      "parallelism": "replicas only" if world > 1 else "single GPU",
                      "l2": "state buffers (2 x %.0f MB) exceed the 126 MB L2; no flush needed" % (b.lay.state_bytes / 1e6)},
           "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "bad_cells": bad, "conservation": conservation,
           "roofline": roofline, "step_roofline": step_view, "kernel_classes": classes}
    b.close()
    del b
    torch.cuda.empty_cache()
    return rec


def measure_small(name, args, local):
    """Configs 0 and 1 (and a large 2D bunch): resident loop fill_guards -> cfl_dt -> step with CUDA events,
    launches per step, per-class device times, and for 2D bunches the tile kernel's ALU fraction."""
    import torch
    from paper_2508_09568_b200.binding import MhdBunch, measure_alu_peak
    kind, dtype, desc = SMALL[name]
    npd = np.float32 if dtype == "f32" else np.float64
    w = W.sod(256, 8, dtype=npd) if kind == "sod" else W.orszag_tang(2048 if kind == "ot2048" else 256, 32, dtype=npd)
    b = MhdBunch(w.n, w.npatch, w.nbr, w.gamma, w.dx, dtype=dtype, device=local)
    b.load(w.U)

    def one_step():
        b.fill_guards(); b.cfl_dt(0.4, sync=False); b.step_dev()
    steps = 200 if w.cells < (1 << 20) else max(3, min(args.steps, args.sub_steps))
    for _ in range(5):
        one_step()
    torch.cuda.synchronize()
    l0 = b.launches
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(b.stream):
        ev0.record(b.stream)
        for _ in range(steps):
            one_step()
        ev1.record(b.stream)
    torch.cuda.synchronize()
    ms = ev0.elapsed_time(ev1) / steps
    launches = (b.launches - l0) / steps
    b.set_timing(True)
    for _ in range(10):
        one_step()
    kt = b.kernel_times()
    b.set_timing(False)
    classes = {k: {"ms_per_step": v[0] / 10, "launches_per_step": v[1] / 10} for k, v in kt.items()}
    rec = {"workload": name, "dtype": dtype, "value": w.cells / (ms * 1e-3), "unit": UNIT, "steps": steps, "ms_per_step": ms,
           "config": {"workload": desc, "patches": w.npatch, "patch": list(w.n), "guard": 3, "courant": 0.4, "step_path": b.path},
           "gpu_launches_per_step": launches, "bad_cells": b.status(), "kernel_classes": classes,
           "note": "events around every launch inflate the per-class times of kernels this short; ms_per_step is the untimed loop"}
    if "step_tile2d" in classes and w.n[1] > 1:      # 2D bunches: the tile kernel against the flops counted in 2D
        tk = classes["step_tile2d"]["ms_per_step"]
        alu_peak = measure_alu_peak(dtype, local)
        rec["roofline"] = {"kernel": "step_tile2d", "bound": "alu", "achieved": STEP_FLOPS_2D * w.cells / (tk * 1e-3) / 1e12,
                           "peak": alu_peak, "unit": "TFLOP/s", "frac": STEP_FLOPS_2D * w.cells / (tk * 1e-3) / 1e12 / alu_peak,
                           "peak_source": "measured FMA chain (mhd_bunch_measure_alu_peak), FMA = 2 flops",
                           "alg_flops_per_launch": STEP_FLOPS_2D * w.cells, "avg_launch_ms": tk, "traffic": ncu_traffic(name, "step_tile2d"), "traffic_source": TRAFFIC_FILE,
                           "share_of_step": tk / sum(c["ms_per_step"] for c in classes.values())}
    b.close()
    del b
    torch.cuda.empty_cache()
    return rec


# ---------------------------------------------------------------- config 4: the sweep ----
ARRANGE = {1: (1, 1, 1), 8: (2, 2, 2), 64: (4, 4, 4), 300: (5, 6, 10), 512: (8, 8, 8), 4096: (16, 16, 16)}


def replicated_bunch(n, P, dtype, device, max_side=256, stream=None):
    """A periodic bunch of P patches whose global field would be too large to build on the host:
    the seeded field is built on a block of at most max_side cells per side and repeated
    periodically ON THE DEVICE (patch (px,py,pz) holds block patch (px mod Bx, ...)), which is again
    a periodic field.  Returns (MhdBunch, Workload of the block, block arrangement)."""
    import torch
    from paper_2508_09568_b200.binding import MhdBunch
    B = tuple(min(p, max(1, max_side // n)) for p in P)
    wb = W.turbulence(N=tuple(n * k for k in B), n=n, dtype=np.float32 if dtype == "f32" else np.float64, config=2, patches=B)
    nbr = W.neighbour_table(P, (True, True, True))
    npatch = P[0] * P[1] * P[2]
    dx = tuple(1.0 / (n * max(P)) for _ in range(3))
    b = MhdBunch(wb.n, npatch, nbr, wb.gamma, dx, dtype=dtype, device=device, workspace_bytes=1 << 30, stream=stream)
    src = torch.from_numpy(wb.U).to(b.device)                 # [8, block patches, mz, my, mx]
    v = b.view()
    ids = np.arange(npatch)
    px, py, pz = ids % P[0], (ids // P[0]) % P[1], ids // (P[0] * P[1])
    img = (px % B[0]) + B[0] * ((py % B[1]) + B[1] * (pz % B[2]))
    for q in range(B[0] * B[1] * B[2]):
        sel = torch.from_numpy(ids[img == q]).to(b.device)
        for f in range(8):                                    # field by field: no large temporaries
            v[f].index_copy_(0, sel, src[f, q].unsqueeze(0).expand(len(sel), -1, -1, -1))
    torch.cuda.synchronize(b.device)       # the copies ran on torch's current stream, which need not be the bunch's
    return b, wb, B


def replay_us_per_step(b, one, steps):
    """Device time per step of `steps` back-to-back steps captured in ONE CUDA graph and replayed:
    the kernels of the loop with no per-call launch cost between them.  The capture holds kernel launches only
    (the loop neither copies nor synchronises).  None if the capture is refused."""
    import torch
    try:
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=b.stream):
            for _ in range(steps):
                one()
        b.stream.synchronize()
        best = None
        for _ in range(3):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            with torch.cuda.stream(b.stream):
                e0.record()
                g.replay()
                e1.record()
            e1.synchronize()
            t = e0.elapsed_time(e1) * 1e3 / steps
            best = t if best is None else min(best, t)
        del g
        return best
    except Exception as e:                      # a capture that failed leaves nothing half-done on the stream
        print("graph capture refused: %s" % str(e).splitlines()[0][:120], file=sys.stderr)
        return None


def sweep(args, local):
    """BASELINE.json config 4: patch sizes x bunch sizes, fp32, config-2 field construction; per
    point the resident loop's rate with per-call launches (wall clock), the same steps replayed from
    one CUDA graph (device time, no launch cost between kernels) and the launch-overhead share
    1 - graph/wall that the paper's bunching study is about (Fig. 5)."""
    import torch
    from paper_2508_09568_b200.binding import MhdBunch
    sizes = [int(x) for x in args.sizes.split(",")]
    bunches = [int(x) for x in args.bunches.split(",")]
    pts = [(n, k) for n in sizes for k in bunches] + ([(24, 300)] if 24 in sizes else [])
    out = []
    for n, k in pts:
        P = ARRANGE[k]
        N = tuple(n * p for p in P)
        rec = {"patch": n, "bunch": k, "cells": k * n ** 3}
        try:
            side = torch.cuda.Stream(device=local)     # a stream of its own: the default stream cannot be captured
            if max(N) > 512:
                b, wb, B = replicated_bunch(n, P, "f32", local, stream=side)
                rec["field"] = "block of %dx%dx%d patches repeated periodically on the device" % B
            else:
                w = W.turbulence(N=N, n=n, dtype=np.float32, config=2, patches=P)
                b = MhdBunch(w.n, w.npatch, w.nbr, w.gamma, w.dx, dtype="f32", device=local, stream=side)
                b.load(w.U)
            if args.fused_cfl != 2 and b.path == "onepass":
                b.set_tuning("fused_cfl", args.fused_cfl)
        except Exception as e:
            rec["skipped"] = str(e).splitlines()[0][:100]
            out.append(rec)
            continue

        def one():
            b.fill_guards(); b.cfl_dt(0.4, sync=False); b.step_dev()
        steps = max(3, min(args.steps, 20))
        for _ in range(3):
            one()
        torch.cuda.synchronize()
        l0 = b.launches
        t0 = time.perf_counter()
        for _ in range(steps):
            one()
        torch.cuda.synchronize()
        wall = (time.perf_counter() - t0) / steps
        launches = (b.launches - l0) / steps
        graph_us = replay_us_per_step(b, one, steps)
        b.set_timing(True)
        for _ in range(steps):
            one()
        kt = b.kernel_times()
        b.set_timing(False)
        busy = sum(v[0] for v in kt.values()) * 1e-3 / steps
        share = None if graph_us is None else max(0.0, 1.0 - graph_us / (wall * 1e6))
        rec.update({"step_path": b.path, "launches_per_step": launches, "wall_us": wall * 1e6, "graph_us": graph_us,
                    "busy_us": busy * 1e6, "value": rec["cells"] / wall,
                    "value_graph": None if graph_us is None else rec["cells"] / (graph_us * 1e-6),
                    "launch_overhead_share": share,
                    "share_is": "1 - (device time per step of the timed steps replayed from one CUDA graph) / (wall time per step with per-call launches)",
                    "bad_cells": b.status()})
        b.close()
        del b
        torch.cuda.empty_cache()
        out.append(rec)
        print(json.dumps(rec), file=sys.stderr, flush=True)
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c2", choices=sorted(WORKLOADS) + sorted(SMALL) + ["c4"])
    ap.add_argument("--sub", default="c2f64,c3,c3f64,c0,c1,c1f32,ot2048,ot2048f64",
                    help="sub-records added to the default (c2) line: comma list of workloads, or 'none'")
    ap.add_argument("--sub-steps", type=int, default=20, help="timed steps of each sub-record")
    ap.add_argument("--cpu-steps", type=int, default=20, help="oracle steps for the cpu_baseline legs")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--host-chunk", type=int, default=0, help="patches per chunk of the host-streaming path (0: library default)")
    ap.add_argument("--path", default="auto", choices=["auto", "staged", "two_kernel", "onepass"],
                    help="which CUDA implementation of the step runs (include/mhd_bunch.h, MHD_PATH_*)")
    ap.add_argument("--explicit-fill", action="store_true",
                    help="materialise the guard shell in HBM every step (the fill is otherwise folded into the step's halo loads)")
    ap.add_argument("--fused-cfl", type=int, default=2, choices=[0, 1, 2],
                    help="one-pass step: reduce the new level's CFL rates in the step's epilogue (MHD_TUNE_FUSED_CFL; "
                         "2 = the library's choice: on bunches of at most one wave of tiles)")
    ap.add_argument("--sizes", default="16,24,32,64", help="c4: patch sizes")
    ap.add_argument("--bunches", default="1,8,64,512,4096", help="c4: bunch sizes")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))

    # ---------------------------------------------------------------- reference arm ----
    if args.impl == "reference":
        if rank != 0:
            return 0
        steps = max(1, args.steps)
        warm = max(0, min(args.warmup, 2))          # the oracle has no caches to warm: two steps at most
        r = run_oracle_sample(steps, warm)
        wdesc = WORKLOADS[args.workload if args.workload in WORKLOADS else "c2"][3]
        line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
                "warmup": warm, "ms_per_step": 1e3 * r["seconds"] / steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": wdesc, "sample": r["sample"]},
                "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")},
                "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                "gpu_launches": 0}
        print(json.dumps(line))
        return 0

    # --------------------------------------------------------------------- our arm ----
    import torch
    import torch.distributed as dist

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    if args.workload == "c4":
        pts = sweep(args, local) if rank == 0 else []
        if rank == 0:
            best = max((p for p in pts if "value" in p), key=lambda p: p["value"])
            print(json.dumps({"metric": METRIC, "value": best["value"], "unit": UNIT, "n_gpus": 1, "steps": args.steps,
                              "warmup": 3, "ms_per_step": best["wall_us"] / 1e3, "higher_is_better": True, "scaling": "weak",
                              "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                              "config": {"workload": "config4: bunching sweep, value = best point", "best": [best["patch"], best["bunch"]]},
                              "sweep": pts}))
        if world > 1:
            dist.destroy_process_group()
        return 0

    if args.workload in SMALL:
        if rank == 0:
            r = measure_small(args.workload, args, local)
            print(json.dumps({"metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": 1, "steps": r["steps"], "warmup": 5,
                              "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                              "dtype": r["dtype"], "data": "synthetic", "config": r["config"], "gpu_launches": r["gpu_launches_per_step"] * r["steps"],
                              "roofline": r.get("roofline"), "kernel_classes": r["kernel_classes"], "note": r["note"]}))
        if world > 1:
            dist.destroy_process_group()
        return 0

    field_cache = {}
    head = measure(args.workload, args, local, world, rank, field_cache, headline=True)
    subs = []
    if args.workload == "c2" and args.sub != "none":
        for name in [s for s in args.sub.split(",") if s]:
            try:
                if name in SMALL:
                    if rank == 0:
                        subs.append(measure_small(name, args, local))
                    continue
                r = measure(name, args, local, world, rank, field_cache, headline=False)
                subs.append({k: r[k] for k in ("workload", "dtype", "value", "unit", "steps", "ms_per_step", "config", "e2e",
                                               "gpu_launches", "bad_cells", "roofline", "step_roofline", "kernel_classes")})
            except Exception as e:                       # a sub-record must never cost the headline
                subs.append({"workload": name, "error": str(e).splitlines()[0][:200]})
    field_cache.clear()

    # ---- the oracle beside it (rank 0, N=1 only): one thread, and all host cores --------
    cpu = cpu_all = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = run_oracle_sample(args.cpu_steps, 1)
        cpu_all = run_oracle_sample(args.cpu_steps, 1, all_cores=True)

    if rank == 0:
        line = {"metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": head["steps"],
                "warmup": head["warmup"], "ms_per_step": head["ms_per_step"], "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": head["dtype"], "data": "synthetic",
                "config": head["config"], "clocks": head["clocks"], "e2e": head["e2e"], "gpu_launches": head["gpu_launches"],
                "bad_cells": head["bad_cells"], "conservation": head["conservation"], "roofline": head["roofline"],
                "step_roofline": head["step_roofline"], "kernel_classes": head["kernel_classes"],
                "cpu_baseline": cpu, "cpu_baseline_all_cores": cpu_all, "sub_records": subs}
        # Compact digest LAST on the line (a record that keeps only the tail of the output still holds it): the
        # metric is "(fp32/fp64)", so the fp64 half and the other configurations, one short entry each, no blobs.
        def brief(r):
            rf = r.get("roofline") or {}
            e = r.get("e2e") or {}
            return {"dtype": r.get("dtype"), "value": r.get("value"), "ms_per_step": r.get("ms_per_step"),
                    "kernel": rf.get("kernel"), "bound": rf.get("bound"), "frac": rf.get("frac"), "e2e_value": e.get("value")}
        digest = {"c2": brief({**head, "dtype": head["dtype"]})}
        for r in subs:
            digest[r.get("workload", "?")] = brief(r) if "error" not in r else {"error": r["error"]}
        line["value_f64"] = (digest.get("c2f64") or {}).get("value")
        line["roofline_f64"] = {k: (digest.get("c2f64") or {}).get(k) for k in ("kernel", "bound", "frac")}
        line["digest"] = digest
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
