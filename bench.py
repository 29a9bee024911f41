#!/usr/bin/env python
"""bench.py -- throughput of the bunch MHD update on B200 (cell-updates/s).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c2|c3|c3f64|small]
    python bench.py --impl reference ...      # the CPU oracle on a bounded sample

A step = one pass of the whole hot path over the bunch: fill_guards -> cfl_dt (dt stays
on the device) -> step.  The default workload is BASELINE.json config 2 (512 patches of
32^3, fp32, seeded turbulence-like field).  Prints ONE JSON line (see DESIGN.md,
"Measurement").  Multi-GPU: the path does not shard (north_star: one GPU) -- under
torchrun every rank runs an independent replica ("replicas only").
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
# the CPU oracle's bounded sample: the same seeded field construction on 64^3 cells
SAMPLE_N = 64


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


def algorithmic_work(cls, n, ng=3):
    r = lambda a, b: ((n + a + b) / n) ** 3
    f1 = (n + 1) / n
    riemann_flops = 3 * f1 * (28 + 392) + 3 * f1 * f1 * (104 + 453) + 81     # face + edge states, solves, update
    table = {
        # class: (values per cell, flops per cell, bound)
        "fill_guards": (2 * 8 * (r(ng, ng) - 1.0), 0.0, "hbm"),
        "cfl": (8 + 3 / n, CFL_FLOPS, "hbm"),
        "predict": (8 * r(2, 3) + 38 * r(1, 1), STEP_FLOPS_32 - riemann_flops, "hbm"),
        "riemann_update": (38 * r(1, 1) + 8 + 8, riemann_flops, "alu"),
        "step_onepass": (8 * r(2, 3) + 8, STEP_FLOPS_32, "alu"),
        # staged path (general, collapsed dimensions)
        "prim": (8 * r(2, 3) + 8 * r(2, 2), 40.0, "hbm"),
        "emf0": ((3 + 3) * r(2, 2) + 3 * r(1, 2), 70.0, "hbm"),
        "hlld_flux": (3 * ((5 + 7) * r(1, 1) + 3 * r(1, 2) + 5 * r(0, 1)), 3 * f1 * 420, "alu"),
        "emf_2d": (3 * ((5 + 12 + 2) * r(1, 1) + 3 * r(1, 2) + 1 * r(0, 1)), 3 * f1 * f1 * 557, "alu"),
        "update": (8 + 15 * r(0, 1) + 3 * r(0, 1) + 8, 81.0, "hbm"),
    }
    return table.get(cls)


def ncu_traffic(workload, cls):
    """DRAM bytes per launch of a kernel class from the committed ncu capture, or None."""
    path = os.path.join(ROOT, "profiles", "r1_ncu_traffic.txt")
    try:
        return json.load(open(path)).get(workload, {}).get(cls)
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


def run_oracle_sample(steps, warmup):
    """The oracle as it stands on the bounded sample; returns (cell-updates/s, seconds, description)."""
    import oracle
    w = W.turbulence(N=SAMPLE_N, n=32, dtype=np.float32, config=2)
    o = oracle.Oracle(w.n, w.npatch, w.gamma, w.dx)
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
    desc = (f"config-2 field construction on {SAMPLE_N}^3 cells = {w.npatch} patches x 32^3, fp64 oracle, "
            f"fill+cfl+step, {steps} steps, single thread")
    return w.cells * steps / el, el, desc


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c2", choices=sorted(WORKLOADS))
    ap.add_argument("--cpu-steps", type=int, default=20, help="oracle steps for the cpu_baseline leg")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--host-chunk", type=int, default=0, help="patches per chunk of the host-streaming path (0: library default)")
    ap.add_argument("--path", default="auto", choices=["auto", "staged", "two_kernel", "onepass"],
                    help="which CUDA implementation of the step runs (include/mhd_bunch.h, MHD_PATH_*)")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    N, n, dtype, wdesc = WORKLOADS[args.workload]

    # ---------------------------------------------------------------- reference arm ----
    if args.impl == "reference":
        if rank != 0:
            return 0
        steps = max(1, args.steps)
        val, el, desc = run_oracle_sample(steps, max(0, min(args.warmup, 2)))
        line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
                "warmup": args.warmup, "ms_per_step": 1e3 * el / steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": wdesc, "sample": desc},
                "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc},
                "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                "gpu_launches": 0}
        print(json.dumps(line))
        return 0

    # --------------------------------------------------------------------- our arm ----
    import torch
    import torch.distributed as dist
    from paper_2508_09568_b200.binding import MhdBunch

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    w = W.turbulence(N=N, n=n, dtype=np.float32 if dtype == "f32" else np.float64, config=2)
    b = MhdBunch(w.n, w.npatch, w.nbr, w.gamma, w.dx, dtype=dtype, device=local)
    b.load(w.U)
    b.set_path(args.path)
    stream = b.stream
    courant = 0.4

    def one_step():
        b.fill_guards()
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

    for _ in range(max(3, args.warmup)):
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
        for _ in range(args.steps):
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
    value, ms = aggregate_over_ranks(ms, w.cells, args.steps, world, device="cuda")

    # ---- per-kernel-class device times (separate pass, events around every launch) ----
    b.set_timing(True)
    tsteps = min(args.steps, 10)
    for _ in range(tsteps):
        one_step()
    kt = b.kernel_times()
    b.set_timing(False)
    pk = peaks()
    esz = 4 if dtype == "f32" else 8
    from paper_2508_09568_b200.binding import measure_alu_peak
    alu_peak = measure_alu_peak(dtype, local)               # TFLOP/s, FMA-chain, measured now
    alu_nominal = 148 * (128 if dtype == "f32" else 64) * 2 * pk["sm_max_mhz"] * 1e6 / 1e12
    classes = {k: {"ms_per_step": v[0] / tsteps, "launches_per_step": v[1] / tsteps} for k, v in kt.items()}
    tot = sum(c["ms_per_step"] for c in classes.values())
    for k, c in classes.items():
        c["share"] = c["ms_per_step"] / tot
        a = algorithmic_work(k, n)
        if a:
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
    roofline.update({"traffic": ncu_traffic(args.workload, dom), "avg_launch_ms": per_launch_ms,
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
        esteps = max(2, min(args.steps, 10))
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
               "chunk_patches": int(hl.chunk_patches), "chunks": int(hl.nchunk), "overlapped": bool(hl.pipelined),
               "note": "mhd_bunch_step_host: compact host state (interiors only) uploaded from pinned memory, "
                       "stepped and downloaded every step in chunks on two copy streams; wall clock"}

    # ---- the oracle beside it (rank 0, N=1 only) ---------------------------------------
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        val, el, desc = run_oracle_sample(args.cpu_steps, 1)
        cpu = {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc, "seconds": el}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(3, args.warmup), "ms_per_step": ms / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": dtype, "data": "synthetic",
                "config": {"workload": wdesc, "patches": w.npatch, "patch": [n, n, n], "guard": 3, "courant": courant,
                           "chunk_patches": b.chunk, "step_path": b.path, "parallelism": "replicas only" if world > 1 else "single GPU",
                           "l2": "state buffers (2 x %.0f MB) exceed the 126 MB L2; no flush needed" % (b.lay.state_bytes / 1e6)},
                "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "bad_cells": bad, "conservation": conservation,
                "roofline": roofline, "step_roofline": step_view, "kernel_classes": classes, "cpu_baseline": cpu}
        print(json.dumps(line))
    b.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
