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


# algorithmic HBM bytes per interior cell-update of each kernel class, in units of
# sizeof(real): compulsory reads + writes of that pass with perfect on-chip reuse
# (DESIGN.md "Kernels").  m = padded/interior volume ratio of the pass's input halo.
def algorithmic_values_per_cell(cls, n, ng=3):
    r = lambda a, b: ((n + a + b) / n) ** 3
    table = {
        "fill_guards": 2 * 8 * (r(ng, ng) - 1.0),                 # read + write the guard shell, 8 fields
        "cfl": 8 + 3 / n,                                         # 8 fields (+ closing faces), one scalar out
        "prim": 8 * r(2, 3) + 8 * r(2, 2),
        "emf0": (3 + 3) * r(2, 2) + 3 * r(1, 2),
        "predict": (8 + 3) * r(2, 2) + 3 * r(1, 2) + (21 + 6 + 5) * r(1, 1) + 3 * r(1, 2),
        "hlld_flux": 3 * ((5 + 7) * r(1, 1) + 3 * r(1, 2) + 5 * r(0, 1)),      # three directions
        "emf_2d": 3 * ((5 + 12 + 2) * r(1, 1) + 3 * r(1, 2) + 1 * r(0, 1)),    # three edge directions
        "update": 8 + 15 * r(0, 1) + 3 * r(0, 1) + 8,
        "fused_step": 8 * r(2, 3) + 8,
    }
    return table.get(cls)


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

    for _ in range(max(3, args.warmup)):
        one_step()
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
    if world > 1:
        t = torch.tensor([ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    value = world * w.cells * args.steps / (ms * 1e-3)

    # ---- per-kernel-class device times (separate pass, events around every launch) ----
    b.set_timing(True)
    tsteps = min(args.steps, 10)
    for _ in range(tsteps):
        one_step()
    kt = b.kernel_times()
    b.set_timing(False)
    pk = peaks()
    esz = 4 if dtype == "f32" else 8
    classes = {k: {"ms_per_step": v[0] / tsteps, "launches_per_step": v[1] / tsteps} for k, v in kt.items()}
    tot = sum(c["ms_per_step"] for c in classes.values())
    for k, c in classes.items():
        c["share"] = c["ms_per_step"] / tot
        a = algorithmic_values_per_cell(k, n)
        if a:
            c["alg_bytes_per_cell"] = a * esz
            c["alg_gbs"] = a * esz * w.cells / (c["ms_per_step"] * 1e-3) / 1e9
    dom = max((k for k in classes if k != "misc"), key=lambda k: classes[k]["ms_per_step"])
    dc = classes[dom]
    per_launch_ms = dc["ms_per_step"] / dc["launches_per_step"]
    roofline = {"kernel": dom, "bound": "hbm", "achieved": dc.get("alg_gbs"), "peak": pk["hbm_gbs"], "unit": "GB/s",
                "frac": (dc.get("alg_gbs") or 0.0) / pk["hbm_gbs"], "traffic": None, "peak_source": pk["source"],
                "avg_launch_ms": per_launch_ms, "share_of_step": dc["share"],
                "alg_bytes_per_launch": dc.get("alg_bytes_per_cell", 0) * w.cells / dc["launches_per_step"]}
    # whole-step view: compulsory traffic of a fully fused step (16 values per cell)
    step_view = {"compulsory_bytes_per_cell": 16 * esz,
                 "hbm_frac_at_compulsory_bytes": 16 * esz * value / world / 1e9 / pk["hbm_gbs"]}

    # ---- end to end through the host-buffer path of the C ABI -------------------------
    e2e = None
    if not args.no_e2e:
        nbytes = int(b.lay.state_bytes)
        host_in = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
        host_out = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
        b.download_host(host_in)
        esteps = max(2, min(args.steps, 5))
        def e2e_step():
            b.upload_host(host_in)
            one_step()
            b.download_host(host_out)       # synchronises
        e2e_step()
        barrier()
        t0 = time.perf_counter()
        for _ in range(esteps):
            e2e_step()
        torch.cuda.synchronize()
        el = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([el], device="cuda", dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            el = float(t.item())
        e2e = {"value": world * w.cells * esteps / el, "unit": UNIT, "h2d_bytes_per_step": nbytes,
               "d2h_bytes_per_step": nbytes, "steps": esteps,
               "note": "whole bunch uploaded from pinned host memory and downloaded every step (the paper's offload mode)"}

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
                           "chunk_patches": b.chunk, "parallelism": "replicas only" if world > 1 else "single GPU",
                           "l2": "state buffers (2 x %.0f MB) exceed the 126 MB L2; no flush needed" % (b.lay.state_bytes / 1e6)},
                "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "bad_cells": bad,
                "roofline": roofline, "step_roofline": step_view, "kernel_classes": classes, "cpu_baseline": cpu}
        print(json.dumps(line))
    b.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
