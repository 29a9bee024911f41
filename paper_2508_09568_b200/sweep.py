#!/usr/bin/env python
"""Bunching sweep of BASELINE.json config 4: patch sizes 16^3/24^3/32^3/64^3 x bunch sizes
1, 8, 64, 512, 4096 (plus the paper's own optimum, 24^3 x 300: PAPER.md L214), fp32, with the
config-2 field construction.  Per point: cell-updates/s of the resident loop
fill_guards -> cfl_dt -> step, the device-busy time per step (CUDA events around every
launch) and the launch-overhead share 1 - busy/wall (the overhead the
paper's bunching attacks).

    python -m paper_2508_09568_b200.sweep [--steps 20] [--dtype f32] [--out table.md]

Prints a markdown table.  Points whose state does not fit the device, or whose global field
(more than 512^3 cells) is too large to build on the host in reasonable time, are listed as
skipped.  Needs a CUDA device (no CPU fallback).
"""
import argparse
import sys
import time

import numpy as np

from . import workloads as W
from .binding import MhdBunch

# patches per side for each bunch size (periodic arrangements)
ARRANGE = {1: (1, 1, 1), 8: (2, 2, 2), 64: (4, 4, 4), 300: (5, 6, 10), 512: (8, 8, 8), 4096: (16, 16, 16)}


def point(n, npatch, dtype, steps, warmup=3):
    import torch
    P = ARRANGE[npatch]
    N = tuple(n * p for p in P)
    if max(N) > 512:
        return None, "global field of %dx%dx%d cells: not built on the host" % N
    npd = np.float32 if dtype == "f32" else np.float64
    w = W.turbulence(N=N, n=n, dtype=npd, config=2, patches=P)
    try:
        b = MhdBunch(w.n, w.npatch, w.nbr, w.gamma, w.dx, dtype=dtype)
    except Exception as e:      # out of memory on the device
        return None, str(e).splitlines()[0][:80]
    b.load(w.U)

    def one():
        b.fill_guards()
        b.cfl_dt(0.4, sync=False)
        b.step_dev()

    for _ in range(warmup):
        one()
    torch.cuda.synchronize()
    l0 = b.launches
    t0 = time.perf_counter()
    for _ in range(steps):
        one()
    torch.cuda.synchronize()
    wall = (time.perf_counter() - t0) / steps
    launches = (b.launches - l0) / steps
    b.set_timing(True)
    for _ in range(steps):
        one()
    kt = b.kernel_times()
    b.set_timing(False)
    busy = sum(v[0] for v in kt.values()) * 1e-3 / steps
    bad = b.status()
    res = {"n": n, "npatch": npatch, "cells": w.cells, "path": b.path, "wall_us": wall * 1e6, "busy_us": busy * 1e6,
           "launches": launches, "rate": w.cells / wall, "rate_busy": w.cells / busy,
           "overhead": max(0.0, 1.0 - busy / wall), "bad": bad}
    b.close()
    del b
    torch.cuda.empty_cache()
    return res, None


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--dtype", default="f32", choices=["f32", "f64"])
    ap.add_argument("--sizes", default="16,24,32,64")
    ap.add_argument("--bunches", default="1,8,64,512,4096")
    ap.add_argument("--out", default=None)
    args = ap.parse_args()
    sizes = [int(x) for x in args.sizes.split(",")]
    bunches = [int(x) for x in args.bunches.split(",")]
    pts = [(n, k) for n in sizes for k in bunches]
    if 24 in sizes:
        pts.append((24, 300))
    lines = ["| patch | bunch | cells/step | step path | launches/step | wall us/step | device-busy us/step | "
             "G cell-updates/s | launch-overhead share |", "|---|---:|---:|---|---:|---:|---:|---:|---:|"]
    for n, k in pts:
        r, why = point(n, k, args.dtype, args.steps)
        if r is None:
            lines.append(f"| {n}^3 | {k} | {k * n ** 3} | skipped: {why} | | | | | |")
        else:
            lines.append(f"| {n}^3 | {k} | {r['cells']} | {r['path']} | {r['launches']:.0f} | {r['wall_us']:.1f} | "
                         f"{r['busy_us']:.1f} | {r['rate'] / 1e9:.3f} | {r['overhead']:.2f} |")
        print(lines[-1], file=sys.stderr, flush=True)
    txt = "\n".join(lines)
    print(txt)
    if args.out:
        with open(args.out, "w") as fh:
            fh.write(txt + "\n")


if __name__ == "__main__":
    main()
