"""Compile the CPU oracle (TEST INFRASTRUCTURE) into oracle/liboracle_f64.so and _f32.so.

Plain gcc, -O2, no fast-math, no FMA contraction: the arithmetic is what the C says.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "mhd_oracle.c")
HDR = os.path.join(HERE, "mhd_oracle.h")
LIBS = {
    "f64": (os.path.join(HERE, "liboracle_f64.so"), []),
    "f32": (os.path.join(HERE, "liboracle_f32.so"), ["-DORACLE_REAL=float", "-DORACLE_IS_FLOAT=1"]),
}


def _stale(target):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(s) > t for s in (SRC, HDR))


CFLAGS = ["-O2", "-std=c99", "-fPIC", "-shared", "-ffp-contract=off", "-fno-fast-math",
          "-Wall", "-Wextra", "-Wno-unused-parameter", "-Wno-unknown-pragmas"]


def compile_to(src, outdir, keys=("f64", "f32"), extra=()):
    """Compile an oracle source file (the committed one, or a copy a test has edited) into
    outdir/liboracle_<key>.so; returns {key: path}."""
    out = {}
    for key in keys:
        target = os.path.join(outdir, os.path.basename(LIBS[key][0]))
        cmd = ["gcc", *CFLAGS, *extra, "-I", HERE, *LIBS[key][1], src, "-o", target + ".tmp", "-lm"]
        subprocess.run(cmd, check=True, cwd=HERE)
        os.replace(target + ".tmp", target)
        out[key] = target
    return out


def build(force=False):
    for key, (target, defs) in LIBS.items():
        if not force and not _stale(target):
            continue
        compile_to(SRC, HERE, keys=(key,))
    return {k: v[0] for k, v in LIBS.items()}


OMP_LIB = os.path.join(HERE, "liboracle_f64_omp.so")


def build_omp(force=False):
    """The same source with -fopenmp: the `#pragma omp parallel for` over patches in orc_step /
    orc_cfl_dt / orc_fill_guards becomes active (patches are independent between guard fills, no
    change of arithmetic).  Used by bench.py's all-cores cpu_baseline leg only."""
    if force or _stale(OMP_LIB):
        target = OMP_LIB
        cmd = ["gcc", *CFLAGS, "-fopenmp", SRC, "-o", target + ".tmp", "-lm"]
        subprocess.run(cmd, check=True, cwd=HERE)
        os.replace(target + ".tmp", target)
    return OMP_LIB


if __name__ == "__main__":
    print(build(force=True))
    print(build_omp(force=True))
