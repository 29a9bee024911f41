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


def build(force=False):
    for key, (target, defs) in LIBS.items():
        if not force and not _stale(target):
            continue
        cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-ffp-contract=off", "-fno-fast-math",
               "-Wall", "-Wextra", "-Wno-unused-parameter", *defs, SRC, "-o", target + ".tmp", "-lm"]
        subprocess.run(cmd, check=True, cwd=HERE)
        os.replace(target + ".tmp", target)
    return {k: v[0] for k, v in LIBS.items()}


if __name__ == "__main__":
    print(build(force=True))
