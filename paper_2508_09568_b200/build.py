"""Build libmhd_bunch.so (hand-written sm_100a kernels + C ABI) in-tree with nvcc."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
TARGET = os.path.join(HERE, "libmhd_bunch.so")
SOURCES = [os.path.join(CSRC, "mhd_bunch.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in ("mhd_math.cuh", "bunch_types.cuh", "stage_kernels.cuh", "fused_kernels.cuh", "onepass_kernel.cuh", "tile_kernel.cuh", "tma_utils.cuh", "host_stream_kernels.cuh")] + \
    [os.path.join(os.path.dirname(HERE), "include", "mhd_bunch.h")]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "--shared", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def stale():
    if not os.path.exists(TARGET):
        return True
    t = os.path.getmtime(TARGET)
    return any(os.path.getmtime(s) > t for s in DEPS)


def build(force=False, verbose=False):
    if not force and not stale():
        return TARGET
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    extra = os.environ.get("MHD_BUNCH_NVCC_FLAGS", "").split()      # build-time knobs (e.g. -DONEPASS_NPW=4)
    cmd = [nvcc, *NVCC_FLAGS, *extra, *SOURCES, "-o", TARGET + ".tmp"]
    r = subprocess.run(cmd, capture_output=True, text=True, cwd=HERE)
    log = r.stdout + r.stderr
    with open(os.path.join(HERE, "build.log"), "w") as fh:
        fh.write(" ".join(cmd) + "\n" + log)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + log[-4000:])
    os.replace(TARGET + ".tmp", TARGET)
    if verbose:
        print(log)
    return TARGET


if __name__ == "__main__":
    build(force=True, verbose=True)
