"""CPU-side checks of the C-ABI library: it builds for sm_100a, loads, exports every symbol
include/mhd_bunch.h declares, validates arguments on the host, and refuses to compute
without a GPU (no CPU fallback).  No kernel is launched here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2508_09568_b200 import binding as B
from paper_2508_09568_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    txt = open(os.path.join(ROOT, "include", "mhd_bunch.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(mhd_bunch_[a-z_0-9]+)\s*\(", txt)))


def test_library_exports_every_declared_symbol():
    lib = B.load_library()
    names = declared_symbols()
    assert len(names) >= 17
    for n in names:
        assert hasattr(lib, n), n
    assert set(names) == set(B.ABI_SYMBOLS)


def test_library_is_sm100a_only():
    import subprocess
    out = subprocess.run(["cuobjdump", "--list-elf", B._build.TARGET], capture_output=True, text=True).stdout
    assert "sm_100a" in out and "sm_90" not in out and "sm_80" not in out


@pytest.mark.parametrize("n,dtype,pitch", [((32, 32, 32), B.MHD_F32, 40), ((24, 24, 24), B.MHD_F32, 32),
                                           ((16, 16, 16), B.MHD_F64, 24), ((64, 64, 64), B.MHD_F32, 72),
                                           ((32, 32, 1), B.MHD_F64, 40), ((32, 1, 1), B.MHD_F64, 40)])
def test_query_layout(n, dtype, pitch):
    d = B.make_desc(n, 7, 5 / 3, (0.1, 0.1, 0.1), dtype)
    lay = B.query(d)
    m = W.padded(n)
    assert tuple(lay.m) == m
    assert lay.stride[4] == 1 and lay.stride[3] == pitch and lay.stride[2] == pitch * m[1]
    assert lay.stride[1] >= pitch * m[1] * m[2] and lay.stride[0] == 7 * lay.stride[1]
    esz = 4 if dtype == B.MHD_F32 else 8
    assert ((lay.origin + 3) * esz) % 16 == 0                 # interior cell 0 on a 16-byte boundary
    assert (pitch * esz) % 16 == 0
    assert lay.state_bytes == 8 * lay.stride[0] * esz
    assert lay.workspace_min <= lay.workspace_best


def test_query_rejects_bad_descriptions():
    lib = B.load_library()
    lay = B.Layout()
    def rc(**kw):
        args = dict(n=(8, 8, 8), npatch=2, gamma=1.4, dx=(1, 1, 1), dtype=B.MHD_F32)
        args.update(kw)
        d = B.make_desc(**args)
        return lib.mhd_bunch_query(C.byref(d), C.byref(lay))
    assert rc() == 0
    assert rc(ng=2) == -1                      # the scheme needs width 3
    assert rc(n=(2, 8, 8)) == -1               # active dimension thinner than the guard shell
    assert rc(n=(1, 1, 1)) == -1
    assert rc(npatch=0) == -1
    assert rc(gamma=1.0) == -1
    assert rc(dx=(1, 0, 1)) == -1
    assert rc(dtype=5) == -1
    assert rc(limiter=3) == -1
    assert rc(emf_solver=2) == -1
    assert rc(flux_solver=2) == -1 and rc(flux_solver=1) == 0
    assert lib.mhd_bunch_query(None, C.byref(lay)) == -1
    assert lib.mhd_bunch_strerror(-1) and lib.mhd_bunch_strerror(-3)


def test_create_validates_on_the_host_and_never_falls_back_to_cpu():
    import torch
    lib = B.load_library()
    d = B.make_desc((8, 8, 8), 2, 1.4, (1, 1, 1))
    lay = B.query(d)
    nbr = W.neighbour_table((2, 1, 1), (True, True, True))
    h = C.c_void_p()
    a = np.zeros(lay.state_bytes + 64, dtype=np.uint8)
    base = (a.ctypes.data + 15) // 16 * 16
    # host-side argument checks come first: aliasing, misalignment, bad neighbour ids, small workspace
    assert lib.mhd_bunch_create(C.byref(d), nbr.ctypes.data, base, base, base, lay.workspace_min, C.byref(h)) == -1
    assert lib.mhd_bunch_create(C.byref(d), nbr.ctypes.data, base + 4, base + 1 << 20, base, lay.workspace_min, C.byref(h)) == -1
    bad = nbr.copy(); bad[0, 0] = 2
    assert lib.mhd_bunch_create(C.byref(d), bad.ctypes.data, base, base + (1 << 30), base + (2 << 30),
                                lay.workspace_min, C.byref(h)) == -1
    assert lib.mhd_bunch_create(C.byref(d), nbr.ctypes.data, base, base + (1 << 30), base + (2 << 30), 16, C.byref(h)) == -2
    if not torch.cuda.is_available():
        # valid arguments but no device: MHD_ECUDA, and the Python class refuses too
        rc = lib.mhd_bunch_create(C.byref(d), nbr.ctypes.data, base, base + (1 << 30), base + (2 << 30),
                                  lay.workspace_min, C.byref(h))
        assert rc == -3 and b"no CUDA device" in lib.mhd_bunch_last_cuda_error()
        with pytest.raises(RuntimeError):
            B.MhdBunch((8, 8, 8), 2, nbr, 1.4, (1, 1, 1))
    # null handles are errors, not crashes
    assert lib.mhd_bunch_step(None, 0.1) == -4 and lib.mhd_bunch_fill_guards(None) == -4
    assert lib.mhd_bunch_destroy(None) == -4


def test_product_package_does_not_import_the_oracle():
    import subprocess, sys
    code = ("import sys; sys.path.insert(0, %r); import paper_2508_09568_b200.binding, paper_2508_09568_b200.workloads; "
            "assert not any(m == 'oracle' or m.startswith('oracle.') for m in sys.modules)") % ROOT
    subprocess.run([sys.executable, "-c", code], check=True)
    for root, _, files in os.walk(os.path.join(ROOT, "paper_2508_09568_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert "oracle" not in open(os.path.join(root, f)).read().replace("the CPU oracle", "").replace("CPU oracle's", ""), f


def test_no_named_barrier_inside_a_convergence_region():
    """The one-pass kernel's named barriers are the .aligned forms, which ptxas takes as a promise
    that the warp is whole; it once merged the convergence region of a divergent `if` with an outer
    one that ended after a bar.arrive, so that a warp arrived twice and the CTA hung (see
    onepass_kernel.cuh).  The source now keeps every barrier at the top level of its loop; this
    disassembles the built library and checks the result: no BAR.SYNC / BAR.ARV with a non-zero id
    (named barrier) may lie inside a BSSY ... BSYNC region that holds a lane-predicated forward
    branch before it."""
    import re
    import shutil
    import subprocess
    # a toolchain test: it needs the CUDA toolkit's disassembler and a built library; boxes without
    # either skip it instead of failing the CPU tier
    exe = shutil.which("cuobjdump") or ("/usr/local/cuda/bin/cuobjdump" if os.path.exists("/usr/local/cuda/bin/cuobjdump") else None)
    if exe is None:
        pytest.skip("cuobjdump is not installed")
    if not os.path.exists(B._build.TARGET):
        pytest.skip("libmhd_bunch.so is not built")
    txt = subprocess.run([exe, "-sass", B._build.TARGET], capture_output=True, text=True, check=True).stdout
    checked = 0
    for f in re.split(r"\n\s*Function : ", txt)[1:]:
        name = f.split("\n", 1)[0].strip()
        if "k_step_onepass" not in name:
            continue
        ins = [(int(m.group(1), 16), m.group(2).strip())
               for m in (re.match(r"\s*/\*([0-9a-f]{4,6})\*/\s+(.*?);", l) for l in f.splitlines()) if m]
        regions = [(a, int(m.group(1), 16)) for a, x in ins
                   for m in [re.match(r"(?:@!?U?P\d+\s+)?BSSY(?:\.\w+)*\s+B\d+,\s*0x([0-9a-f]+)", x)] if m]
        bars = [(a, x) for a, x in ins if re.search(r"\bBAR\.(SYNC|ARV)", x) and not re.search(r"BAR\.SYNC(\.\w+)*\s+0x0\s*$", x)]
        # a change of the disassembly format must fail here, not pass with nothing parsed
        assert len(ins) > 1000 and regions, (name, len(ins), len(regions))
        assert len(bars) >= 10, name
        for a, x in bars:
            for s, e in regions:
                if s < a < e:
                    inside = [(ba, bx) for ba, bx in ins if s < ba < a and re.match(r"@!?P\d+\s+BRA\b", bx)
                              and ba < int(re.search(r"0x([0-9a-f]+)", bx).group(1), 16) <= e]
                    assert not inside, (name, hex(a), x, [(hex(p), q) for p, q in inside[:3]])
        checked += 1
    assert checked >= 8
