"""Host-side checks of the C-ABI boundary that need no GPU: the library loads, exports every symbol
include/streams.h declares, the ctypes structs have the C layout, and argument validation works."""
import ctypes as C
import os
import re
import subprocess
import tempfile

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "streams.h")


@pytest.fixture(scope="module")
def blib():
    from paper_2004_02276_b200 import build
    build.build()
    from paper_2004_02276_b200 import binding
    return binding


def test_exports_every_declared_symbol(blib):
    src = open(HEADER).read()
    declared = set(re.findall(r"\b(streams_[a-z0-9_]+)\s*\(", src))
    assert declared, "no prototypes found"
    L = blib.lib()
    for name in sorted(declared):
        assert hasattr(L, name), f"{name} declared in streams.h but not exported"
    assert declared == set(blib.EXPORTS)


def test_struct_layout_matches_c(blib):
    prog = r'''
#include <stdio.h>
#include <stddef.h>
#include "streams.h"
int main(void){
  printf("%zu %zu %zu\n", sizeof(streams_grid), sizeof(streams_params), sizeof(streams_diag));
  printf("%zu %zu %zu %zu\n", offsetof(streams_params, visc_model), offsetof(streams_params, bc), offsetof(streams_params, fs), offsetof(streams_params, dt_fixed));
  printf("%zu\n", offsetof(streams_params, weno_order));
  printf("%zu %zu %zu\n", offsetof(streams_diag, weno_ifaces), offsetof(streams_diag, nonfinite), offsetof(streams_diag, max_speed));
  return 0; }'''
    with tempfile.TemporaryDirectory() as td:
        cfile = os.path.join(td, "t.c")
        open(cfile, "w").write(prog)
        exe = os.path.join(td, "t")
        subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), cfile, "-o", exe], check=True)
        out = subprocess.run([exe], capture_output=True, text=True, check=True).stdout.split()
    vals = [int(x) for x in out]
    P, D = blib.StreamsParams, blib.StreamsDiag
    assert vals[:3] == [C.sizeof(blib.StreamsGrid), C.sizeof(P), C.sizeof(D)]
    assert vals[3:7] == [P.visc_model.offset, P.bc.offset, P.fs.offset, P.dt_fixed.offset]
    assert vals[7] == P.weno_order.offset
    assert vals[8:11] == [D.weno_ifaces.offset, D.nonfinite.offset, D.max_speed.offset]


def test_workspace_and_validation(blib):
    import workloads as W
    wl = W.config3_channel(256, 128, 128)
    n = wl.npoints
    nb = blib.workspace_bytes(wl.grid, wl.params)
    assert (2 * 7 + 2 * 5) * 8 * n <= nb < (2 * 7 + 2 * 5) * 8 * n + (64 << 20)   # two primitive states (7 fields) + two RK registers (5) + small arrays
    wl5 = W.config5_channel_big()
    assert blib.workspace_bytes(wl5.grid, wl5.params) < 60e9          # fits 180 GB HBM with room for the input copy
    bad = dict(wl.params, order=5)
    assert blib.workspace_bytes(wl.grid, bad) == 0
    bad = dict(wl.params, bc=[0, 6, 1, 1, 0, 0])                       # periodic on one x face only
    assert blib.workspace_bytes(wl.grid, bad) == 0
    bad = dict(wl.params, weno_enable=1, sensor_eps=0.0)
    assert blib.workspace_bytes(wl.grid, bad) == 0
    assert blib.workspace_bytes(wl.grid, dict(wl.params, weno_order=7)) == 0
    assert blib.workspace_bytes(wl.grid, dict(wl.params, weno_order=3)) == blib.workspace_bytes(wl.grid, dict(wl.params, weno_order=0)) > 0
    # create without a workspace fails with ENOMEM before any CUDA call
    g, p = blib.make_grid(wl.grid), blib.make_params(wl.params)
    import numpy as np
    xs = [np.ascontiguousarray(a) for a in (wl.x, wl.y, wl.z)]
    h = C.c_void_p()
    dbl = C.POINTER(C.c_double)
    rc = blib.lib().streams_create(C.byref(g), xs[0].ctypes.data_as(dbl), xs[1].ctypes.data_as(dbl), xs[2].ctypes.data_as(dbl),
                                   C.byref(p), None, 0, None, C.byref(h))
    assert rc == blib.STREAMS_ENOMEM and b"workspace" in blib.lib().streams_last_error(None)
    assert blib.lib().streams_step(None, 1) == blib.STREAMS_EINVAL


def test_product_never_imports_oracle():
    """The product path must not route through the oracle (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2004_02276_b200")
    for dirpath, _d, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.lower(), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r'#include\s+[<"][^">]*\bstreams\.h[">]', txt), f
            assert not re.search(r"^\s*(from|import)\s+paper_2004_02276_b200\.(binding|build)", txt, re.M), f
            assert "libstreams_b200" not in txt and "CDLL(" not in txt.replace("C.CDLL(_build.build())", ""), f
