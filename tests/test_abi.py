"""The C-ABI library builds, loads and exports every symbol include/*.h declares; host-side argument
validation (no compute calls: there is no GPU on the CPU test box)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import fs_workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def fs():
    from paper_2505_23940_b200 import build
    build.build()
    import paper_2505_23940_b200 as fs
    return fs


def _declared():
    inc = os.path.join(ROOT, "include")
    src = "\n".join(open(os.path.join(inc, f)).read() for f in sorted(os.listdir(inc)) if f.endswith(".h"))
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(fs_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_all_exported(fs):
    names = _declared()
    assert len(names) >= 15
    L = fs.lib()
    for n in names:
        assert hasattr(L, n), n
    assert sorted(fs.SYMBOLS) == names


def test_library_has_no_torch_or_oracle_dependency(fs):
    import subprocess
    out = subprocess.run(["ldd", fs.LIB_PATH], capture_output=True, text=True).stdout
    assert "torch" not in out and "oracle" not in out and "c10" not in out


def test_struct_layout_matches_header(fs):
    # sizeof as the C compiler sees it == the ctypes mirror (catches field drift)
    import subprocess, tempfile
    code = '#include "fs.h"\n#include <stdio.h>\nint main(){printf("%zu %zu %zu\\n", sizeof(fs_params), sizeof(fs_step_info), sizeof(fs_poisson_info));return 0;}\n'
    with tempfile.TemporaryDirectory() as d:
        p = os.path.join(d, "s.c")
        open(p, "w").write(code)
        subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), p, "-o", os.path.join(d, "s")])
        a, b, c = map(int, subprocess.check_output([os.path.join(d, "s")]).split())
    assert (a, b, c) == (C.sizeof(fs.fs_params), C.sizeof(fs.fs_step_info), C.sizeof(fs.fs_poisson_info))


def test_workspace_bytes_and_validation_on_host(fs):
    L = fs.lib()
    n = C.c_size_t(0)
    cfg = W.taylor_green()
    P, _ = fs.make_params(cfg)
    assert L.fs_workspace_bytes(C.byref(P), C.byref(n)) == 0
    N = 32 ** 3
    assert 14 * N * 8 <= n.value <= 16 * N * 8 + (1 << 20)          # 9 velocity-shaped + 5 pressure-shaped fields
    P32, _ = fs.make_params(dict(cfg, dtype="f32"))
    n32 = C.c_size_t(0)
    assert L.fs_workspace_bytes(C.byref(P32), C.byref(n32)) == 0 and n32.value < n.value
    # invalid: tiny grid, mixed periodicity, non-monotone yf, GMG on a walled grid
    for bad in (dict(cfg, nx=1), dict(cfg, dt=0.0), dict(cfg, bc=["periodic", "noslip"] + ["periodic"] * 4)):
        Pb, _ = fs.make_params(bad)
        assert L.fs_workspace_bytes(C.byref(Pb), C.byref(n)) == 1
    ch = W.channel(n=16)
    yf = np.array(ch["yf"]); yf[3] = yf[2]
    Pb, keep = fs.make_params(dict(ch, yf=yf))
    assert L.fs_workspace_bytes(C.byref(Pb), C.byref(n)) == 1
    Pb, keep = fs.make_params(dict(ch, precond="gmg"))
    assert L.fs_workspace_bytes(C.byref(Pb), C.byref(n)) == 6
    assert L.fs_workspace_bytes(None, C.byref(n)) == 1
    # convection scheme out of range; a grid with more xy tiles than reduction partials; 32-bit field offsets
    Pb, _ = fs.make_params(cfg); Pb.convection = 2
    assert L.fs_workspace_bytes(C.byref(Pb), C.byref(n)) == 1
    Pb, _ = fs.make_params(dict(cfg, nx=4096, ny=1024, nz=2))
    assert L.fs_workspace_bytes(C.byref(Pb), C.byref(n)) == 6
    Pb, _ = fs.make_params(dict(cfg, nx=2048, ny=1024, nz=1024))
    assert L.fs_workspace_bytes(C.byref(Pb), C.byref(n)) == 6
    # GMG V(2,2) carries the second residual buffer of the fused update; other V(nu1,nu2) do not
    h = W.hit(n=32, device="cpu"); h["init"] = None
    n22, n11 = C.c_size_t(0), C.c_size_t(0)
    Pg, _ = fs.make_params(h)
    assert L.fs_workspace_bytes(C.byref(Pg), C.byref(n22)) == 0
    Pg, _ = fs.make_params(dict(h, mg_nu1=1, mg_nu2=1))
    assert L.fs_workspace_bytes(C.byref(Pg), C.byref(n11)) == 0
    assert 32 ** 3 * 8 <= n22.value - n11.value <= 32 ** 3 * 8 + 512
    assert L.fs_status_string(6) == b"unsupported configuration"
    # NULL handles never crash
    assert L.fs_grid_destroy(None) == 1 and L.fs_step(None, 1, None) == 1
    assert L.fs_kernels_used(None, None, 0, None) == 1


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2505_23940_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                s = open(os.path.join(dp, f)).read()
                assert "import oracle" not in s and "from oracle" not in s and "fs_oracle" not in s, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            s = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2505_23940_b200 import" not in s and "libfs.so" not in s and "fs_internal" not in s, f
