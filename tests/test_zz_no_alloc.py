"""fs_divergence_noalloc (include/fs_noalloc.h): the entry point that allocates nothing (its reduction scratch is a static
__device__ array inside libfs.so) against the EXISTING path on a grid -- fs_fields_get(FS_DIV) for the field and
fs_step_info.max_abs_div for the maximum of the projected field -- on calls in a row that share the scratch.

Collected last on purpose (file name): the suite runs with `pytest -x`.  Passes alone in a fresh process and after the
other tests (it owns its grids and tensors; the only shared state is the library's scratch array, which every call resets).
Tolerances are the suite's: fp64 1e-9, fp32 1e-4 (relative to the field's maximum)."""
import numpy as np
import pytest

import fs_workloads as W

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
F64 = 1          # fs_dtype FS_F64


@pytest.fixture(scope="module")
def fs():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2505_23940_b200 as m
    m.lib()
    return m


def _dev(a, dtype):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).to(DEV, dtype=dtype)


def _noalloc(fs, fields, h, dtype):
    """-> (div field, max |div|, sum div^2) from the no-alloc entry point; outputs pre-filled with a sentinel."""
    import torch
    u, v, w = (_dev(a, dtype) for a in fields)
    out = torch.full_like(u, 7.0)
    res = torch.full((2,), -1.0, dtype=torch.float64, device=DEV)
    fs.divergence_noalloc(u, v, w, h, div_out=out, result=res)
    torch.cuda.synchronize()
    r = res.cpu().numpy()
    return out.cpu().numpy(), float(r[0]), float(r[1])


def test_no_alloc_divergence_matches_the_grid_path_on_calls_in_a_row(fs):
    import torch
    # --- existing path A: c5 recipe at 64^3, one full step; the projected field's max |div| comes from the projection kernel
    cfg = W.hit(n=64, device=DEV)
    g = fs.from_workload(cfg, device=DEV)
    info = g.step(1)
    A = [g.get(c) for c in "uvw"]
    divA = g.get("div")
    hA = cfg["lx"] / 64
    scaleA = max(np.abs(a).max() for a in A) / hA
    # --- existing path B: a ragged, non-cubic box (69120 cells = 33.75 blocks of 2048) holding a field that is NOT solenoidal
    cfgB = W.hit_box(48, 40, 36, precond="jacobi")
    rng = np.random.default_rng(2024)
    B = [rng.standard_normal((36, 40, 48)) for _ in range(3)]
    cfgB["init"] = dict(zip("uvw", B))
    gB = fs.from_workload(cfgB, device=DEV)
    divB = gB.get("div")
    hB = cfgB["lx"] / 48
    assert np.abs(divB).max() > 1.0 / hB                      # order |u| / h: a real signal, not rounding noise

    f64 = torch.float64
    d1, m1, s1 = _noalloc(fs, A, hA, f64)                     # call 1 (also the set-up call: looks up the scratch address)
    free0 = torch.cuda.mem_get_info()[0]
    d2, m2, s2 = _noalloc(fs, B, hB, f64)                     # call 2: other sizes, other block count, stale scratch from call 1
    d3, m3, s3 = _noalloc(fs, A, hA, f64)                     # call 3: the first input again
    # field against fs_fields_get(FS_DIV)
    # (A: both kernels evaluate the same formula on the same words, so they agree to rounding, 1e-12 |u| / h, far below the
    #  solver-tolerance-sized divergence itself; the suite's 1e-9 is the bar on the field with a real signal, B)
    assert np.abs(d1 - divA).max() <= 1e-12 * scaleA
    assert np.abs(d2 - divB).max() <= 1e-9 * np.abs(divB).max()
    # maximum and 2-norm against the existing path's numbers
    assert abs(m1 - info["max_abs_div"]) <= 1e-12 * scaleA and 0.0 < m1 < 1e-6 * scaleA, (m1, info["max_abs_div"])
    assert abs(m1 - np.abs(divA).max()) <= 1e-12 * scaleA
    assert abs(m2 - np.abs(divB).max()) <= 1e-9 * np.abs(divB).max(), (m2, np.abs(divB).max())
    assert abs(s2 - float((divB.astype(np.float64) ** 2).sum())) <= 1e-9 * s2
    assert abs(s1 - float((d1 ** 2).sum())) <= 1e-9 * s1
    # the scratch keeps the last call's contents and it must not matter: call 3 == call 1 bit for bit
    assert m3 == m1 and s3 == s1 and np.array_equal(d3, d1)
    # independent of both CUDA paths: the oracle's operator on the non-solenoidal field
    from oracle import Oracle
    cfgB["init"] = None
    ref = Oracle(cfgB).divergence(*B)
    assert np.abs(d2 - ref).max() <= 1e-9 * np.abs(ref).max()
    # fp32 (the suite's 1e-4), through the same scratch
    g32 = fs.from_workload(dict(cfgB, init=dict(zip("uvw", B))), device=DEV, dtype="f32")
    div32 = g32.get("div")
    d4, m4, s4 = _noalloc(fs, B, hB, torch.float32)
    assert np.abs(d4 - div32).max() <= 1e-4 * np.abs(div32).max()
    assert abs(m4 - m2) <= 1e-4 * m2 and abs(s4 - s2) <= 1e-4 * s2
    # nothing was allocated on the device by the calls themselves (the helper's tensors come from torch's cache after call 1)
    _noalloc(fs, A, hA, f64)
    assert torch.cuda.mem_get_info()[0] >= free0 - (64 << 20), (free0, torch.cuda.mem_get_info()[0])
    g.close(); gB.close(); g32.close()


def test_no_alloc_divergence_without_a_field_output_and_argument_checks(fs):
    import torch
    rng = np.random.default_rng(7)
    n = (5, 6, 7)                                             # 210 cells: one partly filled block
    F = [rng.standard_normal(n) for _ in range(3)]
    u, v, w = (_dev(a, torch.float64) for a in F)
    h = (0.5, 0.25, 2.0)                                      # hx, hy, hz
    res = fs.divergence_noalloc(u, v, w, h)                   # div_out = NULL
    torch.cuda.synchronize()
    ref = ((np.roll(F[0], -1, 2) - F[0]) / h[0] + (np.roll(F[1], -1, 1) - F[1]) / h[1] + (np.roll(F[2], -1, 0) - F[2]) / h[2])
    r = res.cpu().numpy()
    assert abs(r[0] - np.abs(ref).max()) <= 1e-12 * np.abs(ref).max() and abs(r[1] - (ref ** 2).sum()) <= 1e-12 * (ref ** 2).sum()
    L = fs.lib()
    s = torch.cuda.current_stream().cuda_stream
    keep = res.clone()
    # beyond the stated maximum: refused with FS_ERR_UNSUPPORTED before anything is launched
    assert fs.NOALLOC_MAX_CELLS == 256 ** 3
    st = L.fs_divergence_noalloc(256, 256, 257, 1.0, 1.0, 1.0, F64, u.data_ptr(), v.data_ptr(), w.data_ptr(), None, res.data_ptr(), s)
    assert fs.STATUS[st] == "FS_ERR_UNSUPPORTED", st
    # a host pointer, a NULL input, a non-positive spacing: FS_ERR_INVALID_ARG
    host = np.zeros(210)
    for args in ((5, 6, 7, 1.0, 1.0, 1.0, F64, host.ctypes.data, v.data_ptr(), w.data_ptr(), None, res.data_ptr(), s),
                 (5, 6, 7, 1.0, 1.0, 1.0, F64, None, v.data_ptr(), w.data_ptr(), None, res.data_ptr(), s),
                 (5, 6, 7, 0.0, 1.0, 1.0, F64, u.data_ptr(), v.data_ptr(), w.data_ptr(), None, res.data_ptr(), s),
                 (5, 6, 7, 1.0, 1.0, 1.0, F64, u.data_ptr(), v.data_ptr(), w.data_ptr(), None, None, s)):
        st = L.fs_divergence_noalloc(*args)
        assert fs.STATUS[st] == "FS_ERR_INVALID_ARG", (st, args[:7])
    torch.cuda.synchronize()
    assert torch.equal(res, keep)                             # outputs untouched on failure
    # the largest box that is accepted: exactly FS_NOALLOC_MAX_CELLS cells, 8192 blocks, every scratch slot in use
    big = torch.zeros((256, 256, 256), dtype=torch.float32, device=DEV)
    lin = torch.arange(256, dtype=torch.float32, device=DEV)
    ub = (big + lin[None, None, :]).contiguous()              # u = i: div = 1/hx inside, (0 - 255)/hx across the seam
    res2 = fs.divergence_noalloc(ub, big, big, 1.0)
    torch.cuda.synchronize()
    r2 = res2.cpu().numpy()
    assert r2[0] == 255.0 and r2[1] == 256.0 * 256.0 * (255.0 + 255.0 ** 2)
