"""Full-size parity (c5, 512^3, the launch configuration bench.py times: CUDA-graph steps).

The oracle cannot run 512^3 in test time, so (task statement, parity at full size):
  * sampled outputs the oracle can compute one by one -- H^n (S1) and the divergence of the projected field (S8)
    are local stencils, so a 22^3 sub-box cut out of the 512^3 GPU fields and handed to the oracle as a small
    periodic box reproduces them exactly on the sub-box interior (also across the periodic seam);
  * properties that hold at any size -- convergence of the Poisson solve to the stated tolerance (true
    residual recomputed by the projection kernel), iteration counts in the range the oracle shows on the
    128^3 replica (the V-cycle makes them h-independent, pin P14), divergence-free projected field, zero-mean p.
"""
import math
import os

import numpy as np
import pytest

import fs_workloads as W
from oracle import Oracle

pytestmark = pytest.mark.gpu
N = 512
M = 20           # interior of a sampled sub-box


@pytest.fixture(scope="module")
def fs():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2505_23940_b200 as m
    m.lib()
    return m


def _sub(a, k0, j0, i0, m):
    """(m+2)^3 block of a periodic field starting one cell before (k0, j0, i0)."""
    idx = lambda s: np.arange(s - 1, s + m + 1) % N
    return np.ascontiguousarray(a[np.ix_(idx(k0), idx(j0), idx(i0))])


def _small_cfg(cfg, m):
    h = cfg["lx"] / cfg["nx"]
    c = dict(cfg)
    c.update(nx=m + 2, ny=m + 2, nz=m + 2, lx=(m + 2) * h, ly=(m + 2) * h, lz=(m + 2) * h, precond="jacobi", init=None)
    return c


CORNERS = [(100, 200, 300), (N - 7, N - 3, N - 11), (0, 250, N - 1)]      # the last two straddle the periodic seam


def test_c5_512_fp64_sampled_momentum_projection_and_solver_properties(fs):
    cfg = W.hit(n=N, device="cuda:0")
    g = fs.from_workload(cfg, device="cuda:0")
    cfg["init"] = None
    # ---- S1 at full size, sampled: H^n on three sub-boxes against the oracle
    uvw = [g.get(c) for c in "uvw"]
    H = g.momentum_rhs()
    for (k0, j0, i0) in CORNERS:
        o = Oracle(_small_cfg(cfg, M))
        for c, a in zip("uvw", uvw):
            o.set(c, _sub(a, k0, j0, i0, M))
        ref = o.momentum_rhs()
        for c, a, r in zip("uvw", H, ref):
            got = _sub(a, k0, j0, i0, M)[1:-1, 1:-1, 1:-1]
            want = r[1:-1, 1:-1, 1:-1]
            err = np.abs(got - want).max() / np.abs(want).max()
            assert err < 1e-12, ("H" + c, (k0, j0, i0), err)
    del H
    # ---- three graph-replayed steps (what bench.py times)
    info = g.step(3, per_step=True)
    assert info["nan_flag"] == 0 and info["converged"] == 1, info
    assert all(5 <= n <= 16 for n in info["iters_per_step"]), info          # oracle at 128^3: 13, 9, 9, ...
    assert info["rel_residual"] <= 1e-8
    assert info["true_rel_residual"] <= 2e-8                                # recurrence vs true residual in fp64
    assert info["max_abs_div"] < 1e-7, info
    # ---- S8 at full size, sampled: divergence of the projected field, by the oracle's operator
    uvw = [g.get(c) for c in "uvw"]
    umax = max(np.abs(a).max() for a in uvw)
    h = cfg["lx"] / N
    for (k0, j0, i0) in CORNERS:
        o = Oracle(_small_cfg(cfg, M))
        d = o.divergence(*[_sub(a, k0, j0, i0, M) for a in uvw])[1:-1, 1:-1, 1:-1]
        assert np.abs(d).max() <= info["max_abs_div"] * 1.01 + 1e-30               # the kernel's reported maximum bounds it
        assert np.abs(d).max() < 1e-9 * umax / h
    p = g.get("p")
    assert abs(p.mean()) < 1e-10 * np.abs(p).max()
    g.close()


def test_c5_512_fp32_fields_within_1e4_of_fp64_after_5_steps(fs):
    # north_star: fp32 fields within 1e-4 over 5 steps.  At 512^3 the fp64 reference is the fp64 CUDA path, itself
    # compared with the oracle at this size (tests/test_gpu_zz_fullsize_oracle.py and the golden pins below).
    cfg = W.hit(n=N, device="cuda:0")
    g64 = fs.from_workload(cfg, device="cuda:0")
    g32 = fs.from_workload(cfg, device="cuda:0", dtype="f32")
    cfg["init"] = None
    i64 = g64.step(5, per_step=True)
    i32 = g32.step(5, per_step=True)
    assert i32["nan_flag"] == 0 and i32["converged"] == 1 and i32["unconverged_steps"] == 0, i32
    assert all(abs(a - b) <= 1 for a, b in zip(i32["iters_per_step"], i64["iters_per_step"])), (i32["iters_per_step"], i64["iters_per_step"])
    assert i32["rel_residual"] <= 1e-8                                     # recurrence residual (reading A14)
    assert i32["true_rel_residual"] < 2e-3, i32                            # reported, not the criterion: in fp32 the true residual stalls
                                                                           # near eps32 x cond(A) ~ 3e-4 at 512^3 (reading A14)
    used = g32.kernels_used()
    for k in ("k_mg_down<f32,TR16,UPD>", "k_mg_up<f32,TR16,DOT>", "k_pcg_dirapplyv<f32>", "k_projectv<f32>"):
        assert k in used, (k, used)
    errs = {}
    for c in "uvwp":
        ref = g64.get(c)
        errs[c] = float(np.abs(g32.get(c) - ref).max() / np.abs(ref).max())
    assert all(e < 1e-4 for e in errs.values()), errs
    g64.close(); g32.close()


# ---- full size AND full step count, on sampled points: golden values written by tests/golden/make_fullsize_pins.py
#      (a committed script that calls only oracle/; hours of single-threaded oracle time, done once)
def _pins(case):
    path = os.path.join(os.path.dirname(__file__), "golden", "fullsize_%s.txt" % case)
    P = {"ic": {c: [] for c in "uvw"}, "val": {c: [] for c in "uvwp"}, "max": {}}
    for line in open(path):
        f = line.split()
        if not f or f[0].startswith("#"):
            continue
        if f[0] == "steps":
            P["steps"] = int(f[1])
        elif f[0] == "iters":
            P["iters"] = [int(x) for x in f[1:]]
        elif f[0] in ("body_force", "body_disp", "body_vel"):
            P[f[0]] = [float.fromhex(x) for x in f[1:]]
        elif f[0] == "max_abs_div":
            P["max_abs_div"] = float.fromhex(f[1])
        elif f[0] == "max":
            P["max"][f[1]] = float.fromhex(f[2])
        else:
            P[f[0]][f[1]].append((int(f[2]), float.fromhex(f[3])))
    return P


def _pin_case(case):
    # a pin file costs hours of single-threaded oracle time (c4: ~2.5 h); a config whose file has not been written yet
    # is reported as skipped, never silently passed
    have = os.path.exists(os.path.join(os.path.dirname(__file__), "golden", "fullsize_%s.txt" % case))
    return pytest.param(case, marks=pytest.mark.skipif(not have, reason="tests/golden/fullsize_%s.txt not written yet "
                                                       "(python tests/golden/make_fullsize_pins.py %s)" % (case, case)))


@pytest.mark.parametrize("case", [_pin_case(c) for c in ("c2", "c3", "c4", "c5")])
def test_full_size_full_step_count_against_oracle_pins(fs, case):
    import importlib.util
    spec = importlib.util.spec_from_file_location("make_fullsize_pins", os.path.join(os.path.dirname(__file__), "golden", "make_fullsize_pins.py"))
    mk = importlib.util.module_from_spec(spec); spec.loader.exec_module(mk)
    P = _pins(case)
    cfg = W.make(case, device="cuda:0") if case == "c5" else W.make(case)
    assert P["steps"] == cfg["steps"]
    g = fs.from_workload(cfg, device="cuda:0")
    sh = g.shape
    # the stored samples are at the indices the script draws from the config; the initial field must be the one the
    # oracle started from (c5: built by FFT on the device here, on the CPU there: equal to rounding)
    for c in "uvw":
        idx = mk.sample_indices(cfg, c, sh[c])
        assert [q for q, _ in P["ic"][c]] == idx.tolist()
        got = g.get(c).reshape(-1)[idx]
        want = np.array([v for _, v in P["ic"][c]])
        assert np.abs(got - want).max() < 1e-12 * max(1.0, np.abs(want).max()), (case, c)
    ig = g.step(P["steps"], per_step=True)
    assert ig["nan_flag"] == 0 and ig["converged"] == 1 and ig["unconverged_steps"] == 0, ig
    assert all(abs(a - b) <= 1 for a, b in zip(ig["iters_per_step"], P["iters"])), (ig["iters_per_step"], P["iters"])
    errs = {}
    for c in "uvwp":
        a = g.get(c)
        idx = np.array([q for q, _ in P["val"][c]])
        want = np.array([v for _, v in P["val"][c]])
        errs[c] = float(np.abs(a.reshape(-1)[idx] - want).max() / P["max"][c])
        assert abs(np.abs(a).max() - P["max"][c]) < 1e-9 * P["max"][c], (case, c)
    assert all(e < 1e-9 for e in errs.values()), (case, errs)
    for k in ("body_force", "body_disp", "body_vel"):
        np.testing.assert_allclose(ig[k], P[k], rtol=1e-9, atol=1e-12)
    g.close()


# ---- a property that holds at any size: the path is deterministic.  Every reduction is added in a fixed order (ticketed
#      partials), the IBM spread walks sorted cell lists, so two runs from the same state agree BIT FOR BIT; a
#      race in a shared-memory ring, a prefetch that lands late or a barrier that lets a CTA through early shows up as a
#      differing word.  Run in the launch configurations bench.py times (c5 at 512^3 in both precisions, CUDA-graph steps;
#      the cooperative whole-solve kernel on c3 / c4 at their stated sizes).
@pytest.mark.parametrize("case,dtype,steps", [("c5", "f64", 2), ("c5", "f32", 2), ("c3", "f64", 3), ("c4", "f64", 3), ("c2", "f64", 2)])
def test_two_runs_from_the_same_state_agree_bit_for_bit(fs, case, dtype, steps):
    runs = []
    for rep in range(2):
        cfg = W.make(case, device="cuda:0") if case == "c5" else W.make(case)
        g = fs.from_workload(cfg, device="cuda:0", dtype=dtype)
        info = g.step(steps, per_step=True)
        assert info["nan_flag"] == 0 and info["converged"] == 1, info
        runs.append((info, {c: g.get(c) for c in "uvwp"}))
        g.close()
    (ia, fa), (ib, fb) = runs
    assert ia["iters_per_step"] == ib["iters_per_step"], (ia["iters_per_step"], ib["iters_per_step"])
    for k in ("rel_residual", "max_abs_div", "body_force", "body_disp", "body_vel"):
        assert np.array_equal(np.asarray(ia[k]), np.asarray(ib[k])), (case, k, ia[k], ib[k])
    for c in "uvwp":
        assert np.array_equal(fa[c], fb[c]), (case, dtype, c, float(np.abs(fa[c] - fb[c]).max()))
