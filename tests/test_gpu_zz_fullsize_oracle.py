"""One COMPLETE fractional step of every BASELINE.json config at its FULL size (c2 128^3 channel, c3 256x128x128
sphere with 3200 markers, c4 384x256x32 cylinder FSI with 2400 markers and the rigid body, c5 512^3 HIT with GMG-PCG),
CUDA path through the C ABI against the CPU oracle, element by element on all four fields: fp64 1e-9 (A9 norm), PCG
iterations +-1, cell lists bit-exact (north_star).  The oracle runs take 1-4 minutes each on one core; conftest.py
starts them as separate processes when the session begins, so they overlap the rest of the GPU suite (this file sorts
last on purpose).  The full STEP COUNTS of the configs are covered on sampled points by tests/test_gpu_fullsize.py
(golden values written by tests/golden/make_fullsize_pins.py)."""
import json
import os

import numpy as np
import pytest

import fs_workloads as W

pytestmark = pytest.mark.gpu
TOL64 = 1e-9


@pytest.fixture(scope="module")
def fs():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2505_23940_b200 as m
    m.lib()
    return m


def relerr(a, b):
    d = float(np.abs(a - b).max())
    s = float(np.abs(b).max())
    return d / s if s > 0 else d


# kernel instantiations each full-size case must have exercised (fs_kernels_used): c2 periodic x, stretched y: the
# vector kernels (momentum included); c3 / c4 bounded x: the generic one-cell projection / right-hand side.  The Jacobi-PCG solve runs as the
# persistent cooperative kernel by default on these L2-sized grids ("coop") and as the streaming pair inside the graph's
# WHILE node with FS_TUNE_COOP=0 ("stream", the path of larger grids): both against the same oracle step.
EXPECT = {
    "c2": ["k_momentumv<f64,central>", "k_div_rhsv<f64>", "k_pcg_initv<f64>", "k_projectv<f64>"],
    "c3": ["k_momentum<f64,central>", "k_div_rhs<f64>", "k_pcg_initv<f64>", "k_project<f64>", "ibm_interpolate", "ibm_spread", "flux_sum"],
    "c4": ["k_momentum<f64,central>", "k_div_rhs<f64>", "k_project<f64>", "ibm_index", "ibm_spread", "step_end"],
}
PCG = {"coop": ["k_pcg_coop<f64>"], "stream": ["k_pcg_dirapply2<f64>", "k_pcg_updatev<f64>"]}


@pytest.mark.parametrize("path", ["coop", "stream"])
@pytest.mark.parametrize("case", ["c2", "c3", "c4"])
def test_one_step_at_full_size_matches_oracle(fs, fullsize_oracle, case, path, monkeypatch):
    if path == "stream":
        monkeypatch.setenv("FS_TUNE_COOP", "0")
    cfg = W.make(case)
    g = fs.from_workload(cfg)
    ig = g.step(1, per_step=True)
    assert ig["nan_flag"] == 0 and ig["converged"] == 1, ig
    used = g.kernels_used()
    for k in EXPECT[case] + PCG[path]:
        assert k in used, (k, used)
    d = fullsize_oracle(case)
    io = json.load(open(os.path.join(d, case + "_info.json")))
    assert abs(ig["pcg_iters"] - io["pcg_iters"]) <= 1, (ig["pcg_iters"], io["pcg_iters"])
    errs = {c: relerr(g.get(c), np.load(os.path.join(d, "%s_%s.npy" % (case, c)))) for c in "uvwp"}
    assert all(e < TOL64 for e in errs.values()), errs
    if cfg.get("markers") is not None:
        a = g.cell_list()
        for k in ("base", "perm", "keys"):
            assert np.array_equal(a[k], np.load(os.path.join(d, "%s_cell_%s.npy" % (case, k)))), k
        assert np.array_equal(a["seg_start"], np.load(os.path.join(d, case + "_cell_seg.npy")))
        assert relerr(g.get("marker_f"), np.load(os.path.join(d, case + "_marker_f.npy"))) < TOL64
        assert relerr(g.get("marker_x"), np.load(os.path.join(d, case + "_marker_x.npy"))) < 1e-14
        np.testing.assert_allclose(ig["body_force"], io["body_force"], rtol=1e-9, atol=1e-12)
        np.testing.assert_allclose(ig["body_disp"], io["body_disp"], rtol=1e-9, atol=1e-15)
        np.testing.assert_allclose(ig["body_vel"], io["body_vel"], rtol=1e-9, atol=1e-15)
    g.close()


def test_one_step_of_c5_at_512_matches_oracle_on_every_cell(fs, fullsize_oracle):
    # the launch configuration bench.py times: 512^3 fp64, CUDA-graph step, k_mg_down / k_mg_up with 32-row tiles (TR16)
    d = fullsize_oracle("c5")
    cfg = W.hit(n=32)
    cfg.update(nx=512, ny=512, nz=512, init=None)
    g = fs.Grid(cfg)
    for c in "uvw":
        g.set(c, np.load(os.path.join(d, "c5_init_%s.npy" % c), mmap_mode="r"))
    ig = g.step(1, per_step=True)
    assert ig["nan_flag"] == 0 and ig["converged"] == 1, ig
    io = json.load(open(os.path.join(d, "c5_info.json")))
    assert abs(ig["pcg_iters"] - io["pcg_iters"]) <= 1, (ig["pcg_iters"], io["pcg_iters"])
    used = g.kernels_used()
    for k in ("k_momentumv<f64,central>", "k_div_rhsv<f64>", "k_pcg_initv<f64>", "k_mg_down<f64,TR16,UPD>", "k_mg_up<f64,TR16,DOT>",
              "k_mg_down<f64,TR8>", "k_pcg_dirapply2<f64>", "k_projectv<f64>"):
        assert k in used, (k, used)
    errs = {}
    for c in "uvwp":
        ref = np.load(os.path.join(d, "c5_%s.npy" % c), mmap_mode="r")
        errs[c] = relerr(g.get(c), ref)
    assert all(e < TOL64 for e in errs.values()), errs
    g.close()
