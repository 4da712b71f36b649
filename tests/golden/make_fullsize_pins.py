"""Writes tests/golden/fullsize_<config>.txt: the CPU oracle's result for a BASELINE.json config at its FULL size
and FULL step count, reduced to what fits a text fixture -- PCG iterations per step, body state, per-field maxima and
the values at seeded sample points (initial condition and final fields).  The GPU parity test
(tests/test_gpu_fullsize.py) replays the same config through the C ABI and compares at 1e-9 (north_star).

    python tests/golden/make_fullsize_pins.py c2|c3|c4|c5 [--steps K]

Calls only oracle/ and fs_workloads (input generators).  Single-threaded oracle: c2 ~25 min, c3 ~30 min, c4 ~2.5 h,
c5 (512^3, ~27 GB) ~35 min on one core.  Sample points: NS seeded flat indices per field; for the IBM configs half of
them are drawn from the box around the markers, where the direct forcing acts.
"""
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
import fs_workloads as W  # noqa: E402
from oracle import Oracle  # noqa: E402

NS = 192


def sample_indices(cfg, name, shape, seed=20250523):
    """NS flat indices into field `name` (shared with the test: pure function of the config)."""
    rng = np.random.default_rng([seed, "uvwp".index(name)])
    n = int(np.prod(shape))
    idx = rng.integers(0, n, size=NS)
    if cfg.get("markers") is not None:
        X = np.asarray(cfg["markers"][0])
        h = cfg["lx"] / cfg["nx"]
        lo = np.floor((X.min(axis=0) - np.array([cfg["x0"], cfg["y0"], cfg["z0"]])) / h).astype(int) - 3
        hi = np.ceil((X.max(axis=0) - np.array([cfg["x0"], cfg["y0"], cfg["z0"]])) / h).astype(int) + 3
        nz, ny, nx = shape
        i = rng.integers(max(lo[0], 0), min(hi[0], nx - 1) + 1, size=NS // 2)
        j = rng.integers(max(lo[1], 0), min(hi[1], ny - 1) + 1, size=NS // 2)
        k = rng.integers(max(lo[2], 0), min(hi[2], nz - 1) + 1, size=NS // 2)
        idx[: NS // 2] = i + nx * (j + ny * k)
    return idx


def main():
    name = sys.argv[1]
    cfg = W.make(name)
    steps = cfg["steps"]
    if "--steps" in sys.argv:
        steps = int(sys.argv[sys.argv.index("--steps") + 1])
    o = Oracle(cfg)
    for c, a in cfg["init"].items():
        o.set(c, a)
    if cfg.get("markers") is not None:
        o.set_markers(*cfg["markers"])
    if cfg.get("body") is not None:
        o.set_body(*cfg["body"])
    ic = {c: np.asarray(cfg["init"][c]).reshape(-1)[sample_indices(cfg, c, o.shape[c])] for c in "uvw"}
    t0 = time.time()
    info = o.step(steps)
    dt = time.time() - t0
    out = os.path.join(HERE, "fullsize_%s.txt" % name)
    with open(out, "w") as f:
        f.write("# %s %dx%dx%d, %d steps: CPU oracle (oracle/fs_oracle.cpp), written by make_fullsize_pins.py in %.0f s\n"
                % (cfg["name"], cfg["nx"], cfg["ny"], cfg["nz"], steps, dt))
        f.write("steps %d\n" % steps)
        f.write("iters %s\n" % " ".join(str(i) for i in info["iters_per_step"]))
        for k in ("body_force", "body_disp", "body_vel"):
            f.write("%s %s\n" % (k, " ".join(float(x).hex() for x in info[k])))
        f.write("max_abs_div %s\n" % float(info["max_abs_div"]).hex())
        for c in "uvw":
            for q, v in zip(sample_indices(cfg, c, o.shape[c]), ic[c]):
                f.write("ic %s %d %s\n" % (c, q, float(v).hex()))
        for c in "uvwp":
            a = o.get(c)
            f.write("max %s %s\n" % (c, float(np.abs(a).max()).hex()))
            for q in sample_indices(cfg, c, a.shape):
                f.write("val %s %d %s\n" % (c, q, float(a.reshape(-1)[q]).hex()))
    print(out, "%.0f s" % dt)


if __name__ == "__main__":
    main()
