"""Runs the CPU oracle for ONE step of a BASELINE.json config at its FULL size in a process of its own and leaves the
result as .npy files (test infrastructure: started by tests/conftest.py when the full-size GPU parity tests are
selected, so that the minutes of single-threaded oracle time overlap the rest of the GPU suite).

    python tests/fullsize_oracle_worker.py <c2|c3|c4|c5> <outdir>

Writes <outdir>/<case>_{u,v,w,p}.npy, the initial fields for c5 (built once, on the CPU, so that both sides start from
bit-identical arrays), <case>_cell_{base,perm,keys,seg}.npy, and <case>_info.json last of all (its presence = done).
Calls only oracle/ and fs_workloads.
"""
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import fs_workloads as W  # noqa: E402
from oracle import Oracle  # noqa: E402


def main():
    case, out = sys.argv[1], sys.argv[2]
    t0 = time.time()
    cfg = W.make(case)
    if case == "c5":
        for c in "uvw":
            np.save(os.path.join(out, "%s_init_%s.npy" % (case, c)), cfg["init"][c])
    o = Oracle(cfg)
    for c, a in cfg["init"].items():
        o.set(c, a)
    if cfg.get("markers") is not None:
        o.set_markers(*cfg["markers"])
    if cfg.get("body") is not None:
        o.set_body(*cfg["body"])
    t1 = time.time()
    info = o.step(1)
    t2 = time.time()
    for c in "uvwp":
        np.save(os.path.join(out, "%s_%s.npy" % (case, c)), o.get(c))
    if cfg.get("markers") is not None:
        o.step(0)
        cl = o.cell_list()
        for k in ("base", "perm", "keys"):
            np.save(os.path.join(out, "%s_cell_%s.npy" % (case, k)), cl[k])
        np.save(os.path.join(out, "%s_cell_seg.npy" % case), cl["seg_start"])
        X, Ub, F = o.markers()
        np.save(os.path.join(out, "%s_marker_x.npy" % case), X)
        np.save(os.path.join(out, "%s_marker_f.npy" % case), F)
    info["setup_s"] = t1 - t0
    info["step_s"] = t2 - t1
    tmp = os.path.join(out, "%s_info.json.tmp" % case)
    json.dump(info, open(tmp, "w"))
    os.replace(tmp, os.path.join(out, "%s_info.json" % case))


if __name__ == "__main__":
    main()
