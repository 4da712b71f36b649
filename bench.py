#!/usr/bin/env python
"""bench.py -- throughput of one full fractional step (all rows of SURVEY.md 8(a)) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--dtype f64|f32] [--n 512]
    python bench.py --impl reference ...      # the CPU oracle, as it stands, on the host cores

Workload (BASELINE.json configs[4], the case north_star's target is stated on): decaying homogeneous
isotropic turbulence, triply periodic n^3 (default 512^3), random-phase solenoidal field with
E(k) ~ k^4 exp(-2 (k/4)^2), u_rms = 1, nu = 1e-3, dt = 5e-4, AB2, GMG-preconditioned CG to rel tol
1e-8.  Synthetic, seeded (fs_workloads.hit).  One "step" = one fs_step = momentum RHS + predictor,
(IBM: none in c5), Poisson RHS, PCG with one V(2,2) cycle per iteration, projection.

Prints ONE JSON line (contract in the task statement): metric Mcell-steps/s, `roofline` for the
dominant kernel (event-timed through fs_profile_step), `cpu_baseline` (oracle on a bounded sample: one step of
the full 512^3 box when the host has the memory, else a labelled 128^3 replica), `e2e` (host buffers in and out
through the C ABI every step), `clocks`, `gpu_launches`, and -- BASELINE.json's metric is "fp64/fp32" -- an
`fp32` block (value, ms_per_step, roofline, clocks) measured in the same process on the same workload.
Multi-GPU: the path does not shard (replicas only) -- every rank advances
its own independent grid, no collective on the data path; timing = max over ranks.
"""
import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "Mcell-steps/s per full fractional step"
UNIT = "Mcell-steps/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"])
    ap.add_argument("--n", type=int, default=512, help="cells per direction of the HIT box (c5: 512)")
    ap.add_argument("--workload", default="c5", choices=["c1", "c2", "c3", "c4", "c5"],
                    help="c5 (default) is the metric's configuration; c1-c4 are the small, L2-resident parity configs "
                         "(launch/latency bound: reported for context in profiles/, fp64 only)")
    ap.add_argument("--ref-n", type=int, default=128, help="replica size the CPU oracle is timed on")
    ap.add_argument("--exec", dest="exec_mode", default="graph", choices=["graph", "stream"],
                    help="graph: one CUDA-graph replay per step (default); stream: same kernels launched directly (for ncu)")
    ap.add_argument("--single-dtype", action="store_true", help="measure only --dtype (default: the other precision too, as an extra block)")
    ap.add_argument("--cpu-replica", action="store_true", help="time the CPU oracle on the --ref-n replica even if the host could hold the full box")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-profile", action="store_true")
    ap.add_argument("--precond", default=None, choices=["none", "jacobi", "gmg"],
                    help="override the workload's Poisson preconditioner (context runs: e.g. c3 with the multigrid of reading G1)")
    ap.add_argument("--traffic-from", nargs="+", metavar="DTYPE=RAW.CSV", help="write profiles/r2_traffic.csv from ncu raw CSV dumps (no GPU run)")
    return ap.parse_args()


# ----------------------------------------------------------------------------------------- clocks
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def max_over_ranks(x, dist, device):
    """Timing rule of the contract: a multi-rank number is the MAX over ranks (replicas run independently,
    the job is as slow as its slowest rank).  dist is None for a single process."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([float(x)], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def csrc_hash():
    """sha256 over the CUDA sources + the ABI header: ties a committed ncu capture to the code it was taken from."""
    from paper_2505_23940_b200.build import csrc_hash as h
    return h()


def ncu_traffic(dtype, label):
    """DRAM bytes per launch of the kernel behind a profile label, from the committed ncu --set full summary
    (profiles/r2_traffic.csv: dtype,label,kernel,grid,dram_read_bytes,dram_write_bytes; first line
    `# csrc_sha256=<hash>` of the sources the capture was taken from).  Returns (bytes or None, note): the capture
    is REFUSED when its hash differs from the sources this run was built from."""
    path = os.path.join(ROOT, "profiles", "r2_traffic.csv")
    if not os.path.exists(path):
        return None, "no committed capture (profiles/r2_traffic.csv)"
    lines = open(path).read().splitlines()
    rec = lines[0].split("=", 1)[1].strip() if lines and lines[0].startswith("# csrc_sha256=") else None
    cur = csrc_hash()
    if rec != cur:
        return None, "committed capture is from other sources (csrc %s..., this build %s...): refused" % (str(rec)[:12], cur[:12])
    for line in lines[1:]:
        f = [x.strip() for x in line.split(",")]
        if len(f) >= 6 and f[0] == dtype and f[1] == label:
            try:
                return float(f[4]) + float(f[5]), "ncu --set full capture of these sources (csrc %s...), profiles/r2_traffic.csv" % cur[:12]
            except ValueError:
                break
    return None, "kernel not in the committed capture"


TRAFFIC_LABELS = (("k_momentum", "momentum_predictor"), ("k_div_rhs", "div_rhs"), ("k_pcg_init", "pcg_init"), ("k_mg_down", "mg_down_l0"),
                  ("k_mg_up", "mg_up_l0"), ("k_pcg_dirapply", "pcg_dir_apply_dot"), ("k_project", "project"), ("k_pflush", "p_flush_mean"))


def traffic_from_ncu(raw_csvs):
    """`python bench.py --traffic-from f64=<raw.csv> f32=<raw.csv>`: turns `ncu -i <rep> --page raw --csv` dumps of
    `ncu --set full ... python bench.py --exec stream --single-dtype --dtype <d>` into profiles/r2_traffic.csv: per dtype and
    profile label the DRAM bytes of the LAST launch of the kernel's largest grid (steady state), stamped with the hash of
    the sources this checkout holds (ncu_traffic refuses the file when the sources change).  No GPU needed."""
    import csv
    out = ["# csrc_sha256=%s" % csrc_hash(),
           "# dtype,label,kernel,grid,dram_read_bytes,dram_write_bytes,duration_us  (per launch; ncu --set full --clock-control none; see r2_ncu_full.md)"]
    for spec in raw_csvs:
        dtype, path = spec.split("=", 1)
        rows = list(csv.reader(open(path)))
        h, units = rows[0], rows[1]
        col = {n: i for i, n in enumerate(h)}

        def val(r, name):
            v, u = float(r[col[name]].replace(",", "")), units[col[name]]
            scale = {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0, "ms": 1e3, "us": 1.0, "ns": 1e-3, "s": 1e6}.get(u, 1.0)
            return v * scale
        best = {}
        for r in rows[2:]:
            name = r[col["Kernel Name"]]
            for prefix, label in TRAFFIC_LABELS:
                if name.split("<")[0].split(" ")[-1].startswith(prefix):
                    grid = r[col["Grid Size"]]
                    ncta = 1
                    for x in grid.strip("()").split(","):
                        ncta *= int(x)
                    if label not in best or ncta >= best[label][0]:
                        best[label] = (ncta, name, grid, val(r, "dram__bytes_read.sum"), val(r, "dram__bytes_write.sum"), val(r, "gpu__time_duration.sum"))
        for label, (ncta, name, grid, rd, wr, us) in sorted(best.items()):
            kn = name.replace("void ", "").split("(")[0].replace(",", ";")
            out.append("%s,%s,%s,%s,%.0f,%.0f,%.1f" % (dtype, label, kn, grid.replace(",", ";"), rd, wr, us))
    path = os.path.join(ROOT, "profiles", "r2_traffic.csv")
    open(path, "w").write("\n".join(out) + "\n")
    print(path)


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def host_info():
    model, mem_kb = "unknown", 0
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                model = line.split(":", 1)[1].strip()
                break
        for line in open("/proc/meminfo"):
            if line.startswith("MemAvailable"):
                mem_kb = int(line.split()[1])
    except OSError:
        pass
    return {"nproc": os.cpu_count(), "cpu_model": model, "mem_available_gb": round(mem_kb / 1048576.0, 1)}


# ----------------------------------------------------------------------------------------- reference arm
WORKLOAD = "c5 decaying HIT %d^3 triply periodic, AB2, GMG-PCG rtol 1e-8 (BASELINE.json configs[4])"


def oracle_sample(n, steps, init=None):
    """The CPU oracle as it stands (single thread, fp64) on an n^3 box of the workload (init: fields to start from,
    else the seeded recipe at that size)."""
    import fs_workloads as W
    from oracle import Oracle
    if init is None:
        cfg = W.hit(n=n)
        init = cfg["init"]
    else:
        cfg = W.hit(n=32)
        L = cfg["lx"]
        cfg.update(nx=n, ny=n, nz=n, lx=L, ly=L, lz=L)
    o = Oracle(cfg)
    for c in "uvw":
        o.set(c, init[c])
    t0 = time.perf_counter()
    info = o.step(steps)
    dt = time.perf_counter() - t0
    return n ** 3 * steps / dt / 1e6, dt, info["iters_per_step"]


def run_reference(a):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n = a.ref_n
    # warm-up on a tiny replica (library load, page-in), then K timed steps of the bounded sample
    oracle_sample(32, max(1, min(a.warmup, 2)))
    v, dt, iters = oracle_sample(n, a.steps)
    hi = host_info()
    sample = ("each step = one step of a %d^3 replica of the workload (same recipe, seed, nu, dt, GMG-PCG rtol 1e-8; %d cells "
              "instead of %d), %d steps, %.1f s; throughput is per cell, so the replica stands for the full box up to cache effects"
              % (n, n ** 3, a.n ** 3, a.steps, dt))
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": a.gpus, "steps": a.steps,
            "warmup": a.warmup, "ms_per_step": 1e3 * dt / a.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD % a.n, "cells": a.n ** 3, "sample_cells": n ** 3, "pcg_iters_per_step": iters},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample, "extrapolated": n != a.n,
                             "nproc": hi["nproc"], "cpu_model": hi["cpu_model"]},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------- our arm
def measure(a, dtype, dev, local, rank, world, dist, with_e2e, with_profile):
    """One grid of the workload in `dtype`: W warm-up steps, K steps between CUDA events on the library's stream
    (inputs resident in HBM), optional e2e leg (host buffers through the C ABI) and per-kernel event timing."""
    import torch
    import fs_workloads as W
    import paper_2505_23940_b200 as fs

    n = a.n
    wbytes = 8 if dtype == "f64" else 4
    if a.workload == "c5":
        cfg = W.hit(n=n, dtype=dtype, device=dev, exec_mode=a.exec_mode)   # seeded IC, built with torch FFT on the device
    else:
        cfg = W.make(a.workload, dtype=dtype, exec_mode=a.exec_mode, **({"precond": a.precond} if a.precond else {}))
    cells = cfg["nx"] * cfg["ny"] * cfg["nz"]
    g = fs.from_workload(cfg, device=dev)
    cfg["init"] = None
    torch.cuda.empty_cache()
    stream = g.stream

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(a.warmup):
        g.step(1, sync=False)
    info_w = g.step(0)
    l0 = g.launch_count()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    g.step(a.steps, sync=False)
    e1.record(stream)
    barrier()
    ms = e0.elapsed_time(e1)
    info = g.step(0)
    launches = g.launch_count() - l0
    clocks = sampler.stop() if rank == 0 else None
    ms = max_over_ranks(ms, dist, dev)
    value = world * cells * a.steps / (ms * 1e-3) / 1e6
    # nothing skipped inside the timed region: every step's PCG converged and no NaN appeared (sticky device counters)
    assert info["unconverged_steps"] == info_w["unconverged_steps"] == 0 and info["nan_steps"] == 0, info

    # ---- end to end through the C ABI with HOST buffers (pinned): per step H2D of u,v,w, fs_step, D2H of u,v,w,p
    e2e = None
    if with_e2e:
        tdt = torch.float64 if dtype == "f64" else torch.float32
        host = {c: torch.empty(g.shape[c], dtype=tdt).pin_memory() for c in "uvwp"}
        npv = {c: host[c].numpy() for c in "uvwp"}
        for c in "uvwp":
            g.get(c, dtype=dtype, out=npv[c])
        ke = max(2, min(a.steps, 3))

        def e2e_step():
            for c in "uvw":
                g.set(c, npv[c])
            g.step(1, sync=False)
            for c in "uvwp":
                g.get(c, dtype=dtype, out=npv[c])

        e2e_step()                                        # warm-up
        barrier()
        t0 = time.perf_counter()
        for _ in range(ke):
            e2e_step()
        barrier()
        dt = time.perf_counter() - t0
        dt = max_over_ranks(dt, dist, dev)
        e2e = {"value": world * cells * ke / dt / 1e6, "unit": UNIT,
               "h2d_bytes_per_step": 3 * cells * wbytes, "d2h_bytes_per_step": 4 * cells * wbytes,
               "steps": ke, "ms_per_step": 1e3 * dt / ke,
               "api": "fs_fields_set(u,v,w: pinned host) -> fs_step(1) -> fs_fields_get(u,v,w,p: pinned host)"}
        # the same traffic for TWO independent grids (replicas), each on its own stream, through the asynchronous
        # field calls: one grid's H2D / D2H runs while the other one steps (PCIe is full duplex), per step and grid the same bytes
        try:
            s2 = torch.cuda.Stream(device=dev)
            with torch.cuda.stream(s2):
                g2 = fs.Grid(dict(cfg, dtype=dtype), device=dev, stream=s2)       # same workload; its fields arrive through the pipeline
            host2 = {c: torch.empty(g.shape[c], dtype=tdt).pin_memory() for c in "uvwp"}
            for c in "uvwp":
                host2[c].copy_(host[c])
            pairs = ((g, host), (g2, host2))

            def pipe_round():
                for gg, hh in pairs:
                    for c in "uvw":
                        gg.set_async(c, hh[c])
                    gg.step(1, sync=False)
                    for c in "uvwp":
                        gg.get_async(c, hh[c])

            pipe_round(); torch.cuda.synchronize(dev)
            barrier()
            t0 = time.perf_counter()
            for _ in range(ke):
                pipe_round()
            torch.cuda.synchronize(dev)
            dtp = max_over_ranks(time.perf_counter() - t0, dist, dev)
            e2e["pipelined_two_replicas"] = {"value": world * 2 * cells * ke / dtp / 1e6, "unit": UNIT, "ms_per_round": 1e3 * dtp / ke,
                                             "note": "two independent grids on two streams, fs_fields_set_async / fs_step / fs_fields_get_async: "
                                                     "the copies of one grid overlap the step and the opposite-direction copies of the other"}
            g2.close(); del g2, host2
        except RuntimeError as ex:      # e.g. not enough memory for a second grid: the serial number stands alone
            e2e["pipelined_two_replicas"] = {"value": None, "note": "skipped: %s" % str(ex)[:120]}
        del host, npv

    # ---- per-kernel event timing (same kernels, stream launches) -> roofline of the dominant kernel
    roof, kernels = None, None
    if with_profile and rank == 0:
        peak, peak_src = peaks()
        ksteps = 2
        prof = g.profile_step(ksteps)
        # the first level-0 down launch of every solve has no residual update to do (2.125 words instead of 4.125)
        if "mg_down_l0" in prof and prof["mg_down_l0"]["bytes"] > 4.0 * wbytes * cells * prof["mg_down_l0"]["launches"]:
            prof["mg_down_l0"]["bytes"] -= 2.0 * wbytes * cells * ksteps
        # the V-cycle levels >= 1 and the one-CTA tail are reported as one entry, "mg_coarse" (per-level times inside it)
        import re
        sub = {k: prof.pop(k) for k in list(prof) if re.fullmatch(r"mg_(down|up)_l[1-9][0-9]*|mg_tail", k)}
        if sub:
            prof["mg_coarse"] = {"launches": sum(v["launches"] for v in sub.values()) + prof.get("mg_coarse", {}).get("launches", 0),
                                 "ms": sum(v["ms"] for v in sub.values()) + prof.get("mg_coarse", {}).get("ms", 0.0),
                                 "bytes": sum(v["bytes"] for v in sub.values()) + prof.get("mg_coarse", {}).get("bytes", 0.0)}
        tot = sum(v["ms"] for v in prof.values())
        kernels = {k: {"launches_per_step": v["launches"] / ksteps, "ms_per_step": v["ms"] / ksteps,
                       "share": v["ms"] / tot if tot else 0.0,
                       "algorithmic_GBps": (v["bytes"] / (v["ms"] * 1e-3) / 1e9) if v["ms"] > 0 else None}
                   for k, v in sorted(prof.items(), key=lambda kv: -kv[1]["ms"])}
        if sub:
            kernels["mg_coarse"]["levels_ms_per_step"] = {k: v["ms"] / ksteps for k, v in sorted(sub.items())}
        top = max(prof.items(), key=lambda kv: kv[1]["ms"])
        ach = top[1]["bytes"] / (top[1]["ms"] * 1e-3) / 1e9
        step_bytes = sum(v["bytes"] for v in prof.values()) / ksteps
        step_s = ms / a.steps * 1e-3
        # SURVEY 8(d) model of the UNFUSED formulation: 25 + 29.4 N_it words per cell-step (GMG-PCG)
        nit = sum(v["launches"] for k, v in prof.items() if k == "pcg_dir_apply_dot") / ksteps
        unfused_bytes = (25.0 + (29.4 if cfg["precond"] == "gmg" else 11.0) * nit) * wbytes * cells
        traffic, traffic_note = ncu_traffic(dtype, top[0])
        roof = {"bound": "hbm", "kernel": top[0], "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                "traffic": traffic, "traffic_source": traffic_note, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": top[1]["bytes"] / top[1]["launches"],
                "avg_launch_ms": top[1]["ms"] / top[1]["launches"], "share_of_step": top[1]["ms"] / tot,
                "step": {"algorithmic_bytes": step_bytes, "achieved": step_bytes / step_s / 1e9,
                         "frac": step_bytes / step_s / 1e9 / peak, "frac_of_nominal_8TBps": step_bytes / step_s / 1e9 / 8000.0,
                         "note": "sum of per-kernel algorithmic bytes (fused kernels: DESIGN.md 7) of one step / graph-replay step time"},
                "step_unfused_model": {"algorithmic_bytes": unfused_bytes, "achieved": unfused_bytes / step_s / 1e9,
                                       "frac": unfused_bytes / step_s / 1e9 / peak, "pcg_iters_per_step": nit,
                                       "note": "SURVEY 8(d): (25 + 29.4 N_it) words per cell-step, every pass a separate kernel"}}
    out = {"value": value, "ms": ms, "info": info, "launches": int(launches), "clocks": clocks, "e2e": e2e, "roofline": roof,
           "kernels": kernels, "cells": cells, "cfg": cfg, "wbytes": wbytes, "kernels_used": g.kernels_used()}
    g.close()
    del g
    torch.cuda.empty_cache()
    return out


def run_ours(a):
    import torch
    import paper_2505_23940_b200 as fs

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product has no CPU fallback")
    fs.lib()
    torch.cuda.set_device(local)
    dev = "cuda:%d" % local
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(dev))

    n = a.n
    m = measure(a, a.dtype, dev, local, rank, world, dist, not a.no_e2e, not a.no_profile)
    cfg, cells, wbytes, info = m["cfg"], m["cells"], m["wbytes"], m["info"]
    if dist is not None:
        dist.barrier()
    # ---- the other precision of BASELINE.json's metric ("fp64/fp32"), same process, same workload and step counts
    other = None
    if not a.single_dtype and a.workload == "c5":
        od = "f32" if a.dtype == "f64" else "f64"
        mo = measure(a, od, dev, local, rank, world, dist, False, not a.no_profile)
        r = mo["roofline"]
        other = {"dtype": od, "value": mo["value"], "unit": UNIT, "ms_per_step": mo["ms"] / a.steps, "steps": a.steps, "warmup": a.warmup,
                 "pcg_iters_last_step": mo["info"]["pcg_iters"], "rel_residual": mo["info"]["rel_residual"],
                 "true_rel_residual": mo["info"]["true_rel_residual"], "max_abs_div": mo["info"]["max_abs_div"],
                 "converged": mo["info"]["converged"], "unconverged_steps": mo["info"]["unconverged_steps"], "nan_steps": mo["info"]["nan_steps"],
                 "gpu_launches": mo["launches"], "clocks": mo["clocks"],
                 "roofline": None if r is None else {k: r[k] for k in ("bound", "kernel", "achieved", "peak", "unit", "frac", "traffic",
                                                                       "traffic_source", "avg_launch_ms", "share_of_step", "step")},
                 "kernels": mo["kernels"]}
        if dist is not None:
            dist.barrier()

    # ---- CPU oracle on a bounded sample (rank 0, N=1 only): one step of the FULL box when the host has the memory
    #      (>= 24 GB; the oracle holds ~27 GB of fp64 fields at 512^3), else the 128^3 replica, labelled
    cpu = None
    if not a.no_cpu and rank == 0 and world == 1:
        hi = host_info()
        full = a.workload == "c5" and not a.cpu_replica and hi["mem_available_gb"] >= 40.0 * (n / 512.0) ** 3
        if full:
            import fs_workloads as W
            init = W.hit(n=n, dtype="f64", device=dev)["init"]
            init = {c: init[c].cpu().numpy() for c in "uvw"}
            torch.cuda.empty_cache()
            v, dt, its = oracle_sample(n, 1, init=init)
            sample = "c5 HIT %d^3 (the full box, same seeded initial field), 1 step from rest (p0 = 0), %d PCG iterations, %.1f s" % (n, its[0], dt)
        else:
            v, dt, its = oracle_sample(a.ref_n, 6)
            sample = "c5 HIT REPLICA %d^3, 6 steps, %.1f s; per-cell throughput taken as the full box's (linear-in-cells extrapolation)" % (a.ref_n, dt)
        cpu = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample + " (single-threaded fp64 C++ oracle)",
               "extrapolated": not full, "nproc": hi["nproc"], "cpu_model": hi["cpu_model"], "mem_available_gb": hi["mem_available_gb"]}

    if rank == 0:
        line = {"metric": METRIC, "value": m["value"], "unit": UNIT, "n_gpus": world, "steps": a.steps, "warmup": a.warmup,
                "ms_per_step": m["ms"] / a.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": a.dtype, "data": "synthetic",
                "config": {"workload": (WORKLOAD % n) if a.workload == "c5"
                           else "%s %dx%dx%d (BASELINE.json configs[%d]; small L2-resident case, context only)" % (cfg["name"], cfg["nx"], cfg["ny"], cfg["nz"], int(a.workload[1]) - 1),
                           "cells": cells, "parallelism": "replicas x%d (no sharding)" % world,
                           "l2": ("inputs larger than L2 (each field %.0f MB vs 126 MB L2)" if cells * wbytes > 126e6 else "fields of %.0f MB: L2 resident, no flush (context run)") % (cells * wbytes / 1e6),
                           "pcg_iters_last_step": info["pcg_iters"], "rel_residual": info["rel_residual"],
                           "true_rel_residual": info["true_rel_residual"], "max_abs_div": info["max_abs_div"],
                           "converged": info["converged"], "nan_flag": info["nan_flag"],
                           "unconverged_steps": info["unconverged_steps"], "nan_steps": info["nan_steps"],
                           "exec": ("one CUDA graph replay per step, PCG loop = conditional WHILE node" if a.exec_mode == "graph"
                                    else "stream launches, host polls the PCG flag"),
                           "kernels_used": m["kernels_used"]},
                "roofline": m["roofline"], "cpu_baseline": cpu, "e2e": m["e2e"], "clocks": m["clocks"],
                "gpu_launches": m["launches"], "kernels": m["kernels"]}
        if other is not None:
            line["fp32" if other["dtype"] == "f32" else "fp64"] = other
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def main():
    a = parse()
    if a.traffic_from:
        traffic_from_ncu(a.traffic_from)
        return
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)


if __name__ == "__main__":
    main()
