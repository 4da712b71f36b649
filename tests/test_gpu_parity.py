"""GPU parity: the CUDA path (through the C ABI, via the thin binding) against the CPU oracle on the
same seeded inputs, element by element.  Acceptance (BASELINE.json north_star):
fp64 fields <= 1e-9 max relative error (per field, ||gpu - oracle||_inf / ||oracle||_inf) after the
config's steps with PCG iteration counts within +-1 per step; fp32 fields <= 1e-4 of the fp64 oracle
over 5 steps; marker indices / perm / keys / seg_start bit-exact."""
import math

import numpy as np
import pytest

import fs_workloads as W

pytestmark = pytest.mark.gpu

TOL64 = 1e-9     # north_star: fp64 fields within 1e-9 max relative error
TOL32 = 1e-4     # north_star: fp32 fields within 1e-4 of the fp64 oracle over 5 steps


@pytest.fixture(scope="module")
def fs():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2505_23940_b200 as fs
    fs.lib()
    return fs


def _oracle(cfg):
    from oracle import Oracle
    o = Oracle(cfg)
    for c, a in cfg.get("init", {}).items():
        o.set(c, a)
    if cfg.get("markers") is not None:
        o.set_markers(*cfg["markers"])
    if cfg.get("body") is not None:
        o.set_body(*cfg["body"])
    if cfg.get("beam") is not None:
        o.set_beam(*cfg["beam"])
    return o


def relerr(a, b):
    """A9 norm: max |a-b| / max |b| (absolute when the reference is identically zero)."""
    d = float(np.abs(np.asarray(a, dtype=np.float64) - b).max())
    s = float(np.abs(b).max())
    return d / s if s > 0 else d


def _rand_fields(cfg, seed, solenoidal_bc=True):
    rng = np.random.default_rng(seed)
    sh = W.shapes(cfg)
    f = {c: rng.standard_normal(sh[c]) for c in "uvw"}
    # boundary-normal faces of bounded directions carry the prescribed values
    if cfg["bc"][0] != "periodic":
        f["u"][:, :, 0] = cfg["bc_vel"][0][0]; f["u"][:, :, -1] = cfg["bc_vel"][1][0]
    if cfg["bc"][2] != "periodic":
        f["v"][:, 0, :] = 0.0; f["v"][:, -1, :] = 0.0
    if cfg["bc"][4] != "periodic":
        f["w"][0] = 0.0; f["w"][-1] = 0.0
    return f


def _cfg_periodic(nx, ny, nz, **kw):
    h = 2 * math.pi / nx
    return W._base(nx=nx, ny=ny, nz=nz, lx=nx * h, ly=ny * h, lz=nz * h, nu=0.01, dt=1e-3, **kw)


def _cfg_channel(nx, ny, nz, **kw):
    j = np.arange(ny + 1)
    yf = np.tanh(2.0 * (2.0 * j / ny - 1.0)) / math.tanh(2.0)
    yf[0], yf[-1] = -1.0, 1.0
    c = W._base(nx=nx, ny=ny, nz=nz, lx=2 * math.pi, ly=2.0, lz=math.pi, y0=-1.0, yf=yf, nu=1 / 180.0, dt=2e-4,
                body_force=[1.0, 0.0, 0.0], **kw)
    c["bc"] = ["periodic", "periodic", "noslip", "noslip", "periodic", "periodic"]
    c["bc_vel"][3] = [0.3, 0.0, -0.2]      # moving lid exercises the 2*u_wall - u ghost
    return c


def _cfg_open(nx, ny, nz, **kw):
    h = 1.0 / 16
    c = W._base(nx=nx, ny=ny, nz=nz, lx=nx * h, ly=ny * h, lz=nz * h, nu=1 / 300.0, dt=5e-3, **kw)
    c["bc"] = ["inflow", "outflow", "slip", "slip", "noslip", "slip"]
    c["bc_vel"][0] = [1.0, 0.0, 0.0]
    c["bc_vel"][1] = [1.0, 0.0, 0.0]
    return c


# ------------------------------------------------------------------------------------ S1 momentum kernel
@pytest.mark.parametrize("kind", ["periodic", "channel", "open"])
def test_momentum_rhs_elementwise(fs, kind):
    # sizes span several 32x4x2 tiles with ragged tails in every direction
    cfg = {"periodic": _cfg_periodic(72, 38, 21), "channel": _cfg_channel(40, 50, 19),
           "open": _cfg_open(70, 27, 22, inflow_noise=0.05, seed=3)}[kind]
    cfg["init"] = _rand_fields(cfg, 11)
    o = _oracle(cfg)
    ref = o.momentum_rhs()
    g = fs.from_workload(cfg)
    got = g.momentum_rhs()
    for c, a, b in zip("uvw", got, ref):
        assert relerr(a, b) < 1e-12, (kind, c, relerr(a, b))
    g.close()


@pytest.mark.parametrize("kind", ["periodic", "channel", "zwalls", "channel_upwind", "periodic_adaptive"])
def test_momentum_vector_kernel_elementwise(fs, kind, monkeypatch):
    # k_momentumv (one 16-byte vector of faces per thread; periodic x, walls in y / z): H^n element-wise against the oracle
    # in fp64 at 1e-12 (cp.async ring variant) and in fp32 (register-load variant) on the scale of fp32 rounding; the
    # predicted field through two full steps; and with FS_TUNE_MOMV=0 the same grid through k_momentum (one face per thread),
    # which otherwise only serves bounded x, odd nx and the LES closures.  Several tiles
    # (120 x 14 cells in fp32, 60 x 14 in fp64) with ragged tails, several z chunks.
    def zwalls(**kw):
        c = _cfg_periodic(136, 34, 40, **kw)
        c["bc"][4], c["bc"][5] = "noslip", "slip"
        c["bc_vel"][4] = [0.2, -0.1, 0.0]
        return c
    mk = {"periodic": lambda **kw: _cfg_periodic(136, 38, 37, **kw), "channel": lambda **kw: _cfg_channel(128, 50, 35, **kw), "zwalls": zwalls,
          "channel_upwind": lambda **kw: _cfg_channel(72, 31, 19, convection="upwind", **kw),
          "periodic_adaptive": lambda **kw: _cfg_periodic(64, 30, 33, cfl=0.3, **kw)}[kind]
    upw = "upwind" if "upwind" in kind else "central"
    cfg = mk()
    cfg["init"] = _rand_fields(cfg, 21)
    o = _oracle(cfg)
    ref = o.momentum_rhs()
    monkeypatch.setenv("FS_TUNE_MOMV", "0")
    g0 = fs.from_workload(cfg)
    got0 = g0.momentum_rhs()
    assert "k_momentum<f64,%s>" % upw in g0.kernels_used(), g0.kernels_used()
    for c, a, b in zip("uvw", got0, ref):
        assert relerr(a, b) < 1e-12, (kind, c, relerr(a, b))
    g0.close()
    monkeypatch.delenv("FS_TUNE_MOMV")
    g = fs.from_workload(cfg)
    got = g.momentum_rhs()
    assert "k_momentumv<f64,%s>" % upw in g.kernels_used(), g.kernels_used()
    for c, a, b in zip("uvw", got, ref):
        assert relerr(a, b) < 1e-12, (kind, c, relerr(a, b))
    io, ig = o.step(2), g.step(2)                      # second step: AB2 with history (variable step when cfl > 0)
    _compare_state(g, o, TOL64)
    assert abs(ig["dt"] - io["dt"]) <= 1e-15 * io["dt"]
    g.close()
    g32 = fs.from_workload(dict(cfg, dtype="f32"))
    got32 = g32.momentum_rhs()
    assert "k_momentumv<f32,%s>" % upw in g32.kernels_used(), g32.kernels_used()
    for c, a, b in zip("uvw", got32, ref):
        assert relerr(a, b) < 2e-5, (kind, c, relerr(a, b))     # fp32: eps32 x the cancellation in the flux differences (|u| / h ~ 50)
    g32.close()


@pytest.mark.parametrize("kind", ["periodic", "channel", "open"])
def test_momentum_rhs_upwind_elementwise(fs, kind):
    # NEXT-3: first-order upwind convective fluxes (random fields: both signs of every advecting velocity)
    cfg = {"periodic": _cfg_periodic(72, 38, 21, convection="upwind"), "channel": _cfg_channel(40, 50, 19, convection="upwind"),
           "open": _cfg_open(70, 27, 22, inflow_noise=0.05, seed=3, convection="upwind")}[kind]
    cfg["init"] = _rand_fields(cfg, 12)
    ref = _oracle(cfg).momentum_rhs()
    g = fs.from_workload(cfg)
    got = g.momentum_rhs()
    for c, a, b in zip("uvw", got, ref):
        assert relerr(a, b) < 1e-12, (kind, c, relerr(a, b))
    g.close()


def test_upwind_full_steps_match_oracle(fs):
    cfg = W.taylor_green(n=24, convection="upwind")
    g, o, ig, io, _ = _run_pair(fs, cfg, 6)
    g.close()
    cfg = W.channel(n=24, convection="upwind", steps=4)
    g, o, ig, io, _ = _run_pair(fs, cfg, 4)
    g.close()


# ------------------------------------------------------------------------------------ S6/S7 Poisson
@pytest.mark.parametrize("kind,pc", [("periodic", "none"), ("periodic", "jacobi"), ("periodic", "gmg"),
                                     ("channel", "jacobi"), ("open", "jacobi"), ("open", "none")])
def test_poisson_solve_matches_oracle(fs, kind, pc):
    if kind == "periodic":
        n = (48, 32, 40) if pc == "gmg" else (44, 30, 37)
        cfg = _cfg_periodic(*n, precond=pc, rtol=1e-10, warm_start=0)
        if pc == "gmg":
            h = 2 * math.pi / 48
            cfg.update(lx=48 * h, ly=32 * h, lz=40 * h)
    elif kind == "channel":
        cfg = _cfg_channel(36, 42, 20, precond=pc, rtol=1e-10, warm_start=0)
    else:
        cfg = _cfg_open(50, 23, 18, precond=pc, rtol=1e-10, warm_start=0)
    rng = np.random.default_rng(5)
    rhs = rng.standard_normal(W.shapes(cfg)["p"])
    o = _oracle(cfg)
    p_ref, iref = o.poisson_solve(rhs)
    g = fs.Grid(cfg)
    p, info = g.poisson_solve(rhs)
    assert info["converged"] == 1 and iref["converged"] == 1
    assert abs(info["iters"] - iref["pcg_iters"]) <= 1, (info, iref)
    assert relerr(p, p_ref) < TOL64, relerr(p, p_ref)
    assert info["true_rel_residual"] < 1e-8
    # warm start from the solution: 0 iterations
    cfg2 = dict(cfg, warm_start=1)
    g2 = fs.Grid(cfg2)
    p2, info2 = g2.poisson_solve(rhs, p0=p)
    assert info2["iters"] <= 1
    g.close(); g2.close()


@pytest.mark.parametrize("path", ["coop", "stream"])
def test_point_pcg_paths_cooperative_and_streaming(fs, path, monkeypatch):
    # point-preconditioned PCG runs as one persistent cooperative kernel on L2-sized grids (k_pcg_coop) and as the streaming
    # kernel pair inside the graph's WHILE node on large ones (k_pcg_dirapply2 + k_pcg_updatev); every parity grid is small,
    # so FS_TUNE_COOP=0 routes this test through the streaming kernels to keep both paths compared with the oracle
    if path == "stream":
        monkeypatch.setenv("FS_TUNE_COOP", "0")
    want = ("k_pcg_coop<f64>",) if path == "coop" else ("k_pcg_dirapply2<f64>", "k_pcg_updatev<f64>")
    rng = np.random.default_rng(6)
    for cfg in (_cfg_periodic(44, 30, 37, precond="jacobi", rtol=1e-10, warm_start=0), _cfg_channel(36, 42, 20, precond="jacobi", rtol=1e-10, warm_start=0),
                _cfg_open(50, 23, 18, precond="none", rtol=1e-10, warm_start=0), _cfg_open(50, 23, 18, precond="jacobi", rtol=1e-10, warm_start=0)):
        rhs = rng.standard_normal(W.shapes(cfg)["p"])
        p_ref, iref = _oracle(cfg).poisson_solve(rhs)
        g = fs.Grid(cfg)
        p, info = g.poisson_solve(rhs)
        assert info["converged"] == 1 and abs(info["iters"] - iref["pcg_iters"]) <= 1, (info, iref)
        assert relerr(p, p_ref) < TOL64 and info["true_rel_residual"] < 1e-8
        used = g.kernels_used()
        assert all(k in used for k in want), (path, used)
        g.close()
    if path == "coop":
        # more 16-byte vectors than resident threads (148 SMs x 4 CTAs x 256): every thread walks its grid-stride loop more than once
        cfg = _cfg_open(256, 64, 40, precond="jacobi", rtol=1e-9, warm_start=0)
        rhs = rng.standard_normal(W.shapes(cfg)["p"])
        p_ref, iref = _oracle(cfg).poisson_solve(rhs)
        g = fs.Grid(cfg)
        p, info = g.poisson_solve(rhs)
        assert info["converged"] == 1 and abs(info["iters"] - iref["pcg_iters"]) <= 1 and relerr(p, p_ref) < TOL64
        g.close()
    # full steps: channel (walls, stretched y) and the FSI cylinder (markers, body, open boundaries), fp64 and fp32
    g, o, ig, io, _ = _run_pair(fs, W.channel(n=32, steps=4), 4)
    assert all(k in g.kernels_used() for k in want)
    g.close()
    cfg = W.cylinder_fsi(scale=8, per_ring=24)
    g, o, ig, io, _ = _run_pair(fs, cfg, 4)
    assert all(k in g.kernels_used() for k in want)
    g32 = fs.from_workload(dict(cfg, dtype="f32"))
    i32 = g32.step(4)
    assert i32["converged"] == 1 and i32["nan_flag"] == 0
    for c_ in "uvp":
        assert relerr(g32.get(c_), o.get(c_)) < 1e-4, c_
    assert ("k_pcg_coop<f32>" if path == "coop" else "k_pcg_updatev<f32>") in g32.kernels_used()
    g.close(); g32.close()


@pytest.mark.parametrize("kind,pc", [("periodic", "jacobi"), ("periodic", "none"), ("channel", "jacobi"), ("open", "jacobi"),
                                     ("periodic", "gmg")])
def test_poisson_solve_fp32_matches_fp64_oracle(fs, kind, pc):
    # fp32 instantiation of the PCG kernels (4 cells per thread in the fused direction+apply kernel when
    # nx % 4 == 0, the one-cell kernel otherwise), all preconditioners, bounded x / y / z
    if kind == "periodic":
        cfg = _cfg_periodic(48, 32, 40, precond=pc, rtol=1e-5, warm_start=0)
        if pc == "gmg":
            h = 2 * math.pi / 48
            cfg.update(lx=48 * h, ly=32 * h, lz=40 * h)
    elif kind == "channel":
        cfg = _cfg_channel(36, 42, 20, precond=pc, rtol=1e-5, warm_start=0)
    else:
        cfg = _cfg_open(52, 23, 18, precond=pc, rtol=1e-5, warm_start=0)
    rng = np.random.default_rng(7)
    rhs = rng.standard_normal(W.shapes(cfg)["p"])
    p_ref, iref = _oracle(dict(cfg, rtol=1e-12)).poisson_solve(rhs)
    g = fs.Grid(dict(cfg, dtype="f32"))
    p, info = g.poisson_solve(rhs)
    assert info["converged"] == 1, info
    assert relerr(p, p_ref) < 2e-4, relerr(p, p_ref)
    g.close()


def test_poisson_zero_rhs_and_max_iter(fs):
    cfg = _cfg_periodic(32, 32, 32, precond="jacobi", rtol=1e-12, warm_start=0, max_iter=3)
    g = fs.Grid(cfg)
    p, info = g.poisson_solve(np.zeros(W.shapes(cfg)["p"]))
    assert info["iters"] == 0 and info["converged"] == 1 and np.all(p == 0.0)
    rng = np.random.default_rng(1)
    p, info = g.poisson_solve(rng.standard_normal(W.shapes(cfg)["p"]))
    assert info["iters"] == 3 and info["converged"] == 0
    g.close()


@pytest.mark.parametrize("dims", [(48, 32, 40), (136, 56, 72), (8, 8, 8), (64, 64, 64)])
def test_gmg_vcycle_elementwise(fs, dims):
    # several xy tiles of the fused kernels (60 x 12 cells), ragged tile tails, several z chunks, and a
    # box smaller than one tile (8^3: the tile wraps around the periodic box more than once)
    cfg = _cfg_periodic(*dims, precond="gmg")
    rng = np.random.default_rng(2)
    r = rng.standard_normal(W.shapes(cfg)["p"])
    z_ref = _oracle(cfg).vcycle(r)
    g = fs.Grid(cfg)
    z = g.gmg_vcycle(r)
    assert relerr(z, z_ref) < 1e-12, relerr(z, z_ref)
    g.close()


@pytest.mark.parametrize("bounded", [(1, 1, 1), (0, 1, 0), (1, 0, 1)])
def test_gmg_on_bounded_grids_matches_oracle(fs, bounded):
    # reading G1: multigrid on uniform boxes with Neumann pressure faces (boundary fluxes dropped on every level, true-diagonal
    # Jacobi); per-sweep kernels with the boundary flags.  V-cycle element-wise, V(1,2) too, Poisson solve, fp32 solve
    h = 1.0 / 16
    kinds = (("inflow", "outflow"), ("slip", "noslip"), ("noslip", "slip"))

    def mk(**kw):
        kw.setdefault("rtol", 1e-10)
        cfg = W._base(nx=48, ny=32, nz=40, lx=48 * h, ly=32 * h, lz=40 * h, nu=0.01, dt=1e-3, precond="gmg", warm_start=0, **kw)
        cfg["bc"] = [kinds[d][s_] if bounded[d] else "periodic" for d in range(3) for s_ in range(2)]
        return cfg
    rng = np.random.default_rng(8)
    for kw in (dict(), dict(mg_nu1=1, mg_nu2=2, mg_coarse_sweeps=5)):
        cfg = mk(**kw)
        r = rng.standard_normal(W.shapes(cfg)["p"])
        z_ref = _oracle(cfg).vcycle(r)
        g = fs.Grid(cfg)
        z = g.gmg_vcycle(r)
        assert relerr(z, z_ref) < 1e-12, (bounded, kw, relerr(z, z_ref))
        assert "k_mg_down<f64,TR8>" not in g.kernels_used()            # the fused periodic legs must not run on a bounded grid
        g.close()
    cfg = mk()
    rhs = rng.standard_normal(W.shapes(cfg)["p"])
    p_ref, iref = _oracle(cfg).poisson_solve(rhs)
    g = fs.Grid(cfg)
    p, info = g.poisson_solve(rhs)
    assert info["converged"] == 1 and abs(info["iters"] - iref["pcg_iters"]) <= 1 and iref["pcg_iters"] < 25, (info, iref)
    assert relerr(p, p_ref) < TOL64 and info["true_rel_residual"] < 1e-8
    g.close()
    g32 = fs.Grid(dict(mk(rtol=1e-6), dtype="f32"))
    p32, i32 = g32.poisson_solve(rhs)
    assert i32["converged"] == 1 and relerr(p32, p_ref) < TOL32
    g32.close()


def test_sphere_with_gmg_pcg_full_steps_match_oracle(fs):
    # the c3 recipe (open box, 400 markers) with the multigrid preconditioner instead of Jacobi: same fields, a tenth of the iterations
    cfg = W.sphere(scale=4, n_markers=400, precond="gmg", rtol=1e-10)
    g, o, ig, io, _ = _run_pair(fs, cfg, 5)
    assert max(io["iters_per_step"]) < 40
    cj = W.sphere(scale=4, n_markers=400, rtol=1e-10)
    oj = _oracle(cj); ij = oj.step(5)
    assert min(ij["iters_per_step"]) > 4 * max(io["iters_per_step"])
    assert relerr(o.get("u"), oj.get("u")) < 1e-7                     # the preconditioner changes the path to the solution, not the solution
    g.close()


@pytest.mark.parametrize("nu", [(1, 1, 16), (3, 2, 8), (0, 2, 4), (2, 2, 0)])
def test_gmg_vcycle_other_smoothing_counts(fs, nu):
    # V(nu1, nu2) other than the fused V(2,2) fast path: the generic per-sweep kernels (fs_kernels_mg.cu), incl. nu1 = 0
    # (no pre-smoothing: restriction of the bare right-hand side) and no coarsest-level sweeps
    cfg = _cfg_periodic(48, 32, 40, precond="gmg", mg_nu1=nu[0], mg_nu2=nu[1], mg_coarse_sweeps=nu[2])
    rng = np.random.default_rng(3)
    r = rng.standard_normal(W.shapes(cfg)["p"])
    z_ref = _oracle(cfg).vcycle(r)
    g = fs.Grid(cfg)
    z = g.gmg_vcycle(r)
    assert relerr(z, z_ref) < 1e-12, (nu, relerr(z, z_ref))
    g.close()


def test_gmg_pcg_with_v11_cycle_matches_oracle(fs):
    # PCG around the generic V-cycle: separate r.z and update kernels (no fused update, no second residual buffer)
    h = 2 * math.pi / 48
    cfg = _cfg_periodic(48, 32, 40, precond="gmg", rtol=1e-10, warm_start=0, mg_nu1=1, mg_nu2=1)
    cfg.update(lx=48 * h, ly=32 * h, lz=40 * h)
    rhs = np.random.default_rng(5).standard_normal(W.shapes(cfg)["p"])
    p_ref, iref = _oracle(cfg).poisson_solve(rhs)
    g = fs.Grid(cfg)
    p, info = g.poisson_solve(rhs)
    assert info["converged"] == 1 and abs(info["iters"] - iref["pcg_iters"]) <= 1, (info, iref)
    assert relerr(p, p_ref) < TOL64
    g.close()


# ------------------------------------------------------------------------------------ S2-S5 IBM
def _markers(cfg, n, seed, spread_cells=6.0):
    rng = np.random.default_rng(seed)
    h = cfg["lx"] / cfg["nx"]
    lo = np.array([cfg["x0"], cfg["y0"], cfg["z0"]])
    L = np.array([cfg["lx"], cfg["ly"], cfg["lz"]])
    centre = lo + 0.5 * L
    xyz = centre + spread_cells * h * (rng.random((n, 3)) - 0.5) * 2.0
    # some markers exactly on faces / centres (floor ties) and coincident pairs (sort stability)
    xyz[0] = lo + h * np.array([5.0, 7.0, 6.0])
    xyz[1] = lo + h * np.array([5.5, 7.5, 6.5])
    xyz[2] = xyz[1]
    xyz[3] = xyz[7]
    vel = rng.standard_normal((n, 3))
    dvol = h ** 3 * (0.5 + rng.random(n))
    return xyz, vel, dvol


@pytest.mark.parametrize("delta", ["roma3", "peskin4"])
@pytest.mark.parametrize("kind", ["periodic", "open"])
def test_ibm_cell_list_bit_exact_and_interp_spread_elementwise(fs, kind, delta):
    n = 700
    if kind == "periodic":
        cfg = _cfg_periodic(24, 20, 16, delta=delta, max_markers=n)
        cfg["markers"] = _markers(cfg, n, 9, spread_cells=14.0)       # supports wrap around the box
    else:
        cfg = _cfg_open(40, 30, 28, delta=delta, max_markers=n)
        cfg["markers"] = _markers(cfg, n, 9, spread_cells=8.0)
    cfg["init"] = _rand_fields(cfg, 4)
    o = _oracle(cfg)
    g = fs.from_workload(cfg)
    a, b = g.cell_list(), o.cell_list()
    assert a["nseg"] == b["nseg"]
    for k in ("base", "perm", "keys", "seg_start"):
        assert np.array_equal(a[k], b[k]), k
    U_ref = o.interpolate(*[cfg["init"][c] for c in "uvw"])
    U = g.ibm_interpolate()
    assert relerr(U, U_ref) < 1e-13
    F = np.random.default_rng(8).standard_normal((n, 3))
    f_ref = o.spread(F)
    g.ibm_spread(F)
    for c, fr in zip("uvw", f_ref):
        got = g.get(c) - cfg["init"][c]
        assert np.abs(got - fr).max() <= 1e-12 * np.abs(fr).max(), c
        assert np.array_equal(got != 0.0, fr != 0.0) or np.abs(got[fr == 0.0]).max() < 1e-13
    g.close()


def test_ibm_empty_and_single_marker(fs):
    cfg = _cfg_periodic(16, 16, 16, max_markers=4)
    g = fs.Grid(cfg)
    g.set_markers(np.zeros((0, 3)))
    assert g.cell_list()["nseg"] == 0
    xyz = np.array([[1.0, 2.0, 3.0]])
    g.set_markers(xyz)
    from oracle import Oracle
    o = Oracle(cfg); o.set_markers(xyz)
    a, b = g.cell_list(), o.cell_list()
    for k in ("base", "perm", "keys", "seg_start"):
        assert np.array_equal(a[k], b[k]), k
    with pytest.raises(fs.FsError):
        g.set_markers(np.zeros((5, 3)))          # > max_markers
    g.close()


# ------------------------------------------------------------------------------------ NEXT-2: strong coupling (Algorithm 1)
def test_strong_coupling_matches_oracle(fs):
    # a light 2-DOF body (added mass matters): same sweeps, same xi, same fields as the oracle's Algorithm 1; N = 1 is the
    # weak scheme; mask-forced body with strong coupling too (the solid velocity seen by the fluid is the latest iterate)
    def light(**kw):
        cfg = W.cylinder_fsi(scale=8, per_ring=16, rtol=1e-10, **kw)
        m, c, k, dof = cfg["body"]
        cfg["body"] = (0.25 * m, 0.05, k, 3)
        return cfg
    for kw in (dict(coupling_max_iters=30, coupling_tol=1e-12), dict(coupling_max_iters=3, coupling_tol=0.0),
               dict(coupling_max_iters=30, coupling_tol=1e-10, time_scheme="rk3")):
        cfg = light(**kw)
        o = _oracle(cfg); g = fs.from_workload(cfg)
        for x in (o, g):
            x.set_body_state([0.02, 0.01, 0.0], [0.0, 0.0, 0.0])
        for s_ in range(2):
            io = o.step(1); ig = g.step(1)
            assert ig["coupling_iters"] == io["coupling_iters"] >= 3, (ig["coupling_iters"], io["coupling_iters"])
            assert abs(ig["pcg_iters"] - io["pcg_iters"]) <= 3 * io["coupling_iters"]
            assert abs(ig["coupling_xi"] - io["coupling_xi"]) <= 1e-6 * io["coupling_xi"] + 1e-30
        _compare_state(g, o, TOL64)
        for k_ in ("body_force", "body_disp", "body_vel"):
            np.testing.assert_allclose(ig[k_], io[k_], rtol=1e-9, atol=1e-13)
        assert relerr(g.get("marker_x"), o.markers()[0]) < 1e-14 and ig["step"] == 2 and abs(ig["time"] - io["time"]) < 1e-15
        g.close()
    # weak == coupling_max_iters 1, bitwise on the GPU
    g1 = fs.from_workload(light()); g2 = fs.from_workload(light(coupling_max_iters=1))
    g1.step(3); i2 = g2.step(3)
    assert i2["coupling_iters"] == 1
    for c in "uvwp":
        assert np.array_equal(g1.get(c), g2.get(c))
    g1.close(); g2.close()


# ------------------------------------------------------------------------------------ NEXT-2: flexible beam (Eq. 13-17, Newmark-beta)
def test_flexible_beam_matches_oracle(fs):
    # a clamped flexible plate in a cross flow (the shape of PAPER.md section 3.3.1): beam matrices / frequencies of the host
    # setup (Cholesky + Jacobi rotations) against the oracle's (inverse iteration), then weak coupling over 10 steps and
    # strong coupling (Algorithm 1) over 3: state, load vector, markers, fields, sweeps
    for kw, steps in ((dict(), 10), (dict(coupling_max_iters=25, coupling_tol=1e-12), 3), (dict(coupling_max_iters=4, coupling_tol=0.0, zeta=0.0), 2)):
        cfg = W.flexible_plate(scale=8, nodes=9, rtol=1e-10, **kw)
        o = _oracle(cfg); g = fs.from_workload(cfg)
        co = o.beam_matrices()[3]; sg = g.beam_state()
        for k_ in ("alpha", "beta", "omega1", "omega2"):
            assert abs(sg[k_] - co[k_]) <= 1e-10 * abs(co[k_]), (k_, sg[k_], co[k_])
        for s_ in range(steps):
            io = o.step(1); ig = g.step(1)
            assert ig["coupling_iters"] == io["coupling_iters"], (ig["coupling_iters"], io["coupling_iters"])
            if kw:
                assert io["coupling_iters"] >= 3 and abs(ig["coupling_xi"] - io["coupling_xi"]) <= 1e-5 * io["coupling_xi"] + 1e-28
        _compare_state(g, o, TOL64, fields="uvp")
        # span-uniform flow: w is PCG-residual noise (1e-12) on both sides, compared on the scale of the velocity field (|u| ~ 1)
        assert np.abs(g.get("w") - o.get("w")).max() < TOL64 * np.abs(o.get("u")).max()
        so, sg = o.beam_state(), g.beam_state()
        assert np.abs(so["w"]).max() > 1e-6                                   # the plate did bend
        for k_ in ("w", "v", "a", "Q"):
            assert relerr(sg[k_], so[k_]) < 1e-8, (kw, k_, relerr(sg[k_], so[k_]))
        xo, uo, fo = o.markers()
        assert relerr(g.get("marker_x"), xo) < 1e-14 and relerr(g.get("marker_u"), uo) < 1e-8 and relerr(g.get("marker_f"), fo) < 1e-8
        for k_ in ("body_force",):
            np.testing.assert_allclose(ig[k_], io[k_], rtol=1e-9, atol=1e-13)
        assert "beam_newmark" in g.kernels_used()
        g.close()
    # ABI: a beam needs workspace, markers, and excludes the rigid body
    cfg = W.flexible_plate(scale=8, nodes=9)
    g = fs.Grid(dict(cfg, max_beam_nodes=4))
    for c_, a_ in cfg["init"].items():
        g.set(c_, a_)
    with pytest.raises(fs.FsError):
        g.set_beam(*cfg["beam"])                                              # no markers yet
    g.set_markers(*cfg["markers"])
    with pytest.raises(fs.FsError):
        g.set_beam(*cfg["beam"])                                              # 9 nodes > max_beam_nodes 4
    g.close()


# ------------------------------------------------------------------------------------ NEXT-4: LES closures
@pytest.mark.parametrize("kind", ["periodic", "channel", "open", "channel_upwind_wallonly"])
def test_les_momentum_rhs_elementwise(fs, kind):
    # Smagorinsky nu_t + flux-form diffusion (+ the Spalding wall model on the no-slip y walls of the channel), random
    # fields, ragged tiles; H^n element-wise against the oracle
    cfg = {"periodic": _cfg_periodic(72, 38, 21, cs=0.17), "channel": _cfg_channel(40, 50, 19, cs=0.12, wall_model=1),
           "open": _cfg_open(70, 27, 22, inflow_noise=0.05, seed=3, cs=0.2, wall_model=1),
           "channel_upwind_wallonly": _cfg_channel(36, 30, 17, cs=0.0, wall_model=1, convection="upwind")}[kind]
    if kind.startswith("channel"):
        cfg["nu"] = 1.0 / 3000.0
    cfg["init"] = _rand_fields(cfg, 13)
    ref = _oracle(cfg).momentum_rhs()
    g = fs.from_workload(cfg)
    got = g.momentum_rhs()
    for c, a, b in zip("uvw", got, ref):
        assert relerr(a, b) < 1e-12, (kind, c, relerr(a, b))
    used = g.kernels_used()
    assert any("LES" in k for k in used), used
    g.close()


def test_wmles_channel_64_runs_and_matches_oracle(fs):
    # the paper's WMLES workload shape (Table 5: 2 pi x 2 x pi, 64^3), Re_tau-2000-like viscosity, Smagorinsky + wall model
    # (initial field: the c2 recipe's Poiseuille profile + noise for nu = 1/180, then run at the lower viscosity)
    def wm(n, **kw):
        c = W.channel(n=n, cs=0.1, wall_model=1, **kw)
        c["nu"] = 1.0 / 2000.0
        return c
    cfg = wm(64, beta=1e-6, steps=4)
    g, o, ig, io, _ = _run_pair(fs, cfg, 4)
    assert ig["max_abs_div"] < 1e-5
    g.close()
    cfg = wm(24, time_scheme="rk3", cfl=0.3, dt=1e-3)
    g, o, ig, io, _ = _run_pair(fs, cfg, 3, iters_pm=3)            # with Runge-Kutta stages and the CFL step on top
    assert abs(ig["dt"] - io["dt"]) < 1e-13 * io["dt"]
    g.close()
    o5 = _oracle(wm(24)); o5.step(5)
    g = fs.from_workload(wm(24), dtype="f32"); g.step(5)
    errs = {c: relerr(g.get(c), o5.get(c)) for c in "uvwp"}
    assert all(e < TOL32 for e in errs.values()), errs
    g.close()


# ------------------------------------------------------------------------------------ NEXT-3: Runge-Kutta, CFL-adaptive dt
def test_rk3_matches_oracle_and_the_stability_polynomial(fs):
    cfg = W.taylor_green(n=16, nu=0.1, dt=0.05, time_scheme="rk3", rtol=1e-13)
    g, o, ig, io, _ = _run_pair(fs, cfg, 5, iters_pm=3)           # iterations are summed over the three stage solves
    h = 2 * math.pi / 16
    z = -0.1 * (8.0 / h ** 2 * math.sin(h / 2) ** 2) * 0.05
    assert abs(np.abs(g.get("u")).max() / np.abs(cfg["init"]["u"]).max() - (1 + z + z * z / 2 + z ** 3 / 6) ** 5) < 1e-12
    assert abs(ig["time"] - 0.25) < 1e-15 and ig["dt"] == 0.05
    g.close()
    # nonlinear cases: GMG-PCG HIT box (fused V-cycle path, three WHILE nodes per graph) and the walled channel
    for cfg, steps in ((W.hit(n=32, time_scheme="rk3"), 3), (W.channel(n=24, time_scheme="rk3"), 3),
                       (W.cylinder_fsi(scale=8, per_ring=12, time_scheme="rk3"), 3)):
        g, o, ig, io, _ = _run_pair(fs, cfg, steps, iters_pm=3)
        np.testing.assert_allclose(ig["body_disp"], io["body_disp"], rtol=1e-9, atol=1e-15)
        np.testing.assert_allclose(ig["body_force"], io["body_force"], rtol=1e-9, atol=1e-12)
        assert "rk_combine" in g.kernels_used()
        g.close()
    # graph replay == direct launches, bit for bit; fp32 within 1e-4 of the oracle
    cfg = W.hit(n=32, time_scheme="rk3")
    g1 = fs.from_workload(cfg, exec_mode="graph"); g2 = fs.from_workload(cfg, exec_mode="stream")
    i1 = g1.step(2, per_step=True); i2 = g2.step(2, per_step=True)
    assert i1["iters_per_step"] == i2["iters_per_step"]
    for c in "uvwp":
        assert np.array_equal(g1.get(c), g2.get(c)), c
    g1.close(); g2.close()
    o = _oracle(cfg); o.step(3)
    g = fs.from_workload(cfg, dtype="f32"); g.step(3)
    errs = {c: relerr(g.get(c), o.get(c)) for c in "uvwp"}
    assert all(e < TOL32 for e in errs.values()), errs
    g.close()


@pytest.mark.parametrize("scheme", ["ab2", "euler", "rk3"])
def test_cfl_adaptive_dt_matches_oracle(fs, scheme):
    # the step size is chosen on the device from max|u| of the current field; same sequence of dt as the oracle
    for cfg in (W.channel(n=24, cfl=0.35, dt=1e-3, time_scheme=scheme), W.cylinder_fsi(scale=8, per_ring=12, cfl=0.2, dt=2e-2, time_scheme=scheme)):
        o = _oracle(cfg)
        g = fs.from_workload(cfg)
        dts = []
        for s_ in range(5):
            io = o.step(1); ig = g.step(1)
            assert abs(ig["dt"] - io["dt"]) <= 1e-13 * io["dt"], (s_, ig["dt"], io["dt"])
            assert abs(ig["pcg_iters"] - io["pcg_iters"]) <= (3 if scheme == "rk3" else 1)
            dts.append(io["dt"])
        assert abs(ig["time"] - io["time"]) < 1e-12 * io["time"]
        assert max(dts) < cfg["dt"] and len(set(dts)) > 1            # the CFL limit is active and moves
        _compare_state(g, o, TOL64)
        assert "dt_cfl" in g.kernels_used()
        g.close()


# ------------------------------------------------------------------------------------ NEXT-1: the paper's eps-mask IBM
def _sphere_mask(cfg, centre, radius):
    c = W.coords(cfg)
    d2 = ((c["xc"][None, None, :] - centre[0]) ** 2 + (c["yc"][None, :, None] - centre[1]) ** 2 + (c["zc"][:, None, None] - centre[2]) ** 2)
    return (d2 < radius ** 2).astype(np.uint8)


@pytest.mark.parametrize("kind", ["periodic", "open"])
def test_mask_face_classes_bit_exact(fs, kind):
    cfg = _cfg_periodic(26, 19, 14, solid_mask=1) if kind == "periodic" else _cfg_open(30, 21, 17, solid_mask=1)
    rng = np.random.default_rng(41)
    eps = (rng.random(W.shapes(cfg)["p"]) < 0.2).astype(np.uint8)
    eps[:, :3, :4] = 1; eps[-2:, :, -3:] = 1                       # solid cells on the box faces / across the periodic seam
    from oracle import Oracle
    o = Oracle(cfg); o.set_solid_mask(eps)
    g = fs.Grid(cfg); g.set_solid_mask(eps)
    for name, ref in zip(("mask_u", "mask_v", "mask_w"), o.face_masks()):
        assert np.array_equal(g.get(name), ref), name
    g.close()
    g = fs.Grid(dict(cfg, solid_mask=0))
    with pytest.raises(fs.FsError) as e:
        g.set_solid_mask(eps)                                      # workspace was not reserved
    assert e.value.status == 2
    g.close()


@pytest.mark.parametrize("delta", ["roma3", "peskin4"])
def test_mask_ibm_full_steps_match_oracle(fs, delta):
    # sphere-shaped solid in the c3-shaped open box; the markers on its surface carry a rigid rotation to the IB points
    # (Eq. 18-19), the solid itself translates with u_c (Eq. 23); 6 steps, fields 1e-9, forces, face classes bit-exact
    cfg = W.sphere(scale=4, n_markers=400, delta=delta, solid_mask=1)
    X = cfg["markers"][0]
    ctr = np.array([cfg["lx"] / 4.0, cfg["ly"] / 2.0, cfg["lz"] / 2.0])
    vel = np.cross(np.array([0.0, 0.0, 0.8]), X - ctr)
    cfg["markers"] = (X, vel, cfg["markers"][2])
    cfg["mask"] = (_sphere_mask(cfg, ctr, 0.5), [0.05, -0.02, 0.0])
    o = _oracle(cfg); o.set_solid_mask(*cfg["mask"])
    g = fs.from_workload(cfg)
    for name, ref in zip(("mask_u", "mask_v", "mask_w"), o.face_masks()):
        assert np.array_equal(g.get(name), ref), name
    io = o.step(6); ig = g.step(6, per_step=True)
    assert ig["converged"] == 1 and all(abs(a - b) <= 1 for a, b in zip(ig["iters_per_step"], io["iters_per_step"]))
    _compare_state(g, o, TOL64)
    np.testing.assert_allclose(ig["body_force"], io["body_force"], rtol=1e-9, atol=1e-12)
    assert relerr(g.get("marker_f"), o.markers()[2]) < 1e-12        # wdot_i / F_Ni of Eq. 18-19
    used = g.kernels_used()
    assert "mask_forcing" in used and "mask_ib_points" in used and "ibm_spread" in used and "ibm_interpolate" not in used, used
    g.close()


def test_mask_ibm_without_markers_rigid_body_and_fp32(fs):
    # mask only (IB points not forced), the solid moving with a 2-DOF rigid body (u_c = body velocity); fp64 1e-9, fp32 1e-4
    cfg = W.cylinder_fsi(scale=8, per_ring=12, solid_mask=1)
    cfg["markers"] = None; cfg["max_markers"] = 0
    m, _, k, _ = cfg["body"]
    cfg["body"] = (m, 0.1, k, 3)
    c = W.coords(cfg)
    eps = (((c["xc"][None, None, :] - cfg["lx"] / 3.0) ** 2 + (c["yc"][None, :, None] - cfg["ly"] / 2.0) ** 2) < 0.25).astype(np.uint8)
    eps = np.broadcast_to(eps, W.shapes(cfg)["p"]).copy()
    cfg["mask"] = (eps, None)
    o = _oracle(cfg); o.set_solid_mask(eps)
    g = fs.from_workload(cfg)
    io = o.step(8); ig = g.step(8, per_step=True)
    assert all(abs(a - b) <= 1 for a, b in zip(ig["iters_per_step"], io["iters_per_step"]))
    _compare_state(g, o, TOL64)
    for k_ in ("body_force", "body_disp", "body_vel"):
        np.testing.assert_allclose(ig[k_], io[k_], rtol=1e-9, atol=1e-13)
    assert abs(io["body_vel"][0]) > 0 and abs(io["body_force"][0]) > 0
    g.close()
    o5 = _oracle(cfg); o5.set_solid_mask(eps); o5.step(5)
    g = fs.from_workload(cfg, dtype="f32")
    g.step(5)
    errs = {c_: relerr(g.get(c_), o5.get(c_)) for c_ in "uvwp"}
    assert all(e < TOL32 for e in errs.values()), errs
    g.close()


# ------------------------------------------------------------------------------------ fp32 across the variants of the step
@pytest.mark.parametrize("variant", ["rk3", "adaptive_upwind", "les_channel", "strong_body", "beam_strong", "gmg_rk3"])
def test_fp32_variants_within_1e4_of_the_fp64_oracle(fs, variant):
    # north_star: fp32 fields within 1e-4 of the fp64 oracle over 5 steps -- for every variant of the step, not only the plain
    # AB2 path (k_momentumv<f32>, the LES variant of k_momentum<f32>, k_pcg_coop<f32>, the GMG kernels in fp32, Newmark / RK4 in
    # fp64 next to fp32 fields); structure state within 1e-4 too
    if variant == "rk3":
        cfg = _cfg_periodic(64, 40, 32, time_scheme="rk3", rtol=1e-8); cfg["init"] = {c_: 0.3 * a for c_, a in _rand_fields(cfg, 31).items()}
    elif variant == "adaptive_upwind":
        cfg = _cfg_channel(64, 34, 24, convection="upwind", cfl=0.25, rtol=1e-8); cfg["init"] = {c_: 0.5 * a for c_, a in _rand_fields(cfg, 32).items()}
    elif variant == "les_channel":
        cfg = _cfg_channel(48, 32, 24, cs=0.1, wall_model=1, rtol=1e-8); cfg["init"] = {c_: 0.5 * a for c_, a in _rand_fields(cfg, 33).items()}
    elif variant == "strong_body":
        cfg = W.cylinder_fsi(scale=8, per_ring=16, rtol=1e-8, coupling_max_iters=6, coupling_tol=1e-6)
        m, c_, k_, dof = cfg["body"]; cfg["body"] = (0.5 * m, 0.05, k_, 3)
    elif variant == "beam_strong":
        cfg = W.flexible_plate(scale=8, nodes=9, rtol=1e-8, coupling_max_iters=6, coupling_tol=1e-6)
    else:
        h = 2 * math.pi / 64
        cfg = _cfg_periodic(64, 32, 48, precond="gmg", time_scheme="rk3", rtol=1e-7, max_iter=100); cfg.update(lx=64 * h, ly=32 * h, lz=48 * h)
        cfg["init"] = {c_: 0.3 * a for c_, a in _rand_fields(cfg, 34).items()}
    o = _oracle(cfg)
    io = o.step(5)
    g = fs.from_workload(dict(cfg, dtype="f32"))
    ig = g.step(5)
    assert ig["nan_flag"] == 0 and ig["converged"] == 1 and ig["unconverged_steps"] == 0, ig
    scale = max(np.abs(o.get(c_)).max() for c_ in "uvw")
    for c_ in "uvw":
        assert np.abs(g.get(c_) - o.get(c_)).max() < TOL32 * scale, (variant, c_, np.abs(g.get(c_) - o.get(c_)).max() / scale)
    assert relerr(g.get("p"), o.get("p")) < 10 * TOL32, (variant, relerr(g.get("p"), o.get("p")))   # p = (rho / dt) x a velocity difference: one digit less
    assert abs(ig["dt"] - io["dt"]) <= 1e-5 * io["dt"] and abs(ig["time"] - io["time"]) <= 1e-5 * io["time"]
    if variant == "strong_body":
        np.testing.assert_allclose(ig["body_disp"], io["body_disp"], rtol=2e-3, atol=1e-9)
    if variant == "beam_strong":
        assert relerr(g.beam_state()["w"], o.beam_state()["w"]) < 2e-3
    used = g.kernels_used()
    want = {"rk3": "k_momentumv<f32,central>", "adaptive_upwind": "k_momentumv<f32,upwind>", "les_channel": "k_momentum<f32,central,LES>",
            "strong_body": "k_pcg_coop<f32>", "beam_strong": "beam_newmark", "gmg_rk3": "k_mg_up<f32,TR8,DOT>"}[variant]
    assert want in used, (variant, used)
    g.close()


# ------------------------------------------------------------------------------------ full steps
def _compare_state(g, o, tol, fields="uvwp"):
    errs = {}
    for c in fields:
        errs[c] = relerr(g.get(c), o.get(c))
    # w of 2-D flows is identically zero in the oracle: relerr is then absolute
    bad = {c: e for c, e in errs.items() if not e < tol}
    assert not bad, errs
    return errs


def _run_pair(fs, cfg, steps, tol=TOL64, iters_pm=1):
    o = _oracle(cfg)
    g = fs.from_workload(cfg)
    io = o.step(steps)
    ig = g.step(steps, per_step=True)
    assert ig["nan_flag"] == 0 and ig["converged"] == 1
    for a, b in zip(ig["iters_per_step"], io["iters_per_step"]):
        assert abs(a - b) <= iters_pm, (ig["iters_per_step"], io["iters_per_step"])
    errs = _compare_state(g, o, tol)
    assert ig["step"] == io["step"] == steps
    return g, o, ig, io, errs


def test_c1_taylor_green_10_steps(fs):
    cfg = W.taylor_green()
    g, o, ig, io, _ = _run_pair(fs, cfg, 10)
    assert ig["max_abs_div"] < 1e-12
    # the same closed form that pins the oracle (tests/golden/taylor_green_pins.txt, AB2 a10)
    assert abs(np.abs(g.get("u")).max() / np.abs(cfg["init"]["u"]).max() - 0.9998006613990811) < 1e-11
    g.close()


def test_c2_channel_reduced_20_steps(fs):
    cfg = W.channel(n=48)
    g, o, ig, io, _ = _run_pair(fs, cfg, 20)
    g.close()


def test_c3_sphere_reduced_20_steps(fs):
    cfg = W.sphere(scale=4, n_markers=400)
    g, o, ig, io, _ = _run_pair(fs, cfg, 20)
    np.testing.assert_allclose(ig["body_force"], io["body_force"], rtol=1e-9, atol=1e-12)
    a, b = g.cell_list(), o.cell_list()
    for k in ("base", "perm", "keys", "seg_start"):
        assert np.array_equal(a[k], b[k]), k
    assert relerr(g.get("marker_f"), o.markers()[2]) < 1e-9
    g.close()


def test_c4_cylinder_fsi_reduced_50_steps(fs):
    cfg = W.cylinder_fsi(scale=4, per_ring=40)
    g, o, ig, io, _ = _run_pair(fs, cfg, 50)
    np.testing.assert_allclose(ig["body_disp"], io["body_disp"], rtol=1e-9, atol=1e-15)
    np.testing.assert_allclose(ig["body_vel"], io["body_vel"], rtol=1e-9, atol=1e-15)
    np.testing.assert_allclose(ig["body_force"], io["body_force"], rtol=1e-9, atol=1e-12)
    # the moving body's cell list is rebuilt every step: still bit-exact at the end
    o.step(0)
    a, b = g.cell_list(), o.cell_list()
    assert relerr(g.get("marker_x"), o.markers()[0]) < 1e-14
    g.close()


def test_two_dof_rigid_body_fsi_reduced(fs):
    # SURVEY 8(f) NEXT-2, first item: the 2-DOF (in-line + transverse) oscillator of Eq. 12,
    # with damping, weak coupling; the body moves in x and y and its cell list is rebuilt every step
    cfg = W.cylinder_fsi(scale=4, per_ring=40)
    m, _, k, _ = cfg["body"]
    cfg["body"] = (m, 0.3, k, 3)
    g, o, ig, io, _ = _run_pair(fs, cfg, 30)
    assert abs(io["body_disp"][0]) > 0 and abs(io["body_disp"][1]) > 0 and io["body_disp"][2] == 0
    np.testing.assert_allclose(ig["body_disp"], io["body_disp"], rtol=1e-9, atol=1e-15)
    np.testing.assert_allclose(ig["body_vel"], io["body_vel"], rtol=1e-9, atol=1e-15)
    np.testing.assert_allclose(ig["body_force"], io["body_force"], rtol=1e-9, atol=1e-12)
    assert relerr(g.get("marker_x"), o.markers()[0]) < 1e-14
    g.close()


def test_c5_hit_64_fp64_10_steps(fs):
    cfg = W.hit(n=64)
    g, o, ig, io, _ = _run_pair(fs, cfg, 10)
    g.close()


def test_c5_hit_64_fp32_5_steps(fs):
    cfg = W.hit(n=64)
    o = _oracle(cfg)
    io = o.step(5)
    g = fs.from_workload(cfg, dtype="f32")
    ig = g.step(5, per_step=True)
    assert ig["nan_flag"] == 0 and ig["converged"] == 1 and ig["unconverged_steps"] == 0, ig
    assert all(abs(a - b) <= 1 for a, b in zip(ig["iters_per_step"], io["iters_per_step"])), (ig["iters_per_step"], io["iters_per_step"])
    errs = {c: relerr(g.get(c), o.get(c)) for c in "uvwp"}
    assert all(e < TOL32 for e in errs.values()), errs
    g.close()


def test_tr16_instantiation_vcycle_and_full_steps_on_64x384x64(fs):
    # ny >= 384 selects the 32-row tiles (TR = 16) of the fused V-cycle legs -- the instantiation bench.py times at
    # 512^3 -- on a box the oracle steps in seconds: V-cycle element-wise, 10 fp64 steps (1e-9, iterations +-1) and
    # 5 fp32 steps (1e-4); each part asserts that it ran the instantiation it is meant for.
    cfg = W.hit_box(64, 384, 64)
    r = np.random.default_rng(6).standard_normal(W.shapes(cfg)["p"])
    o = _oracle(cfg)
    z_ref = o.vcycle(r)
    g = fs.from_workload(cfg)
    z = g.gmg_vcycle(r)
    assert relerr(z, z_ref) < 1e-12, relerr(z, z_ref)
    used = g.kernels_used()
    assert "k_mg_down<f64,TR16>" in used and "k_mg_up<f64,TR16>" in used, used
    io5 = o.step(5)
    ref5 = {c: o.get(c) for c in "uvwp"}
    io10 = o.step(5)
    ig = g.step(10, per_step=True)
    assert ig["nan_flag"] == 0 and ig["converged"] == 1
    want = io5["iters_per_step"] + io10["iters_per_step"]
    assert all(abs(a - b) <= 1 for a, b in zip(ig["iters_per_step"], want)), (ig["iters_per_step"], want)
    _compare_state(g, o, TOL64)
    used = g.kernels_used()
    for k in ("k_mg_down<f64,TR16,UPD>", "k_mg_up<f64,TR16,DOT>", "k_pcg_dirapply2<f64>", "k_projectv<f64>", "k_div_rhsv<f64>", "k_pcg_initv<f64>"):
        assert k in used, (k, used)
    g.close()
    g = fs.from_workload(cfg, dtype="f32")
    i32 = g.step(5, per_step=True)
    assert i32["nan_flag"] == 0 and i32["converged"] == 1
    assert all(abs(a - b) <= 1 for a, b in zip(i32["iters_per_step"], io5["iters_per_step"])), (i32["iters_per_step"], io5["iters_per_step"])
    errs = {c: relerr(g.get(c), ref5[c]) for c in "uvwp"}
    assert all(e < TOL32 for e in errs.values()), errs
    used = g.kernels_used()
    assert "k_mg_down<f32,TR16,UPD>" in used and "k_mg_up<f32,TR16,DOT>" in used and "k_pcg_dirapplyv<f32>" in used, used
    g.close()


def test_graph_and_stream_modes_agree_bitwise(fs):
    cfg = W.sphere(scale=4, n_markers=300)
    g1 = fs.from_workload(cfg, exec_mode="graph")
    g2 = fs.from_workload(cfg, exec_mode="stream")
    i1 = g1.step(5, per_step=True); i2 = g2.step(5, per_step=True)
    assert i1["iters_per_step"] == i2["iters_per_step"]
    for c in "uvwp":
        assert np.array_equal(g1.get(c), g2.get(c)), c
    g1.close(); g2.close()


def test_p16_restart_is_bit_exact(fs):
    cfg = W.cylinder_fsi(scale=4, per_ring=40)
    g = fs.from_workload(cfg)
    g.step(10)
    ref = {c: g.get(c) for c in "uvwp"}
    ref_body = g.body_state()
    a = fs.from_workload(cfg)
    a.step(5)
    state = {c: a.get(c) for c in ("u", "v", "w", "p", "hu", "hv", "hw")}
    mx, mu = a.get("marker_x"), a.get("marker_u")
    disp, vel, _ = a.body_state()
    b = fs.Grid(dict(cfg))
    for c, v in state.items():
        b.set(c, v)
    b.set_markers(mx, mu, cfg["markers"][2])
    b.set_body(*cfg["body"])
    b.set_body_state(disp, vel)
    b.set_history(1, 5)
    b.step(5)
    for c in "uvwp":
        assert np.array_equal(b.get(c), ref[c]), c
    assert np.array_equal(b.body_state()[0], ref_body[0])
    g.close(); a.close(); b.close()


def test_async_steps_equal_sync_steps(fs):
    cfg = W.taylor_green()
    g1 = fs.from_workload(cfg); g2 = fs.from_workload(cfg)
    g1.step(6)
    g2.step(3, sync=False); g2.step(3, sync=False)
    for c in "uvwp":
        assert np.array_equal(g1.get(c), g2.get(c))
    assert g1.launch_count() == g2.launch_count() > 0
    g1.close(); g2.close()


def test_device_pointer_io_and_dtype_conversion(fs):
    import torch
    cfg = W.taylor_green()
    g = fs.from_workload(cfg, dtype="f32")
    u64 = torch.from_numpy(cfg["init"]["u"]).cuda()
    g.set("u", u64)                                   # fp64 device -> fp32 grid
    out = torch.empty_like(u64)
    g.get("u", out=out)
    assert torch.allclose(out, u64, atol=1e-7)
    host32 = g.get("u", dtype="f32")
    assert host32.dtype == np.float32 and np.abs(host32 - cfg["init"]["u"]).max() < 1e-7
    g.close()


def test_async_field_io_on_two_streams_equals_the_synchronous_calls(fs):
    # fs_fields_set_async / fs_fields_get_async (pipelines over independent grids): two grids on two streams fed from
    # pinned host buffers give bit for bit what one grid fed through the synchronous calls gives
    import torch
    cfg = W.taylor_green(n=24)
    ref = fs.from_workload(cfg)
    ref.step(3)
    s2 = torch.cuda.Stream()
    grids = [fs.Grid(cfg), fs.Grid(cfg, stream=s2)]
    host = [{c: torch.from_numpy(np.ascontiguousarray(cfg["init"][c])).pin_memory() for c in "uvw"} for _ in grids]
    out = [{c: torch.empty(ref.shape[c], dtype=torch.float64).pin_memory() for c in "uvwp"} for _ in grids]
    for g_, h_, o_ in zip(grids, host, out):
        for c in "uvw":
            g_.set_async(c, h_[c])
        g_.step(3, sync=False)
        for c in "uvwp":
            g_.get_async(c, o_[c])
    torch.cuda.synchronize()
    for o_ in out:
        for c in "uvwp":
            assert np.array_equal(o_[c].numpy(), ref.get(c)), c
    with pytest.raises(fs.FsError):
        grids[0].set_async("marker_x", host[0]["u"])
    for g_ in grids + [ref]:
        g_.close()


def test_marker_support_touching_a_wall_is_unsupported(fs):
    # same rule, same threshold as the oracle (pin P22): 1.5 h (Roma) from a non-periodic boundary
    cfg = _cfg_open(40, 30, 28, max_markers=4)
    h = 1.0 / 16
    g = fs.Grid(cfg)
    mid = np.array([20 * h, 15 * h, 14 * h])
    ok = np.stack([mid, mid]); ok[0, 0] = 1.5 * h + 1e-9; ok[1, 1] = 30 * h - 1.5 * h - 1e-9
    g.set_markers(ok)
    assert g.cell_list()["perm"].size == 2
    for d, bad in ((0, 1.49 * h), (1, 30 * h - 1.49 * h), (2, 1.2 * h)):
        x = mid.copy(); x[d] = bad
        with pytest.raises(fs.FsError) as e:
            g.set_markers(x[None, :])
        assert e.value.status == fs.FS_ERR_UNSUPPORTED
        assert g.cell_list()["nseg"] == 0                         # refused: the grid keeps no markers
    g.close()
    # a moving body that carries its markers into the wall: reported by the synchronous fs_step, state info still filled
    cfg = W.cylinder_fsi(scale=8, per_ring=12, rtol=1e-8)
    g = fs.from_workload(cfg)
    g.set_body_state([0.0, 0.0, 0.0], [0.0, 400.0, 0.0])
    g.step(1)
    info = fs.fs_step_info()
    import ctypes as C
    st = fs.lib().fs_step(g.h, 1, C.byref(info))
    assert st == fs.FS_ERR_UNSUPPORTED and info.step == 2
    g.close()


def test_step_info_is_filled_when_pcg_does_not_converge_and_sticky_counters_count(fs):
    import ctypes as C
    cfg = W.channel(n=24, max_iter=3)
    g = fs.from_workload(cfg)
    info = fs.fs_step_info()
    st = fs.lib().fs_step(g.h, 2, C.byref(info))
    assert st == fs.FS_ERR_NOT_CONVERGED                           # fs.h: *last is valid for this status
    assert info.pcg_iters == 3 and info.converged == 0 and info.step == 2 and info.unconverged_steps == 2 and info.nan_steps == 0
    g.step(3, sync=False)                                           # asynchronous steps are counted too
    assert g.step(0)["unconverged_steps"] == 5
    g.close()
    g = fs.from_workload(W.taylor_green())
    assert g.step(4)["unconverged_steps"] == 0
    g.close()


def test_two_grids_in_one_process_and_device_guard(fs):
    # per-device kernel attributes are applied per grid (not once per process), and every entry point runs on the
    # grid's own device: two GMG grids stepped alternately, on two GPUs when the box has them
    import torch
    ndev = torch.cuda.device_count()
    cfgs = [W.hit(n=32), W.hit(n=32, seed=5)]
    devs = ["cuda:0", "cuda:%d" % (1 if ndev > 1 else 0)]
    gs = [fs.from_workload(c, device=d) for c, d in zip(cfgs, devs)]
    torch.cuda.set_device(0)
    for _ in range(2):
        for g in gs:
            assert g.step(1)["converged"] == 1
    assert torch.cuda.current_device() == 0                         # the caller's device is restored
    for g, c in zip(gs, cfgs):
        o = _oracle(c); o.step(2)
        _compare_state(g, o, TOL64)
        g.close()
    # a workspace that is not device memory is refused
    import ctypes as C
    P, keep = fs.make_params(cfgs[0])
    n = C.c_size_t(0)
    assert fs.lib().fs_workspace_bytes(C.byref(P), C.byref(n)) == 0
    host = np.zeros(n.value + 256, dtype=np.uint8)
    ptr = (host.ctypes.data + 255) & ~255
    h = C.c_void_p()
    assert fs.lib().fs_grid_create(C.byref(P), C.c_void_p(ptr), n.value, None, C.byref(h)) == 1


def test_launch_count_counts_every_loop_body_replay(fs):
    # graph mode, 32^3 GMG V(2,2): 9 fixed kernels per step (momentum, div_rhs, pcg_init, 4 x finish, project, step_end)
    # + 4 per loop-body replay (level-0 down leg, one-CTA tail for 16^3..4^3, level-0 up leg, direction+apply); the
    # fused residual update makes the body run once more than the solve iterates
    cfg = W.hit(n=32)
    g = fs.from_workload(cfg)
    prev = g.launch_count()
    for _ in range(4):
        info = g.step(1)
        n = g.launch_count()
        assert n - prev == 9 + 4 * (info["pcg_iters"] + 1), (n - prev, info["pcg_iters"])
        prev = n
    g.close()


def test_invalid_arguments(fs):
    cfg = W.taylor_green()
    bad = dict(cfg, nx=1)
    with pytest.raises(fs.FsError):
        fs.Grid(bad)
    bad = dict(cfg, precond="gmg", nz=30, lz=cfg["lz"])        # anisotropic spacing -> unsupported
    with pytest.raises(fs.FsError) as e:
        fs.Grid(bad)
    assert e.value.status == 6
    ch = W.channel(n=16); ch["max_markers"] = 4
    g = fs.Grid(ch)
    with pytest.raises(fs.FsError) as e:
        g.set_markers(np.array([[1.0, 0.0, 1.0]]))               # markers on a y-stretched grid
    assert e.value.status == 6
    g.close()
