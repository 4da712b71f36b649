"""Pins of the CPU oracle's fluid part against closed forms and identities (SURVEY.md 8(c) P1-P7,
P12, P13).  CPU only.  Each test is chosen so that a plausible slip in the oracle (dropped term,
wrong sign / index, transposed operand) fails it."""
import math
import os

import numpy as np
import pytest

import fs_workloads as W
from oracle import Oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _gold(fn):
    out = {}
    for line in open(os.path.join(GOLD, fn)):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            out[k] = float(v)
    return out


def _mk(cfg, fields=True):
    o = Oracle(cfg)
    if fields:
        for c in "uvw":
            o.set(c, cfg["init"][c])
    return o


def _periodic_cfg(nx, ny, nz, lx=2 * math.pi, ly=2 * math.pi, lz=2 * math.pi, **kw):
    return W._base(nx=nx, ny=ny, nz=nz, lx=lx, ly=ly, lz=lz, nu=0.01, dt=1e-3, **kw)


# ---------------------------------------------------------------- P1: Taylor-Green closed form
@pytest.mark.parametrize("scheme", ["euler", "ab2"])
def test_p1_taylor_green_amplitude_and_pressure(scheme):
    g = _gold("taylor_green_pins.txt")
    cfg = W.taylor_green(time_scheme=scheme)
    n, nu, dt = 32, cfg["nu"], cfg["dt"]
    h = 2 * math.pi / n
    kt2 = 8.0 / h ** 2 * math.sin(h / 2) ** 2
    assert abs(kt2 - g["ktilde2"]) < 1e-13
    # amplitude recursion written out here, independent of the oracle
    a = [1.0]
    for s in range(10):
        if scheme == "ab2" and s > 0:
            a.append(a[-1] - nu * dt * kt2 * (1.5 * a[-1] - 0.5 * a[-2]))
        else:
            a.append(a[-1] - nu * dt * kt2 * a[-1])
    assert abs(a[10] - g["a10_" + scheme]) < 1e-14
    o = _mk(cfg)
    info = o.step(10)
    c = W.coords(cfg)
    xf, xc, yf, yc = c["xf"][:-1], c["xc"], c["yf"][:-1], c["yc"]
    u_ref = a[10] * np.sin(xf)[None, None, :] * np.cos(yc)[None, :, None] * np.ones((n, 1, 1))
    v_ref = -a[10] * np.cos(xc)[None, None, :] * np.sin(yf)[None, :, None] * np.ones((n, 1, 1))
    assert np.abs(o.get("u") - u_ref).max() < 2e-12
    assert np.abs(o.get("v") - v_ref).max() < 2e-12
    assert np.abs(o.get("w")).max() < 1e-14
    # O(h^2) distance from the continuous decay, as the golden file states
    assert abs(a[10] - g["a10_continuous"]) < 1e-6
    # pressure of the last step: P * (a0 a_9^2 + a1 a_8^2) (cos 2x + cos 2y)
    P = math.cos(h / 2) ** 2 * (math.sin(h) / h) ** 2 / (4 / h ** 2 * math.sin(h) ** 2)
    assert abs(P - g["P_pressure_factor"]) < 1e-14
    amp2 = a[9] ** 2 if scheme == "euler" else 1.5 * a[9] ** 2 - 0.5 * a[8] ** 2
    p_ref = P * amp2 * (np.cos(2 * xc)[None, None, :] + np.cos(2 * yc)[None, :, None]) * np.ones((n, 1, 1))
    assert np.abs(o.get("p") - p_ref).max() < 1e-9
    assert info["max_abs_div"] < 1e-12            # P7
    assert info["converged"] == 1


def test_p2_pcg_single_mode_converges_in_one_iteration():
    # b holds only cos 2x, cos 2y which share one eigenvalue => 1 iteration (rtol above rounding noise)
    cfg = W.taylor_green(rtol=1e-9, warm_start=0)
    o = _mk(cfg)
    info = o.step(2)          # (later steps inherit the previous solve's residual as div u^n)
    assert info["iters_per_step"] == [1, 1]


# ---------------------------------------------------------------- P3: Laplacian eigenvalues
@pytest.mark.parametrize("mode", [(1, 0, 0), (0, 2, 0), (0, 0, 3), (2, 3, 1), (5, 1, 4)])
def test_p3_laplacian_fourier_eigenvalues(mode):
    nx, ny, nz = 16, 12, 10
    lx, ly, lz = 2 * math.pi, 3.0, 1.7
    o = Oracle(_periodic_cfg(nx, ny, nz, lx, ly, lz))
    i, j, k = np.arange(nx), np.arange(ny), np.arange(nz)
    ph = (2 * math.pi * mode[0] * i / nx)[None, None, :] + (2 * math.pi * mode[1] * j / ny)[None, :, None] \
        + (2 * math.pi * mode[2] * k / nz)[:, None, None]
    lam = 0.0
    for m, n, l in zip(mode, (nx, ny, nz), (lx, ly, lz)):
        h = l / n
        lam -= 4.0 / h ** 2 * math.sin(math.pi * m / n) ** 2
    for f in (np.cos(ph), np.sin(ph + 0.3)):
        out = o.laplacian(f)
        assert np.abs(out - lam * f).max() <= 1e-13 * abs(lam) + 1e-13


# ---------------------------------------------------------------- P4: manufactured Poisson, 2nd order
def test_p4_manufactured_poisson_second_order():
    errs = []
    for n in (16, 32, 64):
        cfg = _periodic_cfg(n, n, n, rtol=1e-11, warm_start=0)
        o = Oracle(cfg)
        c = W.coords(cfg)
        X, Y, Z = c["xc"][None, None, :], c["yc"][None, :, None], c["zc"][:, None, None]
        p_exact = np.cos(X) * np.cos(2 * Y) * np.cos(3 * Z)
        rhs = -14.0 * p_exact
        p, info = o.poisson_solve(rhs)
        assert info["converged"] == 1
        errs.append(np.abs(p - p_exact).max())
    assert 3.7 < errs[0] / errs[1] < 4.3 and 3.8 < errs[1] / errs[2] < 4.2


# ---------------------------------------------------------------- P5: dense direct solve on tiny grids
def _dense_A(o, shape):
    N = int(np.prod(shape))
    A = np.zeros((N, N))
    for q in range(N):
        e = np.zeros(N); e[q] = 1.0
        A[:, q] = o.apply_A(e.reshape(shape)).ravel()
    return A


def _wall_cfg(nx, ny, nz, stretched, **kw):
    yf = None
    if stretched:
        j = np.arange(ny + 1)
        yf = np.tanh(1.5 * (2.0 * j / ny - 1.0)) / math.tanh(1.5)
    cfg = W._base(nx=nx, ny=ny, nz=nz, lx=2.0, ly=2.0, lz=1.5, y0=-1.0, yf=yf, nu=0.05, dt=1e-3, **kw)
    cfg["bc"] = ["periodic", "periodic", "noslip", "noslip", "periodic", "periodic"]
    return cfg


@pytest.mark.parametrize("kind", ["periodic_none", "periodic_jacobi", "periodic_gmg", "walls_stretched", "box_neumann"])
def test_p5_pcg_matches_dense_direct_solve(kind):
    rng = np.random.default_rng(5)
    if kind.startswith("periodic"):
        pc = kind.split("_")[1]
        n = 8
        cfg = _periodic_cfg(n, n, n, precond=pc, rtol=1e-13, warm_start=0, max_iter=500)
    elif kind == "walls_stretched":
        cfg = _wall_cfg(6, 8, 5, True, rtol=1e-13, warm_start=0)
    else:
        cfg = W._base(nx=6, ny=5, nz=7, lx=1.0, ly=1.2, lz=0.9, nu=0.01, dt=1e-3, rtol=1e-13, warm_start=0)
        cfg["bc"] = ["inflow", "outflow", "slip", "slip", "noslip", "noslip"]
    o = Oracle(cfg)
    shape = o.shape["p"]
    A = _dense_A(o, shape)
    assert np.abs(A - A.T).max() < 1e-12 * np.abs(A).max()            # P6 symmetric
    assert np.abs(A @ np.ones(A.shape[0])).max() < 1e-11 * np.abs(A).max()  # P6 A.1 = 0
    w = np.linalg.eigvalsh(A)
    assert w[0] > -1e-10 * w[-1] and w[1] > 1e-8 * w[-1]              # PSD, 1-dim null space
    rhs = rng.standard_normal(shape)
    p, info = o.poisson_solve(rhs)
    assert info["converged"] == 1
    # reference: solve L p = rhs_compatible on the zero-(volume-)mean subspace by least squares
    dyw = np.broadcast_to(np.diff(W.coords(cfg)["yf"])[None, :, None], shape).ravel()
    bh = -dyw * rhs.ravel()
    bh = bh - bh.sum() / dyw.sum() * dyw
    sol = np.linalg.lstsq(A, bh, rcond=None)[0]
    sol -= (sol * dyw).sum() / dyw.sum()
    assert np.abs(p.ravel() - sol).max() < 1e-9 * max(1.0, np.abs(sol).max())
    assert abs((p.ravel() * dyw).sum()) < 1e-10


# ---------------------------------------------------------------- P6: D(G p) = L p
@pytest.mark.parametrize("kind", ["periodic", "walls_stretched"])
def test_p6_div_grad_is_laplacian(kind):
    rng = np.random.default_rng(6)
    cfg = _periodic_cfg(8, 6, 10, lx=1.0, ly=2.0, lz=3.0) if kind == "periodic" else _wall_cfg(6, 9, 5, True)
    o = Oracle(cfg)
    p = rng.standard_normal(o.shape["p"])
    gu, gv, gw = o.gradient(p)
    assert np.abs(o.divergence(gu, gv, gw) - o.laplacian(p)).max() < 1e-10
    # adjointness of D and -G in the volume inner product:  <D u, p>_vol = -<u, G p>_faces
    u, v, w = (rng.standard_normal(o.shape[c]) for c in "uvw")
    if kind != "periodic":
        v[:, 0, :] = 0.0; v[:, -1, :] = 0.0
    dy = np.diff(W.coords(cfg)["yf"])
    vol = dy[None, :, None] * (cfg["lx"] / cfg["nx"]) * (cfg["lz"] / cfg["nz"])
    lhs = (o.divergence(u, v, w) * p * vol).sum()
    if kind == "periodic":
        volv = vol
    else:
        dyc = np.concatenate([[dy[0]], 0.5 * (dy[:-1] + dy[1:]), [dy[-1]]])
        volv = dyc[None, :, None] * (cfg["lx"] / cfg["nx"]) * (cfg["lz"] / cfg["nz"])
    rhs = -((u * gu * vol).sum() + (v * gv * volv).sum() + (w * gw * vol).sum())
    assert abs(lhs - rhs) < 1e-10 * max(1.0, abs(lhs))


# ---------------------------------------------------------------- P7: projection of a solenoidal field is the identity
def test_p7_projection_identity_and_divergence():
    cfg = W.hit(n=16, precond="jacobi", rtol=1e-13, nu=0.0, dt=1e-3, time_scheme="euler")
    o = _mk(cfg)
    u0 = [cfg["init"][c] for c in "uvw"]
    assert np.abs(o.divergence(*u0)).max() < 1e-12        # the harness field is discretely solenoidal
    info = o.step(1)
    assert info["max_abs_div"] < 1e-12
    # with nu = 0 the step is u - dt*P(C(u)); its divergence-free part is untouched to O(dt)
    cu, cv, cw = Oracle.convection(_mk(cfg))
    for a, b, cterm in zip("uvw", u0, (cu, cv, cw)):
        assert np.abs(o.get(a) - b).max() <= 1.0001 * cfg["dt"] * 3 * np.abs(cterm).max() + 1e-12


# ---------------------------------------------------------------- P12: convective conservation
def test_p12_convection_conserves_momentum_and_energy():
    cfg = W.hit(n=16, precond="jacobi")
    o = _mk(cfg)
    cu, cv, cw = o.convection()
    scale = max(np.abs(cu).max(), 1.0)
    for c in (cu, cv, cw):
        assert abs(c.sum()) < 1e-11 * c.size * scale / 100            # momentum
    e = (cfg["init"]["u"] * cu).sum() + (cfg["init"]["v"] * cv).sum() + (cfg["init"]["w"] * cw).sum()
    assert abs(e) < 1e-10 * (np.abs(cu).sum() + np.abs(cv).sum() + np.abs(cw).sum())  # kinetic energy


def test_p12_convection_of_uniform_flow_vanishes_and_galilean_term():
    # u = const => C = 0;  u = U0 + f(y) only => C_x = 0 (no x-variation), pins transposed v/u operands
    cfg = _periodic_cfg(8, 8, 8)
    o = Oracle(cfg)
    o.set("u", np.full(o.shape["u"], 1.3)); o.set("v", np.full(o.shape["v"], -0.4)); o.set("w", np.full(o.shape["w"], 0.7))
    for c in o.convection():
        assert np.abs(c).max() < 1e-13
    # u = sin(y_c), v = V0 const, w = 0  =>  C_x = V0 * d/dy(sin y) discretely = V0*(sin(y+h)-sin(y-h))/(2h)
    c = W.coords(cfg)
    h = c["yc"][1] - c["yc"][0]
    o.set("u", np.sin(c["yc"])[None, :, None] * np.ones(o.shape["u"]))
    o.set("v", np.full(o.shape["v"], 0.5)); o.set("w", np.zeros(o.shape["w"]))
    cu, cv, cw = o.convection()
    ref = 0.5 * (np.sin(c["yc"] + h) - np.sin(c["yc"] - h)) / (2 * h)
    assert np.abs(cu - ref[None, :, None]).max() < 1e-13
    assert np.abs(cv).max() < 1e-13 and np.abs(cw).max() < 1e-13


# ---------------------------------------------------------------- P13: discrete Poiseuille steady state
def test_p13_poiseuille_uniform_y_exact_steady_state():
    ny = 16
    cfg = _wall_cfg(8, ny, 6, False, body_force=[1.0, 0.0, 0.0])
    o = Oracle(cfg)
    c = W.coords(cfg)
    hy = 2.0 / ny
    g, nu = 1.0, cfg["nu"]
    prof = g / (2 * nu) * (1.0 - c["yc"] ** 2 + hy * hy / 4.0)
    o.set("u", prof[None, :, None] * np.ones(o.shape["u"]))
    hu, hv, hw = o.momentum_rhs()
    assert np.abs(hu).max() < 1e-11 * prof.max()
    assert np.abs(hv).max() < 1e-13 and np.abs(hw).max() < 1e-13
    # a full step leaves it unchanged
    o.step(1)
    assert np.abs(o.get("u") - prof[None, :, None]).max() < 1e-11 * prof.max()


def test_p13_poiseuille_stretched_y_tridiagonal_steady_state():
    ny = 24
    cfg = _wall_cfg(6, ny, 4, True, body_force=[1.0, 0.0, 0.0])
    o = Oracle(cfg)
    yf = W.coords(cfg)["yf"]
    dy = np.diff(yf)
    dyc = np.concatenate([[dy[0]], 0.5 * (dy[:-1] + dy[1:]), [dy[-1]]])   # mirrored ghost at walls
    nu = cfg["nu"]
    T = np.zeros((ny, ny)); rhs = -np.ones(ny) / nu
    for j in range(ny):
        up, lo = 1.0 / (dy[j] * dyc[j + 1]), 1.0 / (dy[j] * dyc[j])
        T[j, j] = -(up + lo)
        if j + 1 < ny: T[j, j + 1] = up
        else: T[j, j] -= up              # ghost = -u_j (wall at rest)
        if j > 0: T[j, j - 1] = lo
        else: T[j, j] -= lo
    prof = np.linalg.solve(T, rhs)
    assert prof.min() > 0
    o.set("u", prof[None, :, None] * np.ones(o.shape["u"]))
    hu, _, _ = o.momentum_rhs()
    assert np.abs(hu).max() < 1e-10 * prof.max() * nu / dy.min() ** 2 * 1e-2 + 1e-9


def test_moving_wall_couette_linear_profile_is_steady():
    # top wall moves with U=2 in x and W=-1 in z: linear profiles are exact steady states (pins bc_vel use)
    ny = 12
    cfg = _wall_cfg(6, ny, 6, True)
    cfg["bc_vel"][3] = [2.0, 0.0, -1.0]
    o = Oracle(cfg)
    yc = W.coords(cfg)["yc"]
    s = (yc + 1.0) / 2.0
    o.set("u", 2.0 * s[None, :, None] * np.ones(o.shape["u"]))
    o.set("w", -1.0 * s[None, :, None] * np.ones(o.shape["w"]))
    hu, hv, hw = o.momentum_rhs()
    assert np.abs(hu).max() < 1e-10 and np.abs(hw).max() < 1e-10 and np.abs(hv).max() < 1e-12


def test_oracle_runs_clean_under_address_and_undefined_behaviour_sanitizers(tmp_path):
    """SURVEY 5 (sanitizer row; compute-sanitizer is closed on this pool, so the CPU side is what can be checked): the oracle
    built with -fsanitize=address,undefined runs every branch family (tests/oracle_sanitize_main.cpp) without a report."""
    import os
    import shutil
    import subprocess
    if shutil.which("g++") is None:
        pytest.skip("no g++")
    here = os.path.dirname(os.path.abspath(__file__))
    exe = str(tmp_path / "orc_san")
    cmd = ["g++", "-O1", "-g", "-std=c++17", "-ffp-contract=off", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
           os.path.join(here, "oracle_sanitize_main.cpp"), os.path.join(here, "..", "oracle", "fs_oracle.cpp"), "-o", exe]
    b = subprocess.run(cmd, capture_output=True, text=True)
    if b.returncode != 0 and "sanitize" in b.stderr and "cannot find" in b.stderr:
        pytest.skip("sanitizer runtime not installed")
    assert b.returncode == 0, b.stderr[-2000:]
    r = subprocess.run([exe], capture_output=True, text=True, env=dict(os.environ, ASAN_OPTIONS="detect_leaks=1"))
    assert r.returncode == 0 and "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr, (r.stdout[-500:], r.stderr[-3000:])
    assert "oracle sanitizer run: ok" in r.stdout
