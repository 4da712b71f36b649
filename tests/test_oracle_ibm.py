"""Pins of the oracle's IBM part, rigid body, GMG, boundary handling (SURVEY.md 8(c) P8-P11, P14,
P15 and the mass-balance property of the unpinned outflow readings).  CPU only."""
import math
import os

import numpy as np
import pytest

import fs_workloads as W
import oracle as O
from oracle import Oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _periodic_cfg(nx, ny, nz, lx=None, ly=None, lz=None, **kw):
    h = 0.125
    return W._base(nx=nx, ny=ny, nz=nz, lx=lx or nx * h, ly=ly or ny * h, lz=lz or nz * h, nu=0.01, dt=1e-3, **kw)


# ---------------------------------------------------------------- P8: delta kernels
def test_p8_delta_kernel_printed_values():
    for line in open(os.path.join(GOLD, "delta_kernel_pins.txt")):
        if line.strip() and not line.startswith("#"):
            kind, r, val = line.split()
            assert abs(O.delta_phi(kind, float(r)) - float(val)) < 1e-15
            assert abs(O.delta_phi(kind, -float(r)) - float(val)) < 1e-15


@pytest.mark.parametrize("kind,sumsq", [("roma3", 0.5), ("peskin4", 0.375)])
def test_p8_delta_kernel_moment_identities(kind, sumsq):
    rng = np.random.default_rng(8)
    for x in np.concatenate([rng.uniform(-1, 1, 50), [0.0, 0.5, -0.5, 0.25]]):
        nodes = np.arange(-4, 5)
        ph = np.array([O.delta_phi(kind, x - m) for m in nodes])
        assert abs(ph.sum() - 1.0) < 1e-14                      # zeroth moment
        assert abs(((x - nodes) * ph).sum()) < 1e-14            # first moment
        assert abs((ph * ph).sum() - sumsq) < 1e-14             # sum of squares
        if kind == "peskin4":
            assert abs(ph[nodes % 2 == 0].sum() - 0.5) < 1e-14  # even/odd
    assert O.delta_phi("roma3", 1.5000001) == 0.0 and O.delta_phi("peskin4", 2.0000001) == 0.0


# ---------------------------------------------------------------- P9: interpolation exactness
@pytest.mark.parametrize("kind", ["roma3", "peskin4"])
def test_p9_interpolation_reproduces_constant_and_linear_fields(kind):
    rng = np.random.default_rng(9)
    cfg = _periodic_cfg(16, 12, 10, delta=kind)
    o = Oracle(cfg)
    c = W.coords(cfg)
    # markers well inside so the linear field does not see the periodic jump
    X = np.stack([rng.uniform(0.5, 1.4, 40), rng.uniform(0.5, 0.9, 40), rng.uniform(0.4, 0.8, 40)], axis=1)
    X[0] = [c["xf"][5], c["yc"][4], c["zf"][3]]               # exactly on nodes / faces
    o.set_markers(X)
    a = np.array([0.3, -1.2, 0.7]); b0 = 0.9
    def lin(x, y, z): return b0 + a[0] * x + a[1] * y + a[2] * z
    u = lin(c["xf"][:-1][None, None, :], c["yc"][None, :, None], c["zc"][:, None, None])
    v = lin(c["xc"][None, None, :], c["yf"][:-1][None, :, None], c["zc"][:, None, None])
    w = lin(c["xc"][None, None, :], c["yc"][None, :, None], c["zf"][:-1][:, None, None])
    out = o.interpolate(u, v, w)
    ref = lin(X[:, 0], X[:, 1], X[:, 2])
    for comp in range(3):
        assert np.abs(out[:, comp] - ref).max() < 1e-13
    out = o.interpolate(np.full(o.shape["u"], 2.5), np.full(o.shape["v"], -1.5), np.full(o.shape["w"], 0.5))
    assert np.abs(out - np.array([2.5, -1.5, 0.5])[None, :]).max() < 1e-14


# ---------------------------------------------------------------- P10: adjointness / conservation
@pytest.mark.parametrize("kind", ["roma3", "peskin4"])
def test_p10_spread_is_adjoint_of_interpolate_and_conserves_force(kind):
    rng = np.random.default_rng(10)
    cfg = _periodic_cfg(10, 8, 12, delta=kind)
    o = Oracle(cfg)
    n = 60
    X = np.stack([rng.uniform(-0.3, 1.6, n), rng.uniform(0, 1, n), rng.uniform(0, 1.5, n)], axis=1)  # crosses the wrap
    dV = rng.uniform(0.5, 1.5, n) * 0.125 ** 3
    o.set_markers(X, None, dV)
    F = rng.standard_normal((n, 3))
    g = [rng.standard_normal(o.shape[c]) for c in "uvw"]
    f = o.spread(F)
    Ig = o.interpolate(*g)
    dv = 0.125 ** 3
    lhs = sum((fi * gi).sum() for fi, gi in zip(f, g)) * dv
    rhs = (F * Ig * dV[:, None]).sum()
    assert abs(lhs - rhs) < 1e-12 * max(1.0, abs(rhs))
    for comp in range(3):
        assert abs(f[comp].sum() * dv - (F[:, comp] * dV).sum()) < 1e-13


# ---------------------------------------------------------------- P11: indices and cell list vs brute force
@pytest.mark.parametrize("kind", ["roma3", "peskin4"])
def test_p11_cell_list_and_support_against_brute_force(kind):
    rng = np.random.default_rng(11)
    cfg = _periodic_cfg(8, 6, 5, delta=kind)
    o = Oracle(cfg)
    c = W.coords(cfg)
    n = 200
    X = np.stack([rng.uniform(0, 1.0, n), rng.uniform(0, 0.75, n), rng.uniform(0, 0.625, n)], axis=1)
    X[:6] = X[6:12]                                   # duplicates: same cell, tests stability
    X[20] = [c["xf"][3], c["yf"][2], c["zf"][1]]      # exactly on faces
    X[21] = [c["xc"][3], c["yc"][2], c["zc"][1]]      # exactly on centres (Roma tie r = 1/2)
    o.set_markers(X)
    cl = o.cell_list()
    h = 0.125
    # brute force: containing cell by testing every cell's half-open box
    keys = np.empty(n, dtype=np.int64)
    for l in range(n):
        found = []
        for k in range(5):
            for j in range(6):
                for i in range(8):
                    if (c["xf"][i] <= X[l, 0] < c["xf"][i + 1] and c["yf"][j] <= X[l, 1] < c["yf"][j + 1]
                            and c["zf"][k] <= X[l, 2] < c["zf"][k + 1]):
                        found.append(i + 8 * (j + 6 * k))
        assert len(found) == 1
        keys[l] = found[0]
    order = sorted(range(n), key=lambda l: (keys[l], l))
    assert cl["perm"].tolist() == order
    assert cl["keys"].tolist() == [int(keys[l]) for l in order]
    starts = [r for r in range(n) if r == 0 or keys[order[r]] != keys[order[r - 1]]] + [n]
    assert cl["seg_start"].tolist() == starts
    # support: brute force = all nodes with non-zero weight lie inside [base, base+width)
    width = 3 if kind == "roma3" else 4
    half = 1.5 if kind == "roma3" else 2.0
    for l in range(0, n, 7):
        for comp in range(3):
            for d in range(3):
                org = 0.0 if d == comp else 0.5 * h
                sc = (X[l, d] - org) / h
                b = cl["base"][comp, l, d]
                nz = [m for m in range(-6, 16) if abs(sc - m) < half - 1e-12]
                assert all(b <= m < b + width for m in nz), (l, comp, d, b, nz)


def test_ibm_direct_forcing_drives_marker_velocity_to_target():
    # one step with markers: after forcing, re-interpolated u* is closer to U^b than u~ was; the body
    # force equals -rho sum F dV (Eq. 20 summed, Eq. 12) and total momentum input matches it.
    cfg = W.sphere(scale=4, n_markers=200, rtol=1e-10)
    o = Oracle(cfg)
    for c in "uvw":
        o.set(c, cfg["init"][c])
    o.set_markers(*cfg["markers"])
    info = o.step(1)
    X, Ub, F = o.markers()
    dV = cfg["markers"][2]
    bf = -(F * dV[:, None]).sum(axis=0)
    assert np.abs(bf - np.array(info["body_force"])).max() < 1e-13 * max(1.0, np.abs(bf).max())
    assert info["body_force"][0] > 0.0                      # drag on the sphere points downstream
    assert abs(info["body_force"][1]) < 1e-3 * info["body_force"][0] + 1e-6
    assert info["converged"] == 1 and info["max_abs_div"] < 1e-6


# ---------------------------------------------------------------- P14: GMG
def test_p14_vcycle_is_symmetric_and_positive():
    rng = np.random.default_rng(14)
    cfg = W._base(nx=16, ny=16, nz=16, lx=2.0, ly=2.0, lz=2.0, nu=0.01, dt=1e-3, precond="gmg")
    o = Oracle(cfg)
    a, b = rng.standard_normal((2, 16, 16, 16))
    a -= a.mean(); b -= b.mean()
    Ma, Mb = o.vcycle(a), o.vcycle(b)
    assert abs((Ma * b).sum() - (a * Mb).sum()) < 1e-12 * abs((Ma * b).sum()) + 1e-12
    assert (Ma * a).sum() > 0 and (Mb * b).sum() > 0


def test_p14_gmg_pcg_iterations_h_independent_and_same_solution():
    its = []
    for n in (16, 32, 64):
        cfg = W._base(nx=n, ny=n, nz=n, lx=2 * math.pi, ly=2 * math.pi, lz=2 * math.pi, nu=0.01, dt=1e-3,
                      precond="gmg", rtol=1e-8, warm_start=0, max_iter=100)
        o = Oracle(cfg)
        rng = np.random.default_rng(n)
        rhs = rng.standard_normal((n, n, n))
        p, info = o.poisson_solve(rhs)
        assert info["converged"] == 1
        its.append(info["pcg_iters"])
        if n == 16:
            cfg2 = dict(cfg); cfg2["precond"] = "jacobi"; cfg2["rtol"] = 1e-12; cfg2["max_iter"] = 2000
            p2, info2 = Oracle(cfg2).poisson_solve(rhs)
            assert np.abs(p - p2).max() < 1e-7 * np.abs(p2).max()
            assert info2["pcg_iters"] > info["pcg_iters"]
    assert max(its) - min(its) <= 3, its


# ---------------------------------------------------------------- P15: rigid body
def test_p15_rk4_free_oscillator_and_static_offset():
    m, k = 2.0, 8.0
    om = math.sqrt(k / m)
    errs = []
    for dt in (0.02, 0.01):
        w, wd = 1.0, 0.0
        for _ in range(int(round(1.0 / dt))):
            w, wd = O.rk4_body(m, 0.0, k, 0.0, dt, w, wd)
        errs.append(abs(w - math.cos(om * 1.0)))
    assert errs[1] < 1e-8 and 12 < errs[0] / errs[1] < 20          # 4th order
    # heavy damping + constant force -> static offset F/k
    w, wd = 0.0, 0.0
    for _ in range(4000):
        w, wd = O.rk4_body(1.0, 4.0, 4.0, 3.0, 0.01, w, wd)
    assert abs(w - 0.75) < 1e-10 and abs(wd) < 1e-10


def test_body_coupling_moves_all_markers_by_body_displacement():
    cfg = W.cylinder_fsi(scale=8, per_ring=12, rtol=1e-9)
    o = Oracle(cfg)
    for c in "uvw":
        o.set(c, cfg["init"][c])
    X0 = cfg["markers"][0]
    o.set_markers(*cfg["markers"])
    o.set_body(*cfg["body"])
    info = o.step(3)
    X, Ub, F = o.markers()
    d = X - X0
    assert np.abs(d[:, 0]).max() == 0.0 and np.abs(d[:, 2]).max() == 0.0
    assert np.abs(d[:, 1] - info["body_disp"][1]).max() < 1e-15
    assert np.abs(Ub[:, 1] - info["body_vel"][1]).max() == 0.0 and np.abs(Ub[:, 0]).max() == 0.0


# ---------------------------------------------------------------- unpinned readings: only mass balance
def test_open_domain_mass_balance_after_flux_correction():
    cfg = W.cylinder_fsi(scale=8, per_ring=12, rtol=1e-10)
    o = Oracle(cfg)
    for c in "uvw":
        o.set(c, cfg["init"][c])
    o.set_markers(*cfg["markers"])
    info = o.step(2)
    u = o.get("u")
    h = 1.0 / 16
    net = (u[:, :, -1].sum() - u[:, :, 0].sum()) * h * h
    assert abs(net) < 1e-11 * abs(u[:, :, 0].sum() * h * h)
    assert info["max_abs_div"] < 1e-7
    # inflow face carries the seeded noise: values within U(1 +- a), not all equal
    a = cfg["inflow_noise"]
    assert np.all(np.abs(u[:, :, 0] - 1.0) <= a + 1e-15) and u[:, :, 0].std() > 0.2 * a


def test_inflow_rand_is_a_pure_function_in_unit_interval():
    r = [O.inflow_rand(2024, s, 0, a, b) for s in range(3) for a in range(5) for b in range(5)]
    assert all(0.0 <= x < 1.0 for x in r) and len(set(r)) == len(r)
    assert O.inflow_rand(2024, 1, 0, 3, 4) == O.inflow_rand(2024, 1, 0, 3, 4)
    assert abs(np.mean([O.inflow_rand(7, 0, 0, a, b) for a in range(64) for b in range(64)]) - 0.5) < 0.02
