"""Pins of the oracle's time-integration variants (SURVEY 8(f) NEXT-3 remainder; Table 1):
explicit Runge-Kutta (reading N3-3: three-stage SSP scheme, every stage a full fractional step) and the CFL-adaptive
step size (reading N3-2), incl. Adams-Bashforth with a varying step.  Closed forms on the Taylor-Green mode, whose
discrete convective term is a pure gradient (pin P1), so its amplitude obeys the linear ODE a' = -nu k~^2 a exactly.
CPU only."""
import math

import numpy as np
import pytest

import fs_workloads as W
from oracle import Oracle


def _tg(n=16, **kw):
    cfg = W.taylor_green(n=n, **kw)
    h = 2 * math.pi / n
    kt2 = 8.0 / h ** 2 * math.sin(h / 2) ** 2
    return cfg, h, kt2


def _amp(o, cfg):
    return np.abs(o.get("u")).max() / np.abs(cfg["init"]["u"]).max()


def _mk(cfg):
    o = Oracle(cfg)
    for c in "uvw":
        o.set(c, cfg["init"][c])
    return o


def test_rk3_taylor_green_amplitude_is_the_third_order_stability_polynomial():
    cfg, h, kt2 = _tg(nu=0.1, dt=0.05, time_scheme="rk3", rtol=1e-13)
    z = -cfg["nu"] * kt2 * cfg["dt"]
    R = 1.0 + z + z * z / 2.0 + z ** 3 / 6.0
    o = _mk(cfg)
    info = o.step(5)
    assert abs(_amp(o, cfg) - R ** 5) < 1e-12
    # distinguishable from its neighbours: Euler (1 + z), the second-order polynomial and exp(z)
    for other in (1.0 + z, 1.0 + z + z * z / 2.0, math.exp(z)):
        assert abs(R ** 5 - other ** 5) > 1e-9
    assert info["max_abs_div"] < 1e-12 and np.abs(o.get("w")).max() < 1e-14
    assert abs(info["time"] - 5 * cfg["dt"]) < 1e-15 and info["dt"] == cfg["dt"]


def test_rk3_is_third_order_in_time_on_a_nonlinear_flow():
    # smooth, fully nonlinear periodic flow; error against a small-step reference shrinks 8x per halving of dt
    n = 12
    L = 2 * math.pi
    base = W._base(nx=n, ny=n, nz=n, lx=L, ly=L, lz=L, nu=0.05, rtol=1e-13, time_scheme="rk3", dt=1.0)
    c = W.coords(base)
    xf, xc, yf, yc, zf, zc = c["xf"][:-1], c["xc"], c["yf"][:-1], c["yc"], c["zf"][:-1], c["zc"]
    u0 = np.sin(xf)[None, None, :] * np.cos(yc)[None, :, None] * np.cos(zc)[:, None, None] + 0.3 * np.sin(2 * yc)[None, :, None] * np.ones((n, 1, n))
    v0 = -0.5 * np.cos(xc)[None, None, :] * np.sin(yf)[None, :, None] * np.cos(zc)[:, None, None]
    w0 = -0.5 * np.cos(xc)[None, None, :] * np.cos(yc)[None, :, None] * np.sin(zf)[:, None, None]

    def run(dt, T=0.32):
        cfg = dict(base, dt=dt)
        o = Oracle(cfg)
        # one projection step first would change the comparison: start from the same (discretely solenoidal by construction) field
        o.set("u", u0); o.set("v", v0); o.set("w", w0)
        o.step(int(round(T / dt)))
        return np.concatenate([o.get(k).ravel() for k in "uvw"])
    ref = run(0.005)
    e1 = np.abs(run(0.08) - ref).max()
    e2 = np.abs(run(0.04) - ref).max()
    assert e2 < 1e-5 and 6.0 < e1 / e2 < 10.5, (e1, e2, e1 / e2)


def test_cfl_adaptive_step_size_closed_forms():
    # uniform stream: dt = CFL h / |u|_max exactly; capped by the configured dt
    n = 8
    L = 2.0
    cfg = W._base(nx=n, ny=n, nz=n, lx=L, ly=L, lz=L, nu=0.01, dt=0.5, cfl=0.3, time_scheme="euler")
    o = Oracle(cfg)
    o.set("u", np.full(o.shape["u"], -2.0)); o.set("v", np.full(o.shape["v"], 0.5)); o.set("w", np.zeros(o.shape["w"]))
    info = o.step(1)
    assert info["dt"] == 0.3 * (L / n) / 2.0 and info["time"] == info["dt"]
    o = Oracle(dict(cfg, cfl=30.0))
    o.set("u", np.full(o.shape["u"], -2.0))
    assert o.step(1)["dt"] == 0.5
    # stretched grid: h_min is the smallest cell extent in any direction
    ch = W.channel(n=8, cfl=0.25, time_scheme="euler", dt=1.0)
    o = Oracle(ch)
    o.set("u", np.full(o.shape["u"], 3.0))
    dmin = min(np.diff(ch["yf"]).min(), ch["lx"] / 8, ch["lz"] / 8)
    assert abs(o.step(1)["dt"] - 0.25 * dmin / 3.0) < 1e-16


@pytest.mark.parametrize("scheme", ["euler", "ab2"])
def test_adaptive_dt_taylor_green_amplitude_recursion(scheme):
    # dt_n follows the decaying maximum velocity; Euler: a_{n+1} = a_n (1 - nu k~^2 dt_n); AB2 with the step ratio
    # r = dt_n / dt_{n-1}: a_{n+1} = a_n - nu k~^2 dt_n [(1 + r/2) a_n - (r/2) a_{n-1}]  (Euler start)
    cfg, h, kt2 = _tg(nu=0.5, dt=1.0, cfl=0.2, time_scheme=scheme, rtol=1e-13)
    o = _mk(cfg)
    m0 = max(np.abs(cfg["init"][k]).max() for k in "uvw")
    a, dts = [1.0], []
    for s in range(6):
        dt = min(1.0, 0.2 * h / (a[-1] * m0))
        if scheme == "ab2" and s > 0:
            r = dt / dts[-1]
            a.append(a[-1] - cfg["nu"] * kt2 * dt * ((1 + r / 2) * a[-1] - (r / 2) * a[-2]))
        else:
            a.append(a[-1] * (1 - cfg["nu"] * kt2 * dt))
        dts.append(dt)
        info = o.step(1)
        assert abs(info["dt"] - dt) < 1e-13 * dt, (s, info["dt"], dt)
        assert abs(_amp(o, cfg) - a[-1]) < 1e-12, (s, _amp(o, cfg), a[-1])
    assert dts[-1] > dts[0] * 1.05 and abs(info["time"] - sum(dts)) < 1e-13      # the step grows as the vortex decays
