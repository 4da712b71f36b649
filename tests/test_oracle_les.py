"""Pins of the oracle's LES closures (section 3.4.5): constant
Smagorinsky eddy viscosity (reading N4-1) and the Spalding-law equilibrium wall model (Eq. 27-29, reading N4-2).
CPU only; closed forms, and a root finder that is not the oracle's (scipy brentq) for Spalding's law."""
import math

import numpy as np
import pytest
from scipy.optimize import brentq

import fs_workloads as W
import oracle as O
from oracle import Oracle

KAP, B = 0.4, 5.0


def spalding_residual(up, yp):
    ku = KAP * up
    return up + math.exp(-KAP * B) * (math.exp(ku) - 1 - ku - ku ** 2 / 2 - ku ** 3 / 6) - yp


def test_smagorinsky_on_a_linear_shear_is_cs_delta_squared_times_the_shear_rate():
    # Couette profile between moving no-slip walls, stretched y: |S| = gamma in EVERY cell (the no-slip ghost value
    # 2 u_wall - u continues the linear profile), nu_t = (C_s (hx dy_j hz)^(1/3))^2 gamma
    ny, gam, cs = 10, 1.7, 0.17
    yf = np.tanh(1.3 * (2.0 * np.arange(ny + 1) / ny - 1.0)) / math.tanh(1.3)
    cfg = W._base(nx=6, ny=ny, nz=5, lx=1.2, ly=2.0, lz=0.8, y0=-1.0, yf=yf, nu=0.01, dt=1e-3, cs=cs)
    cfg["bc"] = ["periodic", "periodic", "noslip", "noslip", "periodic", "periodic"]
    cfg["bc_vel"][2] = [-gam, 0.0, 0.0]; cfg["bc_vel"][3] = [gam, 0.0, 0.0]
    o = Oracle(cfg)
    yc = 0.5 * (yf[:-1] + yf[1:])
    o.set("u", np.broadcast_to((gam * yc)[None, :, None], o.shape["u"]).copy())
    o.set("v", np.zeros(o.shape["v"])); o.set("w", np.zeros(o.shape["w"]))
    nut = o.eddy_viscosity()
    want = (cs * np.cbrt(0.2 * np.diff(yf) * 0.16)) ** 2 * gam
    assert np.abs(nut - want[None, :, None]).max() < 1e-14
    # and the momentum right-hand side: d/dy[(nu + nu_t) du/dy] with du/dy = gamma and nu_t varying with dy_j
    hu = o.momentum_rhs()[0]
    nte = np.empty(ny + 1); nte[1:-1] = 0.5 * (want[:-1] + want[1:]); nte[0] = want[0]; nte[-1] = want[-1]
    ref = (nte[1:] - nte[:-1]) * gam / np.diff(yf)
    assert np.abs(hu - ref[None, :, None]).max() < 1e-12


def test_smagorinsky_strain_rate_closed_form_pins_every_gradient():
    # u = A sin y + D sin x, v = B sin z + E sin y, w = C sin x + F sin z on a periodic box: all nine gradients have
    # distinct amplitudes; the discrete derivatives of sines are the exact ones times sin(h)/h (central differences of
    # centre values) or sin(h/2)/(h/2) (face differences), and averaging a sine to the centre multiplies it by cos(h/2)
    n = 12
    L = 2 * math.pi
    h = L / n
    A, Bc, Cc, D, E, F = 0.9, -0.6, 0.4, 0.3, -0.5, 0.7
    cs = 0.2
    cfg = W._base(nx=n, ny=n, nz=n, lx=L, ly=L, lz=L, nu=0.01, dt=1e-3, cs=cs)
    o = Oracle(cfg)
    c = W.coords(cfg)
    xf, xc, yf, yc, zf, zc = c["xf"][:-1], c["xc"], c["yf"][:-1], c["yc"], c["zf"][:-1], c["zc"]
    o.set("u", A * np.sin(yc)[None, :, None] + D * np.sin(xf)[None, None, :] + np.zeros((n, 1, 1)))
    o.set("v", Bc * np.sin(zc)[:, None, None] + E * np.sin(yf)[None, :, None] + np.zeros((1, 1, n)))
    o.set("w", Cc * np.sin(xc)[None, None, :] + F * np.sin(zf)[:, None, None] + np.zeros((1, n, 1)))
    s1, s2 = math.sin(h) / h, math.sin(h / 2) / (h / 2)
    X, Y, Z = xc[None, None, :], yc[None, :, None], zc[:, None, None]
    dudx, dvdy, dwdz = D * np.cos(X) * s2, E * np.cos(Y) * s2, F * np.cos(Z) * s2
    dudy, dvdz, dwdx = A * np.cos(Y) * s1, Bc * np.cos(Z) * s1, Cc * np.cos(X) * s1      # the other three cross terms vanish
    S2 = 2 * (dudx ** 2 + dvdy ** 2 + dwdz ** 2) + dudy ** 2 + dwdx ** 2 + dvdz ** 2
    want = (cs * h) ** 2 * np.sqrt(S2)
    assert np.abs(o.eddy_viscosity() - want).max() < 1e-13
    # cs = 0: the plain constant-viscosity right-hand side, bit for bit
    o0 = Oracle(dict(cfg, cs=0.0))
    for k in "uvw":
        o0.set(k, o.get(k))
    a = o0.momentum_rhs()
    o1 = Oracle(dict(cfg, cs=1e-300))                                                    # LES path with nu_t ~ 0
    for k in "uvw":
        o1.set(k, o.get(k))
    for x, y in zip(a, o1.momentum_rhs()):
        assert np.abs(x - y).max() < 1e-11 * np.abs(x).max()                            # flux form = nu Lap(u) to rounding


@pytest.mark.parametrize("yp_target", [0.01, 0.3, 5.0, 11.0, 30.0, 300.0, 5000.0, 2.0e5])
def test_spalding_law_root_against_an_independent_solver(yp_target):
    nu, y = 1.0e-3, 0.02
    up = brentq(lambda u: spalding_residual(u, yp_target), 0.0, min(yp_target + 1.0, 60.0), xtol=1e-15, rtol=1e-15)
    ut = yp_target * nu / y
    U = up * ut
    got = O.wall_utau(U, y, nu)
    assert abs(got - ut) < 1e-11 * ut, (got, ut)
    assert abs(spalding_residual(U / got, y * got / nu)) < 1e-9 * yp_target
    if yp_target <= 0.3:
        assert abs(got - math.sqrt(nu * U / y)) < 1e-3 * got                # viscous sublayer: u+ = y+
    if 300 <= yp_target <= 5000:
        assert abs(up - (math.log(yp_target) / KAP + B)) < 0.02 * up          # log law
    assert O.wall_utau(0.0, y, nu) == 0.0


def test_wall_model_sets_the_wall_flux_to_the_modelled_stress():
    # uniform stream (u, w) = (U0, W0) between no-slip walls at rest, C_s = 0: the only non-zero flux is the one through the
    # wall faces, H_u(first row) = -(tau_w1 / rho) g / (g + eps) / dy with g = U0 / (dy/2), tau_w1 = tau_w U0 / |U| (Eq. 28-29)
    ny, U0, W0, nu = 8, 2.0, -0.7, 2.0e-4
    cfg = W._base(nx=6, ny=ny, nz=5, lx=1.2, ly=2.0, lz=0.8, y0=-1.0, nu=nu, dt=1e-3, wall_model=1)
    cfg["bc"] = ["periodic", "periodic", "noslip", "noslip", "periodic", "periodic"]
    o = Oracle(cfg)
    o.set("u", np.full(o.shape["u"], U0)); o.set("v", np.zeros(o.shape["v"])); o.set("w", np.full(o.shape["w"], W0))
    hu, hv, hw = o.momentum_rhs()
    dy = 2.0 / ny
    y1 = dy / 2
    Um = math.hypot(U0, W0)
    up = brentq(lambda ut: spalding_residual(Um / ut, y1 * ut / nu), math.sqrt(nu * Um / y1), 2.0, xtol=1e-16, rtol=1e-15)   # root in u_tau
    tau = up ** 2
    for H, comp in ((hu, U0), (hw, W0)):
        g = comp / y1
        want = -(tau * comp / Um) * g / (g + 1e-6) / dy
        assert np.abs(H[:, 0, :] - want).max() < 1e-9 * abs(want)
        assert np.abs(H[:, -1, :] - want).max() < 1e-9 * abs(want)
        assert np.abs(H[:, 1:-1, :]).max() < 1e-13
    assert np.abs(hv).max() < 1e-13
    assert tau > 3 * nu * Um / y1                                             # far above the laminar wall stress: the model acts
    # wall model off: the laminar wall flux -nu (2 U0 / dy) / dy
    o = Oracle(dict(cfg, wall_model=0))
    o.set("u", np.full(o.shape["u"], U0)); o.set("w", np.full(o.shape["w"], W0))
    assert np.abs(o.momentum_rhs()[0][:, 0, :] + nu * 2 * U0 / dy / dy).max() < 1e-12


def test_les_channel_steps_run_and_stay_divergence_free():
    cfg = W.channel(n=16, cs=0.1, wall_model=1, nu=1.0 / 2000.0)
    o = Oracle(cfg)
    for k in "uvw":
        o.set(k, cfg["init"][k])
    info = o.step(3)
    assert info["converged"] == 1 and info["max_abs_div"] < 1e-7 and info["nan_flag"] == 0
    assert o.eddy_viscosity().min() >= 0.0 and o.eddy_viscosity().max() > 0.0
