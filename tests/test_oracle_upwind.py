"""Pins of the oracle's first-order upwind convection (Table 1).

P17a  closed form: a y-independent v = V0 + A sin(k x) carried by a constant u = U0 gives exactly the textbook
      first-order upwind difference U0 (v_i - v_{i-1}) / h (U0 > 0) or U0 (v_{i+1} - v_i) / h (U0 < 0), i.e.
      +-U0 A (2/h) sin(k h / 2) cos(k (x_i -+ h/2)); the u and w equations see no convection at all.
P17b  flux form: the convective term sums to zero over a periodic box for arbitrary fields.
P17c  order: on the Taylor-Green field the error of the upwind term against (u.grad)u = sin x cos x halves with h
      (first order), that of the central term quarters (second order).
"""
import math

import numpy as np
import pytest

import fs_workloads as W
from oracle import Oracle


def _cfg(n, **kw):
    return W._base(nx=n, ny=n, nz=4, lx=2 * math.pi, ly=2 * math.pi, lz=2 * math.pi * 4 / n, nu=0.0, dt=1e-3, **kw)


@pytest.mark.parametrize("U0", [0.7, -1.3])
def test_p17a_upwind_closed_form_constant_advection(U0):
    n, A, V0, kx = 24, 0.4, 0.25, 3
    cfg = _cfg(n, convection="upwind")
    o = Oracle(cfg)
    h = 2 * math.pi / n
    xc = (np.arange(n) + 0.5) * h
    sh = W.shapes(cfg)
    o.set("u", np.full(sh["u"], U0))
    o.set("v", np.broadcast_to(V0 + A * np.sin(kx * xc), sh["v"]).copy())
    o.set("w", np.zeros(sh["w"]))
    cu, cv, cw = o.convection()
    s = 1.0 if U0 > 0 else -1.0
    want = U0 * A * (2.0 / h) * math.sin(kx * h / 2) * np.cos(kx * (xc - s * h / 2))
    assert np.abs(cv - want[None, None, :]).max() < 1e-13
    assert np.abs(cu).max() < 1e-13 and np.abs(cw).max() == 0.0


@pytest.mark.parametrize("scheme", ["upwind", "central"])
def test_p17b_convective_term_sums_to_zero_on_a_periodic_box(scheme):
    cfg = W._base(nx=12, ny=10, nz=9, lx=1.2, ly=1.0, lz=0.9, nu=0.0, dt=1e-3, convection=scheme)
    o = Oracle(cfg)
    rng = np.random.default_rng(4)
    sh = W.shapes(cfg)
    for c in "uvw":
        o.set(c, rng.standard_normal(sh[c]))
    for a in o.convection():
        assert abs(a.sum()) < 1e-10 * np.abs(a).sum()


def _tg_error(n, scheme):
    cfg = _cfg(n, convection=scheme)
    o = Oracle(cfg)
    h = 2 * math.pi / n
    xf, xc = np.arange(n) * h, (np.arange(n) + 0.5) * h
    sh = W.shapes(cfg)
    u = np.sin(xf)[None, None, :] * np.cos(xc)[None, :, None] * np.ones(sh["u"])
    v = -np.cos(xc)[None, None, :] * np.sin(xf)[None, :, None] * np.ones(sh["v"])
    o.set("u", u); o.set("v", v); o.set("w", np.zeros(sh["w"]))
    cu, _, _ = o.convection()
    want = (np.sin(xf) * np.cos(xf))[None, None, :] * np.ones(sh["u"])
    return np.abs(cu - want).max()


def test_p17c_upwind_is_first_order_central_second_order():
    eu = [_tg_error(n, "upwind") for n in (16, 32, 64)]
    ec = [_tg_error(n, "central") for n in (16, 32, 64)]
    assert 1.7 < eu[0] / eu[1] < 2.3 and 1.8 < eu[1] / eu[2] < 2.2, eu
    assert 3.6 < ec[0] / ec[1] < 4.4 and 3.8 < ec[1] / ec[2] < 4.2, ec
