"""Pins of the oracle's paper-literal eps-mask IBM (Eq. 5, Eq. 8-9,
Eq. 18-19, Eq. 23; reading E1 in DESIGN.md 3).  CPU only."""
import math

import numpy as np
import pytest

import fs_workloads as W
import oracle as O
from oracle import Oracle

H = 0.125


def _cfg(nx, ny, nz, bc=None, **kw):
    p = dict(nx=nx, ny=ny, nz=nz, lx=nx * H, ly=ny * H, lz=nz * H, nu=0.02, dt=2e-3, rtol=1e-11)
    p.update(kw)
    c = W._base(**p)
    if bc:
        c["bc"] = list(bc)
    return c


def _block(shape, k, j, i):
    e = np.zeros(shape, dtype=np.uint8)
    e[k[0]:k[1], j[0]:j[1], i[0]:i[1]] = 1
    return e


def _classify(eps, cfg):
    """Brute-force face classes (0 fluid, 1 solid, 2 IB point) written independently with numpy rolls (periodic box)."""
    out = []
    for c, ax in zip("uvw", (2, 1, 0)):
        solid = np.maximum(eps, np.roll(eps, 1, axis=ax))          # face between cell-1 and cell
        nb = np.zeros_like(solid)
        for a in (0, 1, 2):
            for sft in (1, -1):
                nb = np.maximum(nb, np.roll(solid, sft, axis=a))
        out.append(np.where(solid == 1, 1, np.where(nb == 1, 2, 0)).astype(np.uint8))
    return out


def test_mask_eps_zero_reproduces_the_unmasked_step_bit_for_bit():
    # Eq. 9 reduces to the classical Poisson equation when eps = 0
    for cfg in (W.taylor_green(n=12), W.sphere(scale=8, n_markers=4)):
        cfg["markers"] = None
        a, b = Oracle(cfg), Oracle(cfg)
        for o in (a, b):
            for c in "uvw":
                o.set(c, cfg["init"][c] + (0.05 * np.sin(np.arange(cfg["init"][c].size)).reshape(cfg["init"][c].shape) if c != "u" else 0.0))
        b.set_solid_mask(np.zeros(b.shape["p"], dtype=np.uint8), [0.3, 0.0, 0.0])
        ia, ib = a.step(3), b.step(3)
        assert ia["iters_per_step"] == ib["iters_per_step"]
        for c in "uvwp":
            assert np.array_equal(a.get(c), b.get(c)), c


def test_mask_face_classes_against_brute_force():
    cfg = _cfg(10, 9, 8)
    o = Oracle(cfg)
    rng = np.random.default_rng(31)
    eps = (rng.random(o.shape["p"]) < 0.15).astype(np.uint8)
    eps |= _block(o.shape["p"], (2, 5), (3, 6), (4, 8))
    o.set_solid_mask(eps)
    for got, want, c in zip(o.face_masks(), _classify(eps, cfg), "uvw"):
        assert np.array_equal(got, want), c
    # bounded direction: prescribed boundary-normal faces are never forced, cells outside the box are fluid
    cfg = _cfg(8, 6, 6, bc=["inflow", "outflow", "slip", "slip", "periodic", "periodic"])
    o = Oracle(cfg)
    eps = _block(o.shape["p"], (0, 6), (0, 2), (0, 3))
    o.set_solid_mask(eps)
    mu, mv, mw = o.face_masks()
    assert mu[:, :, 0].max() == 0 and mu[:, :, -1].max() == 0 and mv[:, 0, :].max() == 0 and mv[:, -1, :].max() == 0
    assert mu[0, 0, 1] == 1 and mu[0, 0, 3] == 1 and mu[0, 0, 4] == 2 and mu[0, 0, 5] == 0
    assert mv[0, 1, 0] == 1 and mv[0, 2, 0] == 1 and mv[0, 3, 0] == 2 and mw[0, 2, 0] == 2 and mw[0, 1, 0] == 1


def test_mask_block_in_a_uniform_stream_forcing_and_body_force_closed_form():
    # uniform stream U in a periodic box: H = 0, so u~ = U; Eq. 4 + 5 give u* = u_c on every solid face and leave the
    # rest alone (no markers: IB points are not forced); force on the body = -rho sum f dv = rho (U - u_c) / dt x (#faces h^3)
    U = np.array([1.0, -0.4, 0.25]); uc = np.array([0.2, 0.1, 0.0])
    cfg = _cfg(12, 10, 8, rho=1.7)
    o = Oracle(cfg)
    for c, val in zip("uvw", U):
        o.set(c, np.full(o.shape[c], val))
    eps = _block(o.shape["p"], (2, 5), (3, 7), (4, 9))
    o.set_solid_mask(eps, uc)
    masks = o.face_masks()
    ut = o.predict(0); us = o.predict(1)
    for c in range(3):
        assert np.abs(ut[c] - U[c]).max() < 1e-15
        assert np.all(us[c][masks[c] == 1] == uc[c])
        assert np.array_equal(us[c][masks[c] != 1], ut[c][masks[c] != 1])
    info = o.step(1)
    for c in range(3):
        nf = int((masks[c] == 1).sum())
        want = cfg["rho"] * (U[c] - uc[c]) / cfg["dt"] * nf * H ** 3
        assert abs(info["body_force"][c] - want) < 1e-10 * abs(want)
    # faces per component: a 3 x 4 x 5 block has (5+1) x 4 x 3 solid u faces etc.
    assert [(m == 1).sum() for m in masks] == [6 * 4 * 3, 5 * 5 * 3, 5 * 4 * 4]
    assert info["converged"] == 1 and info["max_abs_div"] < 1e-8
    # after the projection the solid faces differ from u_c only by the pressure gradient (Eq. 10 is applied everywhere)
    gp = o.gradient(o.get("p"))
    for c, name in enumerate("uvw"):
        m = masks[c] == 1
        assert np.abs(o.get(name)[m] - (uc[c] - cfg["dt"] / cfg["rho"] * gp[c][m])).max() < 1e-12


@pytest.mark.parametrize("kind,first_row,fn", [("roma3", 1.0, 0.5), ("peskin4", (2.0 + math.sqrt(2.0)) / 4.0, 0.5)])
def test_mask_ib_point_velocity_half_distribution_on_a_flat_wall(kind, first_row, fn):
    # Eq. 18-19 on a flat wall (solid slab below the face plane y_f(j0)), one marker per wall cell (spacing h, dV = h^3)
    # moving with the constant velocity W.  The fluid-side nodes of a tangential component sit at d = h/2, 3h/2 above the
    # wall: F_N = phi(1/2) + phi(3/2) = 1/2 for both kernels (P8), and by the partition of unity in x and z
    #   u_IB(first fluid row) = W phi(1/2) / F_N = W (Roma) or W (2 + sqrt 2) / 4 (Eq. 22 kernel).
    # The wall-normal component's first fluid node is at d = h: phi(1) / (phi(1) + phi(2)) = 1 for both.
    Wv = np.array([0.7, -0.3, 0.45])
    nx, ny, nz, j0 = 8, 12, 6, 5
    cfg = _cfg(nx, ny, nz, delta=kind, max_markers=nx * nz)
    o = Oracle(cfg)
    for c in "uvw":
        o.set(c, np.zeros(o.shape[c]))
    eps = np.zeros(o.shape["p"], dtype=np.uint8); eps[:, 1:j0, :] = 1      # slab of 4 cells; row 0 stays fluid
    o.set_solid_mask(eps, [0.0, 0.0, 0.0])
    xc = (np.arange(nx) + 0.5) * H; zc = (np.arange(nz) + 0.5) * H
    X = np.array([[x, j0 * H, z] for z in zc for x in xc])
    o.set_markers(X, np.tile(Wv, (X.shape[0], 1)))
    us = o.predict(1)
    mu, mv, mw = o.face_masks()
    assert np.all(mu[:, j0, :] == 2) and np.all(mw[:, j0, :] == 2) and np.all(mv[:, j0 + 1, :] == 2) and np.all(mv[:, j0, :] == 1)
    assert np.abs(us[0][:, j0, :] - first_row * Wv[0]).max() < 1e-13
    assert np.abs(us[2][:, j0, :] - first_row * Wv[2]).max() < 1e-13
    assert np.abs(us[1][:, j0 + 1, :] - Wv[1]).max() < 1e-13
    assert np.abs(us[1][:, j0, :]).max() == 0.0                              # solid face: u_c = 0
    assert np.abs(us[0][:, j0 + 1, :]).max() == 0.0                          # second fluid row: not an IB point, untouched
    assert abs(O.delta_phi(kind, 0.5) + O.delta_phi(kind, 1.5) - fn) < 1e-15


def test_mask_rigid_body_velocity_is_the_solid_velocity():
    # with a rigid body attached (Eq. 12) the solid moves with the body: u_c = body velocity (Eq. 8, "exact velocity of
    # the immersed solid"), and the force from the mask forcing drives the oscillator
    cfg = _cfg(12, 10, 6)
    o = Oracle(cfg)
    for c, val in zip("uvw", (1.0, 0.0, 0.0)):
        o.set(c, np.full(o.shape[c], val))
    eps = _block(o.shape["p"], (0, 6), (3, 7), (4, 8))
    o.set_solid_mask(eps, [9.0, 9.0, 9.0])                                    # overridden by the body's velocity
    o.set_body(5.0, 0.0, 2.0, 3)
    o.set_body_state([0.0, 0.0, 0.0], [0.1, -0.2, 0.0])
    us = o.predict(1)
    mu, mv, mw = o.face_masks()
    assert np.all(us[0][mu == 1] == 0.1) and np.all(us[1][mv == 1] == -0.2) and np.all(us[2][mw == 1] == 0.0)
    info = o.step(1)
    nfu = int((mu == 1).sum())
    assert abs(info["body_force"][0] - (1.0 - 0.1) / cfg["dt"] * nfu * H ** 3) < 1e-9
    assert info["body_vel"][0] > 0.1                                          # pushed downstream
