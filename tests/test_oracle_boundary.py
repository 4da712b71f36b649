"""Pins P18-P23 of the oracle's boundary handling, forcing scale and outflow readings (round-1 VERDICT "parity
unpinned" list): each is a closed form or a published value that a plausible slip (slip <-> no-slip mix-up, wrong
sign / speed of the convective outflow update, a dropped dt or dV in the direct forcing, a non-uniform flux shift,
a silently truncated support, a drifting hash constant) fails.  CPU only.

Passages: boundary types PAPER.md L429, L454-456 (Table 1); Eq. 5 at the markers L108; Eq. 3a/3b L89-91;
SURVEY.md 8(c) O1, O4, O5 for the readings of what the paper leaves open."""
import math
import os

import numpy as np
import pytest

import fs_workloads as W
import oracle as O
from oracle import Oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")
H = 0.125


def _cfg(nx, ny, nz, bc, **kw):
    p = dict(nx=nx, ny=ny, nz=nz, lx=nx * H, ly=ny * H, lz=nz * H, nu=0.05, dt=2e-3)
    p.update(kw)
    c = W._base(**p)
    c["bc"] = list(bc)
    return c


def _set(o, u, v, w):
    o.set("u", np.broadcast_to(u, o.shape["u"]).copy())
    o.set("v", np.broadcast_to(v, o.shape["v"]).copy())
    o.set("w", np.broadcast_to(w, o.shape["w"]).copy())


# ---------------------------------------------------------------- P18: tangential ghosts (O1; L455-456)
def test_p18_uniform_stream_between_slip_walls_has_zero_rhs():
    # slip wall: normal velocity 0, tangential ghost = interior (zero gradient) => a uniform stream feels nothing
    cfg = _cfg(10, 8, 6, ["periodic", "periodic", "slip", "slip", "periodic", "periodic"])
    o = Oracle(cfg)
    _set(o, 1.7, 0.0, -0.6)
    for Hc in o.momentum_rhs():
        assert np.abs(Hc).max() < 1e-13


@pytest.mark.parametrize("uw", [0.0, 0.4])
def test_p18_noslip_wall_ghost_is_2uwall_minus_interior(uw):
    # same stream, top wall switched to no-slip moving with uw: ghost = 2 uw - U0, so in the wall row
    # H_u = nu ((2 uw - U0) - U0) / h^2 exactly, and zero everywhere else (bottom wall still slip)
    U0, W0, nu = 1.7, -0.6, 0.05
    cfg = _cfg(10, 8, 6, ["periodic", "periodic", "slip", "noslip", "periodic", "periodic"])
    cfg["bc_vel"][3] = [uw, 0.0, 0.25]
    o = Oracle(cfg)
    _set(o, U0, 0.0, W0)
    hu, hv, hw = o.momentum_rhs()
    assert np.abs(hu[:, -1, :] - nu * 2.0 * (uw - U0) / H ** 2).max() < 1e-12
    assert np.abs(hw[:, -1, :] - nu * 2.0 * (0.25 - W0) / H ** 2).max() < 1e-12
    assert np.abs(hu[:, :-1, :]).max() < 1e-13 and np.abs(hw[:, :-1, :]).max() < 1e-13 and np.abs(hv).max() < 1e-13


def test_p18_inflow_tangential_ghost_and_outflow_zero_gradient():
    # sheared inlet: v = V0 inside, prescribed tangential inflow velocity Vb => ghost = 2 Vb - V0 at -x (Dirichlet),
    # ghost = interior at the convective outlet (+x).  With u = w = 0 the convective terms vanish identically.
    V0, Vb, W0, Wb, nu = 0.8, 0.3, -0.2, 0.5, 0.05
    cfg = _cfg(9, 6, 5, ["inflow", "outflow", "periodic", "periodic", "periodic", "periodic"])
    cfg["bc_vel"][0] = [1.0, Vb, Wb]
    cfg["bc_vel"][1] = [1.0, 9.0, 9.0]          # tangential entries of an outflow face must not matter
    o = Oracle(cfg)
    _set(o, 0.0, V0, W0)
    hu, hv, hw = o.momentum_rhs()
    assert np.abs(hv[:, :, 0] - nu * 2.0 * (Vb - V0) / H ** 2).max() < 1e-12
    assert np.abs(hw[:, :, 0] - nu * 2.0 * (Wb - W0) / H ** 2).max() < 1e-12
    assert np.abs(hv[:, :, 1:]).max() < 1e-13 and np.abs(hw[:, :, 1:]).max() < 1e-13


# ---------------------------------------------------------------- P19: convective outflow (O1 reading)
@pytest.mark.parametrize("side", [1, 0])
def test_p19_convective_outflow_transports_a_linear_profile_exactly(side):
    # du/dt + Uc du/dx = 0, first-order upwind over one cell: for u = a + b x the outlet face moves by -Uc dt b,
    # whatever H is (boundary-normal faces are prescribed, not advanced).  Checked BEFORE the flux correction (stage 0).
    a, b, dt = 1.0, 0.35, 2e-3
    Uc = 1.3 if side else -1.3                    # signed x velocity of the outflow (out of the box on either side)
    bc = ["inflow", "outflow"] if side else ["outflow", "inflow"]
    cfg = _cfg(12, 5, 4, bc + ["periodic"] * 4, dt=dt)
    cfg["bc_vel"][side] = [Uc, 0.0, 0.0]
    cfg["bc_vel"][1 - side] = [a + b * (0.0 if side else 12 * H), 0.0, 0.0]
    o = Oracle(cfg)
    xf = H * np.arange(13)
    u = (a + b * xf)[None, None, :]
    _set(o, u, 0.0, 0.0)
    us, vs, ws = o.predict(0)
    q = -1 if side else 0
    assert np.abs(us[:, :, q] - (u[0, 0, q] - Uc * dt * b)).max() < 1e-15
    # the inflow face carries its prescribed value, interior faces moved by dt H (H = -d(u^2)/dx = -2 b u here)
    assert np.abs(us[:, :, 0 if side else -1] - cfg["bc_vel"][1 - side][0]).max() == 0.0
    assert np.abs(us[:, :, 1:-1] - (u[:, :, 1:-1] + dt * (-2.0 * b * u[:, :, 1:-1]))).max() < 1e-13


def test_p19_convective_outflow_on_a_stretched_y_face_uses_the_wall_cell_height():
    ny = 8
    yf = np.tanh(1.5 * (2.0 * np.arange(ny + 1) / ny - 1.0)) / math.tanh(1.5)
    a, b, Uc, dt = 0.2, 0.6, 0.9, 2e-3
    cfg = _cfg(6, ny, 4, ["periodic", "periodic", "inflow", "outflow", "periodic", "periodic"], dt=dt, yf=yf, y0=-1.0, ly=2.0)
    cfg["bc_vel"][3] = [0.0, Uc, 0.0]
    cfg["bc_vel"][2] = [0.0, a + b * yf[0], 0.0]
    o = Oracle(cfg)
    v = (a + b * yf)[None, :, None]
    _set(o, 0.0, v, 0.0)
    us, vs, ws = o.predict(0)
    assert np.abs(vs[:, -1, :] - (v[0, -1, 0] - Uc * dt * b)).max() < 1e-15


# ---------------------------------------------------------------- P20: direct-forcing scale (I-3 / I-4; Eq. 5, Eq. 3)
@pytest.mark.parametrize("kind,sumsq", [("roma3", 0.5), ("peskin4", 0.375)])
@pytest.mark.parametrize("dvfac", [1.0, 2.0])
def test_p20_one_marker_forcing_moves_interpolated_velocity_by_sum_phi2_cubed(kind, sumsq, dvfac):
    # one marker, dV = dvfac h^3:  I(u*) - I(u~) = dvfac (U^b - I(u~)) (sum phi^2)^3  -- 1/8 (Roma) and 27/512
    # (Eq. 22 kernel) for dvfac = 1; pins the /dt ... *dt pair of I-3 / I-4 and the dV / (hx hy hz) factor
    rng = np.random.default_rng(20)
    cfg = _cfg(12, 10, 9, ["periodic"] * 6, delta=kind, max_markers=1)
    o = Oracle(cfg)
    c = W.coords(cfg)
    def fld(x, y, z): return np.sin(2 * math.pi * x / (12 * H))[None, None, :] * np.cos(2 * math.pi * y / (10 * H))[None, :, None] + 0.3 * np.sin(2 * math.pi * z / (9 * H))[:, None, None] + 0.5
    _set(o, fld(c["xf"][:-1], c["yc"], c["zc"]), 0.7 * fld(c["xc"], c["yf"][:-1], c["zc"]), -0.4 * fld(c["xc"], c["yc"], c["zf"][:-1]))
    X = np.array([[rng.uniform(0.3, 1.1), rng.uniform(0.3, 0.9), rng.uniform(0.3, 0.8)]])
    Ub = np.array([[0.9, -0.3, 0.2]])
    o.set_markers(X, Ub, np.array([dvfac * H ** 3]))
    ut = o.predict(0)
    us = o.predict(1)
    It, Is = o.interpolate(*ut), o.interpolate(*us)
    want = dvfac * (Ub - It) * sumsq ** 3
    assert np.abs((Is - It) - want).max() < 1e-13
    assert np.abs(Ub - It).min() > 1e-2             # the test moves something


# ---------------------------------------------------------------- P21: outflow flux correction (O5 reading)
def test_p21_flux_correction_is_a_uniform_shift_of_the_outflow_faces_only():
    ny = 10
    yf = np.tanh(1.2 * (2.0 * np.arange(ny + 1) / ny - 1.0)) / math.tanh(1.2)
    cfg = _cfg(14, ny, 6, ["inflow", "outflow", "noslip", "noslip", "periodic", "periodic"], yf=yf, y0=-1.0, ly=2.0,
               inflow_noise=0.2, seed=5)
    cfg["bc_vel"][0] = [1.0, 0.0, 0.0]
    cfg["bc_vel"][1] = [1.0, 0.0, 0.0]
    o = Oracle(cfg)
    rng = np.random.default_rng(21)
    sh = W.shapes(cfg)
    u = 1.0 + 0.3 * rng.standard_normal(sh["u"]); v = 0.3 * rng.standard_normal(sh["v"]); w = 0.3 * rng.standard_normal(sh["w"])
    v[:, 0, :] = 0.0; v[:, -1, :] = 0.0
    _set(o, u, v, w)
    a = o.predict(1)
    b = o.predict(2)
    dy = np.diff(yf); hz = H
    area = (dy * hz)[None, :]                                              # x faces: dy_j * hz
    phi = ((a[0][:, :, -1] - a[0][:, :, 0]) * area).sum()                   # net outward flux (walls: v = 0)
    assert abs(phi) > 1e-3                                                  # the noise unbalanced it
    shift = phi / (area.sum() * cfg["nz"])
    d = [bb - aa for aa, bb in zip(a, b)]
    assert np.abs(d[0][:, :, -1] + shift).max() < 1e-14                     # every outflow face: same shift
    assert np.abs(d[0][:, :, :-1]).max() == 0.0 and np.abs(d[1]).max() == 0.0 and np.abs(d[2]).max() == 0.0
    assert abs(((b[0][:, :, -1] - b[0][:, :, 0]) * area).sum()) < 1e-13     # balanced afterwards


# ---------------------------------------------------------------- P22: bounded supports are rejected
@pytest.mark.parametrize("kind,reach", [("roma3", 1.5), ("peskin4", 2.0)])
def test_p22_marker_support_touching_a_wall_is_unsupported(kind, reach):
    # the moment identities P8-P10 need the full support; a support that reaches a prescribed boundary-normal face or
    # leaves the box is refused, exactly at the distance the kernel's half width gives (Roma 1.5 h, Eq. 22 kernel 2 h)
    cfg = _cfg(16, 12, 10, ["inflow", "outflow", "slip", "slip", "periodic", "periodic"], delta=kind, max_markers=2)
    o = Oracle(cfg)
    mid = np.array([8 * H, 6 * H, 5 * H])
    for d in (0, 1):
        L = (16 if d == 0 else 12) * H
        ok_lo, ok_hi = mid.copy(), mid.copy()
        ok_lo[d] = reach * H + 1e-9; ok_hi[d] = L - reach * H - 1e-9
        o.set_markers(np.stack([ok_lo, ok_hi]))
        assert o.cell_list()["perm"].size == 2
        for bad in (reach * H - 0.01 * H, L - reach * H + 0.01 * H):
            x = mid.copy(); x[d] = bad
            with pytest.raises(ValueError, match="unsupported"):
                o.set_markers(x[None, :])
    z = mid.copy(); z[2] = 0.01 * H                      # periodic direction: supports wrap, always fine
    o.set_markers(z[None, :])


def test_p22_moving_body_that_reaches_a_wall_is_reported():
    cfg = W.cylinder_fsi(scale=8, per_ring=12, rtol=1e-8)
    o = Oracle(cfg)
    for c in "uvw":
        o.set(c, cfg["init"][c])
    o.set_markers(*cfg["markers"])
    o.set_body(*cfg["body"])
    o.set_body_state([0.0, 0.0, 0.0], [0.0, 400.0, 0.0])          # flies into the +y slip wall within the step
    o.step(1)
    with pytest.raises(ValueError, match="unsupported"):
        o.step(1)


# ---------------------------------------------------------------- P23: inflow-noise hash (O1 reading)
M64 = (1 << 64) - 1


def _splitmix(z):
    z = (z + 0x9E3779B97F4A7C15) & M64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & M64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & M64
    return z ^ (z >> 31)


def test_p23_inflow_hash_against_published_splitmix64_vectors_and_frozen_table():
    # the finaliser is SplitMix64's; its published outputs for state 0 (stream 0, 1, 2) pin the constants
    s, out = 0, []
    for _ in range(3):
        out.append(_splitmix(s)); s = (s + 0x9E3779B97F4A7C15) & M64
    assert out == [0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4, 0x06C45D188009454F]
    # the chaining over (seed, face, step, a, b) is the builder's reading (O1), restated here
    def ref(seed, step, face, a, b):
        h = _splitmix((seed + 0x632BE59BD9B4E019 * (face + 1)) & M64)
        h = _splitmix((h + step) & M64)
        h = _splitmix((h + (((b & 0xFFFFFFFF) << 32) | (a & 0xFFFFFFFF))) & M64)
        return (h >> 11) * (1.0 / 9007199254740992.0)
    for args in [(2024, 0, 0, 0, 0), (2024, 7, 0, 13, 31), (5, 3, 2, 100, 7), (0, 0, 5, 1, 2), (2 ** 63 + 11, 10 ** 9, 1, 255, 383)]:
        assert O.inflow_rand(*args) == ref(*args), args
    # frozen table written by tests/golden/make_inflow_hash_pins.py (calls only oracle/): the oracle's and the kernel's
    # transcriptions cannot drift together unnoticed
    n = 0
    for line in open(os.path.join(GOLD, "inflow_hash_pins.txt")):
        if line.strip() and not line.startswith("#"):
            seed, step, face, a, b, val = line.split()
            assert O.inflow_rand(int(seed), int(step), int(face), int(a), int(b)) == float.fromhex(val)
            n += 1
    assert n == 8
