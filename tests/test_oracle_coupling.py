"""Pins of the oracle's strong FSI coupling (Algorithm 1; reading N2-1).
CPU only."""
import math

import numpy as np
import pytest

import fs_workloads as W
import oracle as O
from oracle import Oracle


def _mk(cfg):
    o = Oracle(cfg)
    for c in "uvw":
        o.set(c, cfg["init"][c])
    if cfg.get("markers") is not None:
        o.set_markers(*cfg["markers"])
    o.set_body(*cfg["body"])
    return o


def _light(**kw):
    # a light cylinder (mass ratio 0.5 instead of 2): the added-mass effect makes the weak scheme's force lag matter
    cfg = W.cylinder_fsi(scale=8, per_ring=16, rtol=1e-9, **kw)
    m, c, k, dof = cfg["body"]
    cfg["body"] = (0.25 * m, 0.05, k, 3)
    return cfg


def test_one_sub_iteration_is_the_weakly_coupled_scheme_bit_for_bit():
    # "Setting N = 1 recovers a weakly coupled scheme"
    a, b = _mk(_light()), _mk(_light(coupling_max_iters=1, coupling_tol=1e-5))
    ia, ib = a.step(4), b.step(4)
    for c in "uvwp":
        assert np.array_equal(a.get(c), b.get(c))
    assert ia["body_disp"] == ib["body_disp"] and ib["coupling_iters"] == 1


def test_without_fluid_force_the_loop_stops_after_two_sub_iterations_on_the_free_oscillator():
    # no markers => F = 0: w^(1) = w^(2) = one RK4 step of the free oscillator (pin P15), so xi = 0 at k = 2.  (With the
    # paper's 1e-5 the loop would already stop at k = 1: xi compares with the previous time level there, as in Algorithm 1.)
    cfg = _light(coupling_max_iters=50, coupling_tol=1e-30)
    cfg["markers"] = None
    o = _mk(cfg)
    o.set_body_state([0.3, -0.2, 0.0], [0.0, 0.1, 0.0])
    m, c, k, dof = cfg["body"]
    info = o.step(1)
    assert info["coupling_iters"] == 2 and info["coupling_xi"] == 0.0
    for a in range(2):
        w, wd = O.rk4_body(m, c, k, 0.0, cfg["dt"], [0.3, -0.2][a], [0.0, 0.1][a])
        assert info["body_disp"][a] == w and info["body_vel"][a] == wd
    assert info["step"] == 1 and abs(info["time"] - cfg["dt"]) < 1e-18


def test_strong_coupling_converges_to_a_fixed_point_of_fluid_and_structure():
    # run to a tight tolerance: the structure state reproduces itself under one more fluid + structure sweep
    cfg = _light(coupling_max_iters=40, coupling_tol=1e-18)
    o = _mk(cfg)
    o.set_body_state([0.02, 0.01, 0.0], [0.0, 0.0, 0.0])            # xi is a relative change: start away from w = 0
    i1 = o.step(1)
    assert 3 <= i1["coupling_iters"] < 40 and i1["coupling_xi"] < 1e-18
    cfg2 = _light(coupling_max_iters=i1["coupling_iters"] + 4, coupling_tol=0.0)     # never stops early: 4 more sweeps
    o2 = _mk(cfg2)
    o2.set_body_state([0.02, 0.01, 0.0], [0.0, 0.0, 0.0])
    i2 = o2.step(1)
    assert i2["coupling_iters"] == i1["coupling_iters"] + 4 and i2["coupling_xi"] < 1e-18
    np.testing.assert_allclose(i2["body_disp"][:2], i1["body_disp"][:2], rtol=1e-8)
    # markers follow the converged displacement, their velocity is the converged body velocity
    X, Ub, _ = o.markers()
    X0 = cfg["markers"][0]
    for a in range(2):
        assert np.abs((X[:, a] - X0[:, a]) - (i1["body_disp"][a] - [0.02, 0.01][a])).max() < 1e-14
        assert np.all(Ub[:, a] == i1["body_vel"][a])


def test_strong_and_weak_coupling_differ_for_a_light_body_and_the_paper_tolerance_needs_a_few_sweeps():
    weak, strong = _mk(_light()), _mk(_light(coupling_max_iters=100, coupling_tol=1e-8))
    for o in (weak, strong):
        o.set_body_state([0.02, 0.01, 0.0], [0.0, 0.0, 0.0])
    iw, is_ = weak.step(2), strong.step(2)
    assert 2 <= is_["coupling_iters"] <= 20                           # "2-3 sub-iterations per step" (at its 1e-5)
    rel = abs(is_["body_vel"][0] - iw["body_vel"][0]) / abs(is_["body_vel"][0])
    assert rel > 1e-3, rel
    assert is_["converged"] == 1 and is_["max_abs_div"] < 1e-7
