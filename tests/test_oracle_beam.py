"""Pins of the oracle's flexible beam (third item; Eq. 11, Eq. 13-17,
Newmark-beta L177; reading N2-2 in DESIGN.md 3).  CPU only.  Closed forms of Euler-Bernoulli beam theory, an eigen-
solver that is not the oracle's (scipy), and the textbook identity Newmark(1/2, 1/4) = trapezoidal rule."""
import math

import numpy as np
import pytest
import scipy.linalg

import fs_workloads as W
from oracle import Oracle


def _beam(nodes=9, length=1.0, EI=0.7, mu=0.3, zeta=0.0, spacing=None, angle=0.0):
    """A beam in a small periodic box (the fluid is irrelevant for the structural pins)."""
    n = 16
    cfg = W._base(name="beam_box", nx=n, ny=n, nz=4, lx=4.0, ly=4.0, lz=1.0, nu=0.01, dt=1e-2)
    s = np.linspace(0.0, length, nodes) if spacing is None else np.asarray(spacing, dtype=float)
    t = np.array([math.cos(angle), math.sin(angle)])
    xy = np.array([1.3, 1.1])[None, :] + s[:, None] * t[None, :]
    xyz = np.concatenate([xy, np.full((len(s), 1), 0.5)], axis=1)
    o = Oracle(cfg)
    for c in "uvw":
        o.set(c, np.zeros(W.shapes(cfg)[c]))
    o.set_markers(xyz)
    o.set_beam(xy, np.arange(len(s)), EI, mu, zeta)
    return o, s, t


def test_static_tip_load_and_tip_moment_reproduce_the_cantilever_closed_forms():
    # Hermite cubic elements are nodally exact for point loads: w(x) = P x^2 (3L - x) / (6 EI), theta = P x (2L - x) / (2 EI);
    # tip moment: w = M x^2 / (2 EI), theta = M x / EI.  Uneven element lengths on purpose (Eq. 13 carries L_e per element).
    EI, L = 0.7, 1.3
    s = np.array([0.0, 0.1, 0.35, 0.5, 0.9, 1.05, L])
    o, s, _ = _beam(EI=EI, spacing=s)
    K, M, C, coef = o.beam_matrices()
    assert np.abs(K - K.T).max() < 1e-12 * np.abs(K).max() and np.abs(M - M.T).max() < 1e-15
    x = s[1:]
    Q = np.zeros(o.ndof); Q[-2] = 2.5                      # tip force
    w = np.linalg.solve(K, Q)
    assert np.abs(w[0::2] - 2.5 * x * x * (3 * L - x) / (6 * EI)).max() < 1e-11
    assert np.abs(w[1::2] - 2.5 * x * (2 * L - x) / (2 * EI)).max() < 1e-11
    Q = np.zeros(o.ndof); Q[-1] = 0.8                      # tip moment
    w = np.linalg.solve(K, Q)
    assert np.abs(w[0::2] - 0.8 * x * x / (2 * EI)).max() < 1e-11
    assert np.abs(w[1::2] - 0.8 * x / EI).max() < 1e-11
    # consistent mass (Eq. 14): a rigid translation of the whole beam has kinetic energy mu L / 2; with node 0 clamped the
    # deflection block misses that node's share: 1^T M_ww 1 = mu L - (row and column of node 0) = mu (L - 22/35 L_1)
    assert abs(M[0::2, 0::2].sum() - 0.3 * (L - (156.0 + 2 * 54.0) / 420.0 * (s[1] - s[0]))) < 1e-13


def test_modal_frequencies_against_the_cantilever_roots_and_an_independent_eigensolver():
    EI, mu, L = 0.9, 0.25, 1.0
    roots = (1.8751040687119611, 4.694091132974175)       # cos(bL) cosh(bL) = -1
    errs = []
    for nodes in (9, 17):
        o, _, _ = _beam(nodes=nodes, EI=EI, mu=mu)
        K, M, C, coef = o.beam_matrices()
        lam = scipy.linalg.eigh(K, M, eigvals_only=True)
        assert abs(coef["omega1"] - math.sqrt(lam[0])) < 1e-9 * math.sqrt(lam[0])
        assert abs(coef["omega2"] - math.sqrt(lam[1])) < 1e-9 * math.sqrt(lam[1])
        exact = [b * b * math.sqrt(EI / (mu * L ** 4)) for b in roots]
        errs.append([abs(coef["omega1"] - exact[0]) / exact[0], abs(coef["omega2"] - exact[1]) / exact[1]])
    assert errs[1][0] < 1e-6 and errs[1][1] < 5e-5
    assert 10.0 < errs[0][1] / errs[1][1] < 22.0           # consistent mass: fourth-order convergence of the frequencies


def test_rayleigh_damping_puts_the_damping_ratio_on_the_first_two_modes():
    zeta = 0.03
    o, _, _ = _beam(nodes=11, zeta=zeta)
    K, M, C, coef = o.beam_matrices()
    w1, w2 = coef["omega1"], coef["omega2"]
    assert abs(coef["alpha"] - 2 * zeta * w1 * w2 / (w1 + w2)) < 1e-14 and abs(coef["beta"] - 2 * zeta / (w1 + w2)) < 1e-16   # Eq. 16
    assert np.abs(C - (coef["alpha"] * M + coef["beta"] * K)).max() < 1e-12 * np.abs(C).max()                                 # Eq. 15
    lam, phi = scipy.linalg.eigh(K, M)
    for m in range(3):
        z = phi[:, m] @ C @ phi[:, m] / (2.0 * math.sqrt(lam[m]) * (phi[:, m] @ M @ phi[:, m]))
        if m < 2:
            assert abs(z - zeta) < 1e-9
        else:
            assert z > zeta * 1.5                           # stiffness-proportional part grows with frequency


def test_newmark_is_the_trapezoidal_rule_on_the_first_order_system():
    # Newmark-beta with gamma = 1/2, beta = 1/4 (average acceleration) is algebraically the trapezoidal rule on
    # y' = A y + b(t), y = (w, v), when a_n = M^-1 (Q_n - C v_n - K w_n): compare with that formulation built in numpy
    # from the exported matrices, with a random consistent start and a different random load every step.
    o, _, _ = _beam(nodes=7, zeta=0.05)
    K, M, C, _ = o.beam_matrices()
    n = o.ndof
    rng = np.random.default_rng(5)
    w, v, Q0 = rng.standard_normal(n) * 1e-2, rng.standard_normal(n) * 1e-1, rng.standard_normal(n)
    a = np.linalg.solve(M, Q0 - C @ v - K @ w)
    o.set_beam_state(w, v, a)
    dt = 3e-3
    Mi = np.linalg.inv(M)
    A = np.block([[np.zeros((n, n)), np.eye(n)], [-Mi @ K, -Mi @ C]])
    y, Qp = np.concatenate([w, v]), Q0
    for _ in range(25):
        Q = rng.standard_normal(n)
        o.beam_newmark(Q, dt)
        b0, b1 = np.concatenate([np.zeros(n), Mi @ Qp]), np.concatenate([np.zeros(n), Mi @ Q])
        y = np.linalg.solve(np.eye(2 * n) - 0.5 * dt * A, (np.eye(2 * n) + 0.5 * dt * A) @ y + 0.5 * dt * (b0 + b1))
        Qp = Q
    st = o.beam_state()
    assert np.abs(st["w"] - y[:n]).max() < 1e-10 * np.abs(y[:n]).max()
    assert np.abs(st["v"] - y[n:]).max() < 1e-10 * np.abs(y[n:]).max()
    assert np.abs(st["a"] - Mi @ (Qp - C @ st["v"] - K @ st["w"])).max() < 1e-7 * np.abs(st["a"]).max()


def test_undamped_free_vibration_keeps_its_energy_and_has_the_known_period_elongation():
    o, _, _ = _beam(nodes=9)
    K, M, C, coef = o.beam_matrices()
    lam, phi = scipy.linalg.eigh(K, M)
    om, f = math.sqrt(lam[0]), phi[:, 0] * 1e-2
    o.set_beam_state(f, np.zeros_like(f), -lam[0] * f)
    dt, nst = 0.02, 40
    E0 = 0.5 * f @ K @ f
    for _ in range(nst):
        o.beam_newmark(np.zeros(o.ndof), dt)
    st = o.beam_state()
    E = 0.5 * st["v"] @ M @ st["v"] + 0.5 * st["w"] @ K @ st["w"]
    assert abs(E - E0) < 1e-11 * E0
    theta = 2.0 * math.atan(0.5 * om * dt)                 # phase advance per step of the average-acceleration scheme
    assert np.abs(st["w"] - f * math.cos(nst * theta)).max() < 1e-10 * np.abs(f).max()
    assert abs(math.cos(nst * theta) - math.cos(nst * om * dt)) > 1e-3   # i.e. the test can tell the scheme from the exact flow


def test_one_step_from_rest_is_the_effective_stiffness_solve():
    o, _, _ = _beam(nodes=6, zeta=0.1)
    K, M, C, _ = o.beam_matrices()
    Q = np.arange(1.0, o.ndof + 1.0)
    dt = 7e-3
    o.beam_newmark(Q, dt)
    st = o.beam_state()
    w1 = np.linalg.solve(K + 4.0 / dt ** 2 * M + 2.0 / dt * C, Q)
    assert np.abs(st["w"] - w1).max() < 1e-12 * np.abs(w1).max()
    assert np.abs(st["v"] - 2.0 * w1 / dt).max() < 1e-11 * np.abs(w1).max() / dt
    assert np.abs(st["a"] - 4.0 * w1 / dt ** 2).max() < 1e-10 * np.abs(w1).max() / dt ** 2


def _plate(**kw):
    cfg = W.flexible_plate(scale=8, nodes=9, **kw)
    o = Oracle(cfg)
    for c, a in cfg["init"].items():
        o.set(c, a)
    o.set_markers(*cfg["markers"])
    o.set_beam(*cfg["beam"])
    return cfg, o


def test_coupled_step_load_is_the_projected_marker_force_and_markers_ride_on_their_nodes():
    cfg, o = _plate()
    X0 = np.asarray(cfg["markers"][0]).copy()
    node = cfg["beam"][1]
    info = o.step(2)
    x, ub, F = o.markers()
    st = o.beam_state()
    dV = cfg["markers"][2]
    nrm = np.array([-1.0, 0.0])                            # nodes run along +y: n = (-t_y, t_x) = (-1, 0)
    Q = np.zeros(o.ndof)
    for l in range(len(node)):
        if node[l] > 0:
            Q[2 * (node[l] - 1)] += -cfg["rho"] * dV[l] * (F[l, 0] * nrm[0] + F[l, 1] * nrm[1])
    assert np.abs(st["Q"] - Q).max() < 1e-12 * np.abs(Q).max()
    assert np.abs(Q[1::2]).max() == 0.0                    # no nodal moments
    assert Q[0::2].min() < 0.0 and st["w"][-2] < 0.0        # the stream pushes the plate downstream: against n = -x
    wn = np.concatenate([[0.0], st["w"][0::2]]); vn = np.concatenate([[0.0], st["v"][0::2]])
    assert np.abs(x[:, 0] - (X0[:, 0] + wn[node] * nrm[0])).max() < 1e-15
    assert np.abs(x[:, 1] - X0[:, 1]).max() == 0.0 and np.abs(x[:, 2] - X0[:, 2]).max() == 0.0
    assert np.abs(ub[:, 0] - vn[node] * nrm[0]).max() < 1e-15 and np.abs(ub[:, 1:]).max() == 0.0
    assert info["coupling_iters"] == 1


def test_strong_coupling_with_a_beam_reaches_a_fixed_point_and_one_sweep_is_the_weak_scheme():
    cfg, weak = _plate()
    weak.step(3)
    cfg1, one = _plate(coupling_max_iters=1)
    one.step(3)
    assert np.array_equal(weak.beam_state()["w"], one.beam_state()["w"]) and np.array_equal(weak.get("u"), one.get("u"))
    cfgs, strong = _plate(coupling_max_iters=40, coupling_tol=1e-16)
    i1 = strong.step(1)
    assert 2 < i1["coupling_iters"] <= 40
    cfgt, more = _plate(coupling_max_iters=i1["coupling_iters"] + 3, coupling_tol=0.0)
    more.step(1)
    a, b = strong.beam_state()["w"], more.beam_state()["w"]
    assert np.abs(a - b).max() < 1e-6 * np.abs(b).max()     # three more sweeps move the converged iterate by < 1e-6
    wk = weak.beam_state()["w"]
    assert wk.shape == a.shape
