"""Pins of the oracle's geometric multigrid on BOUNDED uniform grids (extension of SURVEY O7g, reading G1 in DESIGN.md 3:
the flux through a boundary face is dropped on every level, the damped-Jacobi smoother uses the true diagonal nnb / h^2).
CPU only.  The V-cycle is compared with the same cycle written as dense matrices built independently in numpy (Kronecker
products of 1-D Neumann / periodic second differences, restriction = mean of 8 children, prolongation = its transpose x 8),
so a wrong neighbour count, a flux that is not dropped, or a wrong transfer fails; plus the dense direct solve (P5) and
symmetry / iteration-count pins (P14) on bounded boxes."""
import numpy as np
import pytest

import fs_workloads as W
from oracle import Oracle


def _cfg(nx, ny, nz, bounded, **kw):
    h = 1.0 / 8
    cfg = W._base(nx=nx, ny=ny, nz=nz, lx=nx * h, ly=ny * h, lz=nz * h, nu=0.01, dt=1e-3, precond="gmg", warm_start=0, **kw)
    kinds = (("inflow", "outflow"), ("slip", "noslip"), ("noslip", "slip"))
    cfg["bc"] = [kinds[d][s] if bounded[d] else "periodic" for d in range(3) for s in range(2)]
    return cfg


def _lap1d(n, h, bounded):
    """-d2/dx2 on n cells: Neumann ends (flux dropped) or periodic."""
    A = np.zeros((n, n))
    for i in range(n):
        for di in (-1, 1):
            k = i + di
            if bounded and (k < 0 or k >= n):
                continue
            A[i, i] += 1.0 / h ** 2
            A[i, k % n] -= 1.0 / h ** 2
    return A


def _neg_lap(nx, ny, nz, h, bounded):
    Ix, Iy, Iz = np.eye(nx), np.eye(ny), np.eye(nz)
    return (np.kron(Iz, np.kron(Iy, _lap1d(nx, h, bounded[0]))) + np.kron(Iz, np.kron(_lap1d(ny, h, bounded[1]), Ix))
            + np.kron(_lap1d(nz, h, bounded[2]), np.kron(Iy, Ix)))


def _restrict(nx, ny, nz):
    cx, cy, cz = nx // 2, ny // 2, nz // 2
    R = np.zeros((cx * cy * cz, nx * ny * nz))
    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                R[(i // 2) + cx * ((j // 2) + cy * (k // 2)), i + nx * (j + ny * k)] = 0.125
    return R


def _vcycle_dense(dims, h, bounded, nu1, nu2, ncoarse, omega, nlev):
    """The V-cycle as a matrix M^-1 (recursive, dense)."""
    nx, ny, nz = dims
    A = _neg_lap(nx, ny, nz, h, bounded)
    Dinv = np.diag(1.0 / np.diag(A))
    N = A.shape[0]

    def smooth(E, n, from_zero):          # E: current iterate as a matrix acting on g (N x N); returns the new one
        for it in range(n):
            E = omega * Dinv if (from_zero and it == 0) else E + omega * Dinv @ (np.eye(N) - A @ E)
        return E
    if nlev == 1:
        return smooth(np.zeros((N, N)), ncoarse, True)
    E = smooth(np.zeros((N, N)), nu1, True) if nu1 > 0 else np.zeros((N, N))
    R = _restrict(nx, ny, nz)
    Mc = _vcycle_dense((nx // 2, ny // 2, nz // 2), 2 * h, bounded, nu1, nu2, ncoarse, omega, nlev - 1)
    E = E + (8.0 * R.T) @ Mc @ R @ (np.eye(N) - A @ E)
    return smooth(E, nu2, False)


@pytest.mark.parametrize("bounded", [(1, 1, 1), (0, 1, 0), (1, 0, 1), (0, 0, 0)])
@pytest.mark.parametrize("nu", [(2, 2, 16), (1, 0, 1), (0, 1, 3)])
def test_vcycle_equals_the_dense_matrix_cycle(bounded, nu):
    dims = (8, 16, 8)                      # 8x16x8 -> 4x8x4: two levels
    cfg = _cfg(*dims, bounded, mg_nu1=nu[0], mg_nu2=nu[1], mg_coarse_sweeps=nu[2])
    o = Oracle(cfg)
    h = cfg["lx"] / cfg["nx"]
    M = _vcycle_dense(dims, h, bounded, nu[0], nu[1], nu[2], cfg["mg_omega"], 2)
    rng = np.random.default_rng(3)
    r = rng.standard_normal(o.shape["p"])
    z = o.vcycle(r)
    ref = (M @ (r.ravel() / h)).reshape(r.shape)          # A = h (-L): z = Vcycle(r / h)
    assert np.abs(z - ref).max() < 1e-12 * np.abs(ref).max(), (bounded, nu)
    if nu[0] == nu[1]:                     # equal pre- and post-smoothing: a symmetric operator, as CG needs (true-diagonal Jacobi, P = 8 R^T)
        assert np.abs(M - M.T).max() < 1e-12 * np.abs(M).max()
    # a mistake the pin must catch: the periodic cycle on the same data is a different operator when a direction is bounded
    if any(bounded):
        Mp = _vcycle_dense(dims, h, (0, 0, 0), nu[0], nu[1], nu[2], cfg["mg_omega"], 2)
        assert np.abs((Mp - M) @ (r.ravel() / h)).max() > 1e-3 * np.abs(ref).max()


@pytest.mark.parametrize("bounded", [(1, 1, 1), (0, 1, 0), (1, 1, 0)])
def test_gmg_pcg_matches_the_dense_direct_solve_on_bounded_boxes(bounded):
    cfg = _cfg(8, 8, 8, bounded, rtol=1e-13, max_iter=200)
    o = Oracle(cfg)
    shape = o.shape["p"]
    N = int(np.prod(shape))
    A = np.zeros((N, N))
    for q in range(N):
        e = np.zeros(N); e[q] = 1.0
        A[:, q] = o.apply_A(e.reshape(shape)).ravel()
    h = cfg["lx"] / cfg["nx"]
    assert np.abs(A - h * _neg_lap(8, 8, 8, h, bounded)).max() < 1e-12 * np.abs(A).max()   # level 0 of the cycle IS the fine operator / h
    rng = np.random.default_rng(4)
    rhs = rng.standard_normal(shape)
    p, info = o.poisson_solve(rhs)
    assert info["converged"] == 1 and info["pcg_iters"] <= 20      # rtol 1e-13 on a two-level 8^3 grid
    bh = -h * rhs.ravel(); bh -= bh.mean()
    sol = np.linalg.lstsq(A, bh, rcond=None)[0]; sol -= sol.mean()
    assert np.abs(p.ravel() - sol).max() < 1e-9 * np.abs(sol).max()


def test_gmg_iterations_on_a_neumann_box_do_not_grow_with_the_grid_and_beat_jacobi():
    its = {}
    for n in (16, 32, 64):
        cfg = _cfg(n, n, n, (1, 1, 1), rtol=1e-8, max_iter=500)
        cfg.update(lx=1.0, ly=1.0, lz=1.0)
        o = Oracle(cfg)
        c = W.coords(cfg)
        X, Y, Z = c["xc"][None, None, :], c["yc"][None, :, None], c["zc"][:, None, None]
        rhs = np.cos(np.pi * X) * np.cos(2 * np.pi * Y) * np.cos(np.pi * Z) + 0.3 * np.cos(5 * np.pi * X)
        p, info = o.poisson_solve(rhs)
        assert info["converged"] == 1
        its[n] = info["pcg_iters"]
        if n == 32:
            pj, ij = Oracle(dict(cfg, precond="jacobi")).poisson_solve(rhs)
            assert ij["pcg_iters"] > 3 * info["pcg_iters"] and np.abs(p - pj).max() < 1e-6 * np.abs(pj).max()
    assert max(its.values()) - min(its.values()) <= 3 and max(its.values()) <= 16, its
