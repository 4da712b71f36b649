"""CPU ORACLE -- test infrastructure, NOT the product.

ctypes wrapper around oracle/fs_oracle.cpp (plain single-threaded fp64 C++ written from
PAPER.md section 2.3 and SURVEY.md 8(c)).  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package; the product
(paper_2505_23940_b200) never does, and this package never imports the product.
"""
import ctypes as C

import numpy as np

from .build import build as _build

BC = {"periodic": 0, "noslip": 1, "slip": 2, "inflow": 3, "outflow": 4}
TIME = {"euler": 0, "ab2": 1, "rk3": 2}
PC = {"none": 0, "jacobi": 1, "gmg": 2}
DELTA = {"roma3": 0, "peskin4": 1}
FIELD = {"u": 0, "v": 1, "w": 2, "p": 3, "hu": 4, "hv": 5, "hw": 6, "div": 7}


class _Params(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("x0", C.c_double), ("y0", C.c_double), ("z0", C.c_double),
                ("lx", C.c_double), ("ly", C.c_double), ("lz", C.c_double),
                ("yf", C.POINTER(C.c_double)),
                ("bc", C.c_int * 6), ("bc_vel", (C.c_double * 3) * 6),
                ("nu", C.c_double), ("rho", C.c_double), ("dt", C.c_double), ("body_force", C.c_double * 3),
                ("time_scheme", C.c_int),
                ("precond", C.c_int), ("rtol", C.c_double), ("max_iter", C.c_int), ("warm_start", C.c_int),
                ("mg_nu1", C.c_int), ("mg_nu2", C.c_int), ("mg_coarse_sweeps", C.c_int), ("mg_omega", C.c_double),
                ("delta", C.c_int), ("seed", C.c_uint64), ("inflow_noise", C.c_double), ("convection", C.c_int),
                ("cs", C.c_double), ("wall_model", C.c_int),
                ("coupling_max_iters", C.c_int), ("coupling_tol", C.c_double), ("cfl", C.c_double)]


class _Info(C.Structure):
    _fields_ = [("pcg_iters", C.c_int), ("converged", C.c_int), ("nan_flag", C.c_int),
                ("rel_residual", C.c_double), ("true_rel_residual", C.c_double), ("max_abs_div", C.c_double),
                ("body_force", C.c_double * 3), ("body_disp", C.c_double * 3), ("body_vel", C.c_double * 3),
                ("step", C.c_longlong), ("dt", C.c_double), ("time", C.c_double),
                ("coupling_iters", C.c_int), ("coupling_xi", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.POINTER(_Params)]
        L.orc_field_size.restype = C.c_longlong
        L.orc_delta_phi.restype = C.c_double
        L.orc_delta_phi.argtypes = [C.c_int, C.c_double]
        L.orc_inflow_rand.restype = C.c_double
        L.orc_inflow_rand.argtypes = [C.c_uint64, C.c_longlong, C.c_int, C.c_int, C.c_int]
        L.orc_wall_utau.restype = C.c_double
        L.orc_wall_utau.argtypes = [C.c_double] * 3
        L.orc_rk4_body.argtypes = [C.c_double] * 5 + [C.POINTER(C.c_double)] * 2
        L.orc_set_body.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_int]
        L.orc_set_history.argtypes = [C.c_void_p, C.c_int, C.c_longlong]
        L.orc_set_beam.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_int), C.c_double, C.c_double, C.c_double]
        L.orc_beam_ndof.argtypes = [C.c_void_p]
        L.orc_beam_matrices.argtypes = [C.c_void_p] + [C.POINTER(C.c_double)] * 4
        L.orc_get_beam_state.argtypes = [C.c_void_p] + [C.POINTER(C.c_double)] * 4
        L.orc_set_beam_state.argtypes = [C.c_void_p] + [C.POINTER(C.c_double)] * 3
        L.orc_beam_newmark.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.c_double]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def info_dict(i):
    return dict(pcg_iters=i.pcg_iters, converged=i.converged, nan_flag=i.nan_flag,
                rel_residual=i.rel_residual, true_rel_residual=i.true_rel_residual,
                max_abs_div=i.max_abs_div, body_force=list(i.body_force), body_disp=list(i.body_disp),
                body_vel=list(i.body_vel), step=i.step, dt=i.dt, time=i.time,
                coupling_iters=i.coupling_iters, coupling_xi=i.coupling_xi)


def delta_phi(kind, r):
    return lib().orc_delta_phi(DELTA[kind], float(r))


def inflow_rand(seed, step, face, a, b):
    return lib().orc_inflow_rand(int(seed), int(step), int(face), int(a), int(b))


def wall_utau(U, y, nu):
    return lib().orc_wall_utau(float(U), float(y), float(nu))


def rk4_body(m, c, k, F, dt, w, wd):
    a, b = C.c_double(w), C.c_double(wd)
    lib().orc_rk4_body(m, c, k, F, dt, C.byref(a), C.byref(b))
    return a.value, b.value


class Oracle:
    """One oracle simulation.  `cfg` is the plain dict produced by fs_workloads (keys = fs_params)."""

    def __init__(self, cfg):
        L = lib()
        P = _Params()
        for k in ("nx", "ny", "nz", "x0", "y0", "z0", "lx", "ly", "lz", "nu", "rho", "dt", "rtol",
                  "max_iter", "warm_start", "mg_nu1", "mg_nu2", "mg_coarse_sweeps", "mg_omega",
                  "seed", "inflow_noise"):
            setattr(P, k, cfg[k])
        self._yf = None
        if cfg.get("yf") is not None:
            self._yf = _f64(cfg["yf"])
            assert self._yf.size == cfg["ny"] + 1
            P.yf = _dp(self._yf)
        for f in range(6):
            P.bc[f] = BC[cfg["bc"][f]]
            for c in range(3):
                P.bc_vel[f][c] = cfg["bc_vel"][f][c]
        for c in range(3):
            P.body_force[c] = cfg["body_force"][c]
        P.time_scheme = TIME[cfg["time_scheme"]]
        P.precond = PC[cfg["precond"]]
        P.delta = DELTA[cfg["delta"]]
        P.convection = {"central": 0, "upwind": 1}[cfg.get("convection", "central")]
        P.cfl = float(cfg.get("cfl", 0.0))
        P.coupling_max_iters = int(cfg.get("coupling_max_iters", 1))
        P.coupling_tol = float(cfg.get("coupling_tol", 1e-5))
        P.cs = float(cfg.get("cs", 0.0))
        P.wall_model = int(cfg.get("wall_model", 0))
        self.h = L.orc_create(C.byref(P))
        if not self.h:
            raise ValueError("oracle: invalid parameters")
        self.h = C.c_void_p(self.h)
        self.nx, self.ny, self.nz = cfg["nx"], cfg["ny"], cfg["nz"]
        bx, by, bz = (cfg["bc"][0] != "periodic", cfg["bc"][2] != "periodic", cfg["bc"][4] != "periodic")
        self.shape = {"u": (self.nz, self.ny, self.nx + bx), "v": (self.nz, self.ny + by, self.nx),
                      "w": (self.nz + bz, self.ny, self.nx), "p": (self.nz, self.ny, self.nx)}
        for a, b in (("hu", "u"), ("hv", "v"), ("hw", "w"), ("div", "p")):
            self.shape[a] = self.shape[b]

    def __del__(self):
        if getattr(self, "h", None):
            lib().orc_destroy(self.h)
            self.h = None

    # ---- state -------------------------------------------------------------
    def set(self, name, arr):
        a = _f64(arr)
        assert a.shape == self.shape[name], (name, a.shape, self.shape[name])
        assert lib().orc_set_field(self.h, FIELD[name], _dp(a)) == 0

    def get(self, name):
        a = np.empty(self.shape[name], dtype=np.float64)
        assert lib().orc_get_field(self.h, FIELD[name], _dp(a)) == 0
        return a

    def set_history(self, have, step):
        lib().orc_set_history(self.h, int(have), int(step))

    def set_markers(self, xyz, vel=None, dvol=None):
        xyz = _f64(xyz).reshape(-1, 3)
        n = xyz.shape[0]
        v = _f64(vel).reshape(-1, 3) if vel is not None else None
        d = _f64(dvol).reshape(-1) if dvol is not None else None
        rc = lib().orc_set_markers(self.h, n, _dp(xyz), _dp(v) if v is not None else None,
                                   _dp(d) if d is not None else None)
        if rc == 2:
            raise ValueError("oracle: unsupported -- a marker support touches a non-periodic boundary")
        if rc:
            raise ValueError("oracle: set_markers failed")
        self.nl = n

    def set_solid_mask(self, eps_cells, uc=None):
        """eps-mask IBM (reading E1): eps_cells (nz, ny, nx) of 0/1, uc the solid's velocity."""
        if eps_cells is None:
            lib().orc_set_solid_mask(self.h, None, None)
            return
        e = np.ascontiguousarray(eps_cells, dtype=np.uint8)
        assert e.shape == self.shape["p"]
        u = _f64(uc if uc is not None else [0.0, 0.0, 0.0])
        rc = lib().orc_set_solid_mask(self.h, e.ctypes.data_as(C.POINTER(C.c_ubyte)), _dp(u))
        if rc:
            raise ValueError("oracle: set_solid_mask failed")

    def face_masks(self):
        m = [np.empty(self.shape[c], dtype=np.uint8) for c in "uvw"]
        lib().orc_get_face_masks(self.h, *[a.ctypes.data_as(C.POINTER(C.c_ubyte)) for a in m])
        return m

    def set_body(self, m, c, k, dof_mask):
        assert lib().orc_set_body(self.h, m, c, k, dof_mask) == 0

    # ---- flexible beam (Eq. 11, 13-17, Newmark-beta; reading N2-2) -------------
    def set_beam(self, node_xy, marker_node, EI, mu_s, zeta_s=0.0):
        xy = _f64(node_xy).reshape(-1, 2)
        mn = np.ascontiguousarray(marker_node, dtype=np.int32)
        assert mn.size == self.nl
        rc = lib().orc_set_beam(self.h, xy.shape[0], _dp(xy), _ip(mn), C.c_double(EI), C.c_double(mu_s), C.c_double(zeta_s))
        if rc:
            raise ValueError("oracle: set_beam failed")
        self.ndof = lib().orc_beam_ndof(self.h)

    def beam_matrices(self):
        n = self.ndof
        K, M, Cm, coef = np.empty((n, n)), np.empty((n, n)), np.empty((n, n)), np.empty(4)
        lib().orc_beam_matrices(self.h, _dp(K), _dp(M), _dp(Cm), _dp(coef))
        return K, M, Cm, dict(alpha=coef[0], beta=coef[1], omega1=coef[2], omega2=coef[3])

    def beam_state(self):
        n = self.ndof
        w, v, a, Q = np.empty(n), np.empty(n), np.empty(n), np.empty(n)
        lib().orc_get_beam_state(self.h, _dp(w), _dp(v), _dp(a), _dp(Q))
        return dict(w=w, v=v, a=a, Q=Q)

    def set_beam_state(self, w, v, a):
        lib().orc_set_beam_state(self.h, _dp(_f64(w)), _dp(_f64(v)), _dp(_f64(a)))

    def beam_newmark(self, Q, dt):
        lib().orc_beam_newmark(self.h, _dp(_f64(Q)), C.c_double(dt))

    def set_body_state(self, disp, vel):
        lib().orc_set_body_state(self.h, _dp(_f64(disp)), _dp(_f64(vel)))

    def body_state(self):
        d, v, f = np.zeros(3), np.zeros(3), np.zeros(3)
        lib().orc_get_body_state(self.h, _dp(d), _dp(v), _dp(f))
        return d, v, f

    def markers(self):
        n = lib().orc_marker_count(self.h)
        x, v, f = np.empty((n, 3)), np.empty((n, 3)), np.empty((n, 3))
        lib().orc_get_markers(self.h, _dp(x), _dp(v), _dp(f))
        return x, v, f

    # ---- the step ----------------------------------------------------------
    def step(self, nsteps=1):
        info = _Info()
        iters = np.zeros(nsteps, dtype=np.int32)
        rc = lib().orc_step(self.h, nsteps, C.byref(info), _ip(iters))
        if rc == 2:
            raise ValueError("oracle: unsupported -- a marker support touches a non-periodic boundary")
        d = info_dict(info)
        d["iters_per_step"] = iters.tolist()
        return d

    def poisson_solve(self, rhs, p0=None):
        rhs = _f64(rhs)
        p = _f64(p0).copy() if p0 is not None else np.zeros_like(rhs)
        info = _Info()
        lib().orc_poisson_solve(self.h, _dp(rhs), _dp(p), C.byref(info))
        return p, info_dict(info)

    # ---- pieces (for pins) ---------------------------------------------------
    def laplacian(self, p):
        p = _f64(p); out = np.empty_like(p)
        lib().orc_laplacian(self.h, _dp(p), _dp(out)); return out

    def apply_A(self, x):
        x = _f64(x); out = np.empty_like(x)
        lib().orc_apply_A(self.h, _dp(x), _dp(out)); return out

    def jacobi_diag(self):
        out = np.empty(self.shape["p"]); lib().orc_jacobi_diag(self.h, _dp(out)); return out

    def divergence(self, u, v, w):
        u, v, w = _f64(u), _f64(v), _f64(w); out = np.empty(self.shape["p"])
        lib().orc_divergence(self.h, _dp(u), _dp(v), _dp(w), _dp(out)); return out

    def gradient(self, p):
        p = _f64(p)
        g = [np.empty(self.shape[c]) for c in "uvw"]
        lib().orc_gradient(self.h, _dp(p), _dp(g[0]), _dp(g[1]), _dp(g[2])); return g

    def momentum_rhs(self):
        g = [np.empty(self.shape[c]) for c in "uvw"]
        lib().orc_momentum_rhs(self.h, _dp(g[0]), _dp(g[1]), _dp(g[2])); return g

    def predict(self, stage):
        """Predicted field without advancing the state: stage 0 after O3, 1 after O4 (IBM), 2 after O5."""
        g = [np.empty(self.shape[c]) for c in "uvw"]
        assert lib().orc_predict(self.h, int(stage), _dp(g[0]), _dp(g[1]), _dp(g[2])) == 0
        return g

    def eddy_viscosity(self):
        out = np.empty(self.shape["p"]); lib().orc_eddy_viscosity(self.h, _dp(out)); return out

    def convection(self):
        g = [np.empty(self.shape[c]) for c in "uvw"]
        lib().orc_convection(self.h, _dp(g[0]), _dp(g[1]), _dp(g[2])); return g

    def vcycle(self, r):
        r = _f64(r); z = np.empty_like(r)
        lib().orc_vcycle(self.h, _dp(r), _dp(z)); return z

    def cell_list(self):
        n = lib().orc_marker_count(self.h)
        base = np.empty((3, n, 3), dtype=np.int32); perm = np.empty(n, dtype=np.int32)
        keys = np.empty(n, dtype=np.int32); seg = np.empty(n + 1, dtype=np.int32); ns = C.c_int(0)
        lib().orc_get_cell_list(self.h, _ip(base), _ip(perm), _ip(keys), _ip(seg), C.byref(ns))
        return dict(base=base, perm=perm, keys=keys, seg_start=seg[:ns.value + 1].copy(), nseg=ns.value)

    def interpolate(self, u, v, w):
        n = lib().orc_marker_count(self.h)
        u, v, w = _f64(u), _f64(v), _f64(w); out = np.empty((n, 3))
        lib().orc_interpolate(self.h, _dp(u), _dp(v), _dp(w), _dp(out)); return out

    def spread(self, F):
        F = _f64(F)
        g = [np.zeros(self.shape[c]) for c in "uvw"]
        lib().orc_spread(self.h, _dp(F), _dp(g[0]), _dp(g[1]), _dp(g[2])); return g
