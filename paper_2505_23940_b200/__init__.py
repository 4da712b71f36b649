"""Thin Python binding of libfs (include/fs.h): argument marshalling only.

Every step of the fractional-step path (section 2.3.1, Eq. 3-10, 12) runs in the CUDA
kernels of paper_2505_23940_b200/csrc; this module converts Python values to the C ABI's plain
pointers and sizes.  PyTorch is used for exactly two things: the device workspace (one uint8 tensor)
and the CUDA stream handle.  There is no CPU fallback: if libfs.so is missing, importing the entry
points raises.  This package never imports oracle/.

    from paper_2505_23940_b200 import Grid
    g = Grid(cfg)                 # cfg: dict with the keys of fs_params (see fs_workloads)
    g.set("u", u0); g.step(10); u = g.get("u")
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfs.so")

FS_OK = 0
STATUS = {0: "FS_OK", 1: "FS_ERR_INVALID_ARG", 2: "FS_ERR_BAD_STATE", 3: "FS_ERR_OOM", 4: "FS_ERR_CUDA",
          5: "FS_ERR_NOT_CONVERGED", 6: "FS_ERR_UNSUPPORTED"}
FS_ERR_NOT_CONVERGED = 5
FS_ERR_UNSUPPORTED = 6
DTYPE = {"f32": 0, "f64": 1}
BC = {"periodic": 0, "noslip": 1, "slip": 2, "inflow": 3, "outflow": 4}
TIME = {"euler": 0, "ab2": 1, "rk3": 2}
PC = {"none": 0, "jacobi": 1, "gmg": 2}
DELTA = {"roma3": 0, "peskin4": 1}
EXEC = {"graph": 0, "stream": 1}
FIELD = {"u": 0, "v": 1, "w": 2, "p": 3, "hu": 4, "hv": 5, "hw": 6, "div": 7,
         "marker_x": 8, "marker_u": 9, "marker_f": 10, "marker_base": 11, "marker_perm": 12,
         "marker_keys": 13, "marker_seg": 14, "body_state": 15, "mask_u": 16, "mask_v": 17, "mask_w": 18}
_INT_FIELDS = ("marker_base", "marker_perm", "marker_keys", "marker_seg")
_BYTE_FIELDS = {"mask_u": "u", "mask_v": "v", "mask_w": "w"}


class fs_params(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("x0", C.c_double), ("y0", C.c_double), ("z0", C.c_double),
                ("lx", C.c_double), ("ly", C.c_double), ("lz", C.c_double),
                ("yf", C.POINTER(C.c_double)),
                ("dtype", C.c_int),
                ("bc", C.c_int * 6), ("bc_vel", (C.c_double * 3) * 6),
                ("nu", C.c_double), ("rho", C.c_double), ("dt", C.c_double), ("body_force", C.c_double * 3),
                ("time_scheme", C.c_int),
                ("precond", C.c_int), ("rtol", C.c_double), ("max_iter", C.c_int), ("warm_start", C.c_int),
                ("mg_nu1", C.c_int), ("mg_nu2", C.c_int), ("mg_coarse_sweeps", C.c_int), ("mg_omega", C.c_double),
                ("delta", C.c_int), ("max_markers", C.c_int),
                ("seed", C.c_uint64), ("inflow_noise", C.c_double),
                ("exec_mode", C.c_int), ("convection", C.c_int), ("solid_mask", C.c_int), ("cs", C.c_double), ("wall_model", C.c_int),
                ("coupling_max_iters", C.c_int), ("coupling_tol", C.c_double), ("cfl", C.c_double),
                ("max_beam_nodes", C.c_int)]


class fs_step_info(C.Structure):
    _fields_ = [("pcg_iters", C.c_int), ("converged", C.c_int), ("nan_flag", C.c_int),
                ("rel_residual", C.c_double), ("true_rel_residual", C.c_double), ("max_abs_div", C.c_double),
                ("body_force", C.c_double * 3), ("body_disp", C.c_double * 3), ("body_vel", C.c_double * 3),
                ("step", C.c_longlong), ("unconverged_steps", C.c_longlong), ("nan_steps", C.c_longlong),
                ("dt", C.c_double), ("time", C.c_double), ("coupling_iters", C.c_int), ("coupling_xi", C.c_double)]


class fs_poisson_info(C.Structure):
    _fields_ = [("iters", C.c_int), ("converged", C.c_int),
                ("rel_residual", C.c_double), ("true_rel_residual", C.c_double)]


# every symbol include/*.h declares (tests check the library exports all of them)
SYMBOLS = ("fs_divergence_noalloc", "fs_workspace_bytes", "fs_grid_create", "fs_grid_destroy", "fs_field_size", "fs_fields_set",
           "fs_fields_get", "fs_fields_set_async", "fs_fields_get_async", "fs_set_history", "fs_set_ibm_markers", "fs_marker_segments", "fs_set_body", "fs_set_solid_mask", "fs_set_beam", "fs_beam_state",
           "fs_set_body_state", "fs_step", "fs_poisson_solve", "fs_ibm_interpolate", "fs_ibm_spread",
           "fs_gmg_vcycle", "fs_momentum_rhs", "fs_profile_step", "fs_profile_count", "fs_profile_entry",
           "fs_profile_reset", "fs_launch_count", "fs_kernels_used", "fs_status_string")

_lib = None


class FsError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        super().__init__("%s failed: %s" % (where, STATUS.get(status, status)))


def lib():
    """Loads libfs.so (built in-tree by paper_2505_23940_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libfs.so not built: run `python -m paper_2505_23940_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, ip, dp = C.c_void_p, C.c_int, C.POINTER(C.c_double)
        L.fs_workspace_bytes.argtypes = [C.POINTER(fs_params), C.POINTER(C.c_size_t)]
        L.fs_grid_create.argtypes = [C.POINTER(fs_params), vp, C.c_size_t, vp, C.POINTER(vp)]
        L.fs_grid_destroy.argtypes = [vp]
        L.fs_field_size.argtypes = [vp, ip, C.POINTER(C.c_longlong)]
        L.fs_fields_set.argtypes = [vp, ip, vp, ip, ip]
        L.fs_fields_get.argtypes = [vp, ip, vp, ip, ip]
        L.fs_fields_set_async.argtypes = [vp, ip, vp]
        L.fs_fields_get_async.argtypes = [vp, ip, vp]
        L.fs_set_history.argtypes = [vp, ip, C.c_longlong]
        L.fs_set_ibm_markers.argtypes = [vp, ip, dp, dp, dp]
        L.fs_marker_segments.argtypes = [vp, C.POINTER(C.c_int)]
        L.fs_set_body.argtypes = [vp, C.c_double, C.c_double, C.c_double, ip]
        L.fs_set_body_state.argtypes = [vp, dp, dp]
        L.fs_set_solid_mask.argtypes = [vp, C.POINTER(C.c_ubyte), dp]
        L.fs_set_beam.argtypes = [vp, C.c_int, dp, C.POINTER(C.c_int), C.c_double, C.c_double, C.c_double]
        L.fs_beam_state.argtypes = [vp, dp, dp, dp, dp, dp]
        L.fs_step.argtypes = [vp, ip, C.POINTER(fs_step_info)]
        L.fs_poisson_solve.argtypes = [vp, vp, vp, ip, ip, C.POINTER(fs_poisson_info)]
        L.fs_ibm_interpolate.argtypes = [vp, dp]
        L.fs_ibm_spread.argtypes = [vp, dp]
        L.fs_gmg_vcycle.argtypes = [vp, dp, dp]
        L.fs_momentum_rhs.argtypes = [vp]
        L.fs_profile_step.argtypes = [vp, ip]
        L.fs_profile_count.argtypes = [vp, C.POINTER(C.c_int)]
        L.fs_profile_entry.argtypes = [vp, ip, C.POINTER(C.c_char_p), C.POINTER(C.c_longlong),
                                       C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.fs_profile_reset.argtypes = [vp]
        L.fs_launch_count.argtypes = [vp, C.POINTER(C.c_longlong)]
        L.fs_kernels_used.argtypes = [vp, C.c_char_p, C.c_size_t, C.POINTER(C.c_size_t)]
        L.fs_divergence_noalloc.argtypes = [ip, ip, ip, C.c_double, C.c_double, C.c_double, ip, vp, vp, vp, vp, vp, vp]
        L.fs_status_string.argtypes = [ip]
        L.fs_status_string.restype = C.c_char_p
        for s in SYMBOLS:
            if s != "fs_status_string":
                getattr(L, s).restype = C.c_int
        _lib = L
    return _lib


def _check(st, where, allow=()):
    if st != FS_OK and st not in allow:
        raise FsError(st, where)
    return st


def make_params(cfg):
    """dict (keys of fs_params, enums as strings) -> (fs_params, keep-alive objects)."""
    P = fs_params()
    for k in ("nx", "ny", "nz", "x0", "y0", "z0", "lx", "ly", "lz", "nu", "rho", "dt", "rtol", "max_iter",
              "warm_start", "mg_nu1", "mg_nu2", "mg_coarse_sweeps", "mg_omega", "seed", "inflow_noise",
              "max_markers"):
        setattr(P, k, cfg[k])
    keep = None
    if cfg.get("yf") is not None:
        keep = np.ascontiguousarray(cfg["yf"], dtype=np.float64)
        if keep.size != cfg["ny"] + 1:
            raise ValueError("yf must have ny+1 entries")
        P.yf = keep.ctypes.data_as(C.POINTER(C.c_double))
    P.dtype = DTYPE[cfg.get("dtype", "f64")]
    for f in range(6):
        P.bc[f] = BC[cfg["bc"][f]]
        for c in range(3):
            P.bc_vel[f][c] = cfg["bc_vel"][f][c]
    for c in range(3):
        P.body_force[c] = cfg["body_force"][c]
    P.time_scheme = TIME[cfg["time_scheme"]]
    P.precond = PC[cfg["precond"]]
    P.delta = DELTA[cfg["delta"]]
    P.exec_mode = EXEC[cfg.get("exec_mode", "graph")]
    P.convection = {"central": 0, "upwind": 1}[cfg.get("convection", "central")]
    P.solid_mask = int(cfg.get("solid_mask", 0))
    P.cfl = float(cfg.get("cfl", 0.0))
    P.max_beam_nodes = int(cfg.get("max_beam_nodes", len(cfg["beam"][0]) if cfg.get("beam") is not None else 0))
    P.coupling_max_iters = int(cfg.get("coupling_max_iters", 1))
    P.coupling_tol = float(cfg.get("coupling_tol", 1e-5))
    P.cs = float(cfg.get("cs", 0.0))
    P.wall_model = int(cfg.get("wall_model", 0))
    return P, keep


def _info_dict(i):
    return dict(pcg_iters=i.pcg_iters, converged=i.converged, nan_flag=i.nan_flag,
                rel_residual=i.rel_residual, true_rel_residual=i.true_rel_residual,
                max_abs_div=i.max_abs_div, body_force=list(i.body_force), body_disp=list(i.body_disp),
                body_vel=list(i.body_vel), step=i.step, unconverged_steps=i.unconverged_steps, nan_steps=i.nan_steps,
                dt=i.dt, time=i.time, coupling_iters=i.coupling_iters, coupling_xi=i.coupling_xi)


class Grid:
    """One fs_grid.  Owns the torch workspace tensor; everything else is a C-ABI call."""

    def __init__(self, cfg, device="cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2505_23940_b200 needs a CUDA device (no CPU fallback)")
        L = lib()
        self._torch = torch
        self.cfg = cfg
        self.device = torch.device(device)
        self.P, self._keep = make_params(cfg)
        nbytes = C.c_size_t(0)
        _check(L.fs_workspace_bytes(C.byref(self.P), C.byref(nbytes)), "fs_workspace_bytes")
        self.workspace_bytes = nbytes.value
        torch.cuda.set_device(self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.workspace = torch.empty(nbytes.value, dtype=torch.uint8, device=self.device)
        h = C.c_void_p()
        _check(L.fs_grid_create(C.byref(self.P), C.c_void_p(self.workspace.data_ptr()), nbytes.value,
                                C.c_void_p(self.stream.cuda_stream), C.byref(h)), "fs_grid_create")
        self.h = h
        self.f64 = cfg.get("dtype", "f64") == "f64"
        nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
        bx, by, bz = (cfg["bc"][0] != "periodic", cfg["bc"][2] != "periodic", cfg["bc"][4] != "periodic")
        self.shape = {"u": (nz, ny, nx + bx), "v": (nz, ny + by, nx), "w": (nz + bz, ny, nx), "p": (nz, ny, nx)}
        for a, b in (("hu", "u"), ("hv", "v"), ("hw", "w"), ("div", "p")):
            self.shape[a] = self.shape[b]
        self.n_markers = 0

    def close(self):
        if getattr(self, "h", None):
            lib().fs_grid_destroy(self.h)
            self.h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- fields ------------------------------------------------------------------------------------
    def field_size(self, name):
        n = C.c_longlong(0)
        _check(lib().fs_field_size(self.h, FIELD[name], C.byref(n)), "fs_field_size")
        return n.value

    def set(self, name, arr):
        """Host numpy array or device torch tensor (fp32/fp64) -> field."""
        torch = self._torch
        if isinstance(arr, torch.Tensor) and arr.is_cuda:
            a = arr.contiguous()
            assert a.dtype in (torch.float32, torch.float64)
            assert a.numel() == self.field_size(name), (name, a.shape)
            dt = DTYPE["f64" if a.dtype == torch.float64 else "f32"]
            _check(lib().fs_fields_set(self.h, FIELD[name], C.c_void_p(a.data_ptr()), dt, 1), "fs_fields_set")
            return
        a = np.asarray(arr)
        if a.dtype != np.float32:
            a = a.astype(np.float64, copy=False)
        a = np.ascontiguousarray(a)
        assert a.size == self.field_size(name), (name, a.shape, self.field_size(name))
        dt = DTYPE["f64" if a.dtype == np.float64 else "f32"]
        _check(lib().fs_fields_set(self.h, FIELD[name], C.c_void_p(a.ctypes.data), dt, 0), "fs_fields_set")

    def get(self, name, dtype="f64", out=None):
        """Field -> host numpy array (or into a device torch tensor `out`)."""
        torch = self._torch
        n = self.field_size(name)
        if out is not None and isinstance(out, torch.Tensor) and out.is_cuda:
            assert out.is_contiguous() and out.numel() == n
            dt = DTYPE["f64" if out.dtype == torch.float64 else "f32"]
            _check(lib().fs_fields_get(self.h, FIELD[name], C.c_void_p(out.data_ptr()), dt, 1), "fs_fields_get")
            return out
        if name in _BYTE_FIELDS:
            a = np.empty(n, dtype=np.uint8)
            _check(lib().fs_fields_get(self.h, FIELD[name], C.c_void_p(a.ctypes.data), DTYPE[dtype], 0), "fs_fields_get")
            return a.reshape(self.shape[_BYTE_FIELDS[name]])
        if name in _INT_FIELDS:
            a = np.empty(n, dtype=np.int32)
        else:
            a = np.empty(n, dtype=np.float64 if dtype == "f64" else np.float32) if out is None else out
        _check(lib().fs_fields_get(self.h, FIELD[name], C.c_void_p(a.ctypes.data), DTYPE[dtype], 0), "fs_fields_get")
        if name in self.shape:
            return a.reshape(self.shape[name])
        if name in ("marker_x", "marker_u", "marker_f"):
            return a.reshape(-1, 3)
        if name == "marker_base":
            return a.reshape(3, -1, 3)
        return a

    def set_async(self, name, host):
        """fs_fields_set_async: enqueue host (pinned torch tensor or numpy array of the grid's dtype) -> field on the grid's stream."""
        ptr = host.data_ptr() if isinstance(host, self._torch.Tensor) else host.ctypes.data
        _check(lib().fs_fields_set_async(self.h, FIELD[name], C.c_void_p(ptr)), "fs_fields_set_async")

    def get_async(self, name, host):
        """fs_fields_get_async: enqueue field -> host buffer on the grid's stream (valid after the stream is synchronised)."""
        ptr = host.data_ptr() if isinstance(host, self._torch.Tensor) else host.ctypes.data
        _check(lib().fs_fields_get_async(self.h, FIELD[name], C.c_void_p(ptr)), "fs_fields_get_async")

    def set_history(self, have, step):
        _check(lib().fs_set_history(self.h, int(have), int(step)), "fs_set_history")

    # ---- markers / body ------------------------------------------------------------------------------
    def set_markers(self, xyz, vel=None, dvol=None):
        dp = C.POINTER(C.c_double)
        xyz = np.ascontiguousarray(xyz, dtype=np.float64).reshape(-1, 3)
        n = xyz.shape[0]
        v = np.ascontiguousarray(vel, dtype=np.float64).reshape(-1, 3) if vel is not None else None
        d = np.ascontiguousarray(dvol, dtype=np.float64).reshape(-1) if dvol is not None else None
        _check(lib().fs_set_ibm_markers(self.h, n, xyz.ctypes.data_as(dp),
                                        v.ctypes.data_as(dp) if v is not None else None,
                                        d.ctypes.data_as(dp) if d is not None else None), "fs_set_ibm_markers")
        self.n_markers = n

    def cell_list(self):
        ns = C.c_int(0)
        _check(lib().fs_marker_segments(self.h, C.byref(ns)), "fs_marker_segments")
        seg = self.get("marker_seg")
        return dict(base=self.get("marker_base"), perm=self.get("marker_perm"), keys=self.get("marker_keys"),
                    seg_start=seg[:ns.value + 1].copy(), nseg=ns.value)

    def set_solid_mask(self, eps_cells, uc=None):
        """fs_set_solid_mask: eps_cells (nz, ny, nx) of 0/1 (None: back to marker forcing), uc the solid's velocity."""
        if eps_cells is None:
            _check(lib().fs_set_solid_mask(self.h, None, None), "fs_set_solid_mask")
            return
        e = np.ascontiguousarray(eps_cells, dtype=np.uint8)
        assert e.shape == self.shape["p"]
        u = np.ascontiguousarray(uc if uc is not None else [0.0, 0.0, 0.0], dtype=np.float64)
        _check(lib().fs_set_solid_mask(self.h, e.ctypes.data_as(C.POINTER(C.c_ubyte)), u.ctypes.data_as(C.POINTER(C.c_double))),
               "fs_set_solid_mask")

    def set_body(self, m, c, k, dof_mask):
        _check(lib().fs_set_body(self.h, m, c, k, dof_mask), "fs_set_body")

    def set_beam(self, node_xy, marker_node, EI, mu_s, zeta_s=0.0):
        """fs_set_beam: flexible Euler-Bernoulli beam (Eq. 13-17, Newmark-beta) riding on the current markers."""
        xy = np.ascontiguousarray(node_xy, dtype=np.float64).reshape(-1, 2)
        mn = np.ascontiguousarray(marker_node, dtype=np.int32)
        _check(lib().fs_set_beam(self.h, xy.shape[0], xy.ctypes.data_as(C.POINTER(C.c_double)), mn.ctypes.data_as(C.POINTER(C.c_int)),
                                 float(EI), float(mu_s), float(zeta_s)), "fs_set_beam")
        self.beam_ndof = 2 * (xy.shape[0] - 1)

    def beam_state(self):
        """fs_beam_state: dict(w, v, a, Q, alpha, beta, omega1, omega2)."""
        dp = C.POINTER(C.c_double)
        out = [np.empty(self.beam_ndof) for _ in range(4)] + [np.empty(4)]
        _check(lib().fs_beam_state(self.h, *[a.ctypes.data_as(dp) for a in out]), "fs_beam_state")
        return dict(w=out[0], v=out[1], a=out[2], Q=out[3], alpha=out[4][0], beta=out[4][1], omega1=out[4][2], omega2=out[4][3])

    def set_body_state(self, disp, vel):
        dp = C.POINTER(C.c_double)
        d = np.ascontiguousarray(disp, dtype=np.float64)
        v = np.ascontiguousarray(vel, dtype=np.float64)
        _check(lib().fs_set_body_state(self.h, d.ctypes.data_as(dp), v.ctypes.data_as(dp)), "fs_set_body_state")

    def body_state(self):
        a = self.get("body_state")
        return a[0:3].copy(), a[3:6].copy(), a[6:9].copy()

    # ---- the path --------------------------------------------------------------------------------------
    def step(self, nsteps=1, sync=True, per_step=False):
        """fs_step.  sync=False: asynchronous (returns None).  per_step: one call per step, collecting
        PCG iteration counts (for parity tests)."""
        L = lib()
        if not sync:
            _check(L.fs_step(self.h, nsteps, None), "fs_step")
            return None
        info = fs_step_info()
        if per_step:
            iters = []
            for _ in range(nsteps):
                _check(L.fs_step(self.h, 1, C.byref(info)), "fs_step", allow=(FS_ERR_NOT_CONVERGED,))
                iters.append(info.pcg_iters)
            d = _info_dict(info)
            d["iters_per_step"] = iters
            return d
        _check(L.fs_step(self.h, nsteps, C.byref(info)), "fs_step", allow=(FS_ERR_NOT_CONVERGED,))
        return _info_dict(info)

    def poisson_solve(self, rhs, p0=None):
        """Host fp64 arrays in and out (parity / pins); device tensors are solved in place."""
        torch = self._torch
        info = fs_poisson_info()
        if isinstance(rhs, torch.Tensor) and rhs.is_cuda:
            assert p0 is not None and p0.is_cuda and p0.dtype == rhs.dtype
            dt = DTYPE["f64" if rhs.dtype == torch.float64 else "f32"]
            st = lib().fs_poisson_solve(self.h, C.c_void_p(rhs.data_ptr()), C.c_void_p(p0.data_ptr()), dt, 1, C.byref(info))
            _check(st, "fs_poisson_solve", allow=(FS_ERR_NOT_CONVERGED,))
            return p0, dict(iters=info.iters, converged=info.converged, rel_residual=info.rel_residual,
                            true_rel_residual=info.true_rel_residual)
        r = np.ascontiguousarray(rhs, dtype=np.float64)
        p = np.ascontiguousarray(p0, dtype=np.float64).copy() if p0 is not None else np.zeros_like(r)
        st = lib().fs_poisson_solve(self.h, C.c_void_p(r.ctypes.data), C.c_void_p(p.ctypes.data), DTYPE["f64"], 0, C.byref(info))
        _check(st, "fs_poisson_solve", allow=(FS_ERR_NOT_CONVERGED,))
        return p, dict(iters=info.iters, converged=info.converged, rel_residual=info.rel_residual,
                       true_rel_residual=info.true_rel_residual)

    # ---- pieces exposed for element-wise parity ----------------------------------------------------------
    def ibm_interpolate(self):
        out = np.empty((self.n_markers, 3), dtype=np.float64)
        _check(lib().fs_ibm_interpolate(self.h, out.ctypes.data_as(C.POINTER(C.c_double))), "fs_ibm_interpolate")
        return out

    def ibm_spread(self, F):
        F = np.ascontiguousarray(F, dtype=np.float64)
        assert F.size == 3 * self.n_markers
        _check(lib().fs_ibm_spread(self.h, F.ctypes.data_as(C.POINTER(C.c_double))), "fs_ibm_spread")

    def gmg_vcycle(self, r):
        r = np.ascontiguousarray(r, dtype=np.float64)
        z = np.empty_like(r)
        dp = C.POINTER(C.c_double)
        _check(lib().fs_gmg_vcycle(self.h, r.ctypes.data_as(dp), z.ctypes.data_as(dp)), "fs_gmg_vcycle")
        return z

    def momentum_rhs(self):
        """H^n of the current u,v,w into hu,hv,hw (S1 kernel alone; u,v,w untouched)."""
        _check(lib().fs_momentum_rhs(self.h), "fs_momentum_rhs")
        return [self.get(c) for c in ("hu", "hv", "hw")]

    def profile_step(self, nsteps=1, reset=True):
        """fs_profile_step: per-kernel {name: dict(launches, ms, bytes)} over nsteps event-timed steps."""
        L = lib()
        if reset:
            _check(L.fs_profile_reset(self.h), "fs_profile_reset")
        _check(L.fs_profile_step(self.h, nsteps), "fs_profile_step")
        n = C.c_int(0)
        _check(L.fs_profile_count(self.h, C.byref(n)), "fs_profile_count")
        out = {}
        for i in range(n.value):
            name, cnt, ms, by = C.c_char_p(), C.c_longlong(0), C.c_double(0), C.c_double(0)
            _check(L.fs_profile_entry(self.h, i, C.byref(name), C.byref(cnt), C.byref(ms), C.byref(by)), "fs_profile_entry")
            out[name.value.decode()] = dict(launches=cnt.value, ms=ms.value, bytes=by.value)
        return out

    def kernels_used(self):
        """Names of the kernel instantiations this grid has enqueued so far (fs_kernels_used)."""
        need = C.c_size_t(0)
        _check(lib().fs_kernels_used(self.h, None, 0, C.byref(need)), "fs_kernels_used")
        buf = C.create_string_buffer(need.value)
        _check(lib().fs_kernels_used(self.h, buf, need.value, None), "fs_kernels_used")
        return [x for x in buf.value.decode().split(";") if x]

    def launch_count(self):
        n = C.c_longlong(0)
        _check(lib().fs_launch_count(self.h, C.byref(n)), "fs_launch_count")
        return n.value


def from_workload(cfg, device="cuda:0", stream=None, **overrides):
    """Grid initialised from an fs_workloads config: fields, markers and body set through the C ABI."""
    c = dict(cfg)
    c.update(overrides)
    g = Grid(c, device=device, stream=stream)
    for name, arr in c.get("init", {}).items():
        g.set(name, arr)
    if c.get("markers") is not None:
        g.set_markers(*c["markers"])
    if c.get("body") is not None:
        g.set_body(*c["body"])
    if c.get("mask") is not None:
        g.set_solid_mask(*c["mask"])
    if c.get("beam") is not None:
        g.set_beam(*c["beam"])
    return g


NOALLOC_MAX_CELLS = 16777216     # FS_NOALLOC_MAX_CELLS (include/fs_noalloc.h)


def divergence_noalloc(u, v, w, h, div_out=None, result=None, stream=None):
    """fs_divergence_noalloc (include/fs_noalloc.h): divergence of a triply periodic staggered field given as CUDA tensors
    of shape (nz, ny, nx), its max norm and squared 2-norm into `result` (2 fp64 words on the device).  The library call
    allocates nothing (its scratch is a static device array: calls that overlap on the GPU race); this wrapper only
    marshals: pass div_out / result to keep it allocation-free, else it creates them with torch.  Asynchronous."""
    import torch
    assert u.is_cuda and u.is_contiguous() and v.is_contiguous() and w.is_contiguous() and u.shape == v.shape == w.shape and u.dtype == v.dtype == w.dtype
    nz, ny, nx = u.shape
    dt = {torch.float32: DTYPE["f32"], torch.float64: DTYPE["f64"]}[u.dtype]
    if result is None:
        result = torch.empty(2, dtype=torch.float64, device=u.device)
    hx, hy, hz = (h, h, h) if np.isscalar(h) else h
    with torch.cuda.device(u.device):
        s = stream if stream is not None else torch.cuda.current_stream().cuda_stream
        _check(lib().fs_divergence_noalloc(nx, ny, nz, hx, hy, hz, dt, u.data_ptr(), v.data_ptr(), w.data_ptr(),
                                           div_out.data_ptr() if div_out is not None else None, result.data_ptr(), s),
               "fs_divergence_noalloc")
    return result
