"""Seeded synthetic workloads c1..c5 (BASELINE.json `configs`; recipe in DESIGN.md "Input recipe").

This module is shared by the oracle tests and by the CUDA path's tests / bench.  It holds
none of the method's arithmetic: it only produces parameters, initial fields and marker sets.
The workloads stand in for the paper's literature benchmarks (section 3: channel
Re_tau=180 L576-582, cylinder / VIV cases L472-501, finite cylinder L630-634, HIT L730-732),
whose reference data are not reproduced here.
"""
import math

import numpy as np

DEFAULTS = dict(
    x0=0.0, y0=0.0, z0=0.0, yf=None,
    bc=["periodic"] * 6, bc_vel=[[0.0, 0.0, 0.0] for _ in range(6)],
    rho=1.0, body_force=[0.0, 0.0, 0.0],
    time_scheme="ab2", precond="jacobi", rtol=1e-10, max_iter=20000, warm_start=1,
    mg_nu1=2, mg_nu2=2, mg_coarse_sweeps=16, mg_omega=6.0 / 7.0,
    delta="roma3", seed=0, inflow_noise=0.0, max_markers=0, dtype="f64",
)


def _base(**kw):
    cfg = {k: (v.copy() if isinstance(v, list) else v) for k, v in DEFAULTS.items()}
    cfg["bc_vel"] = [[0.0, 0.0, 0.0] for _ in range(6)]
    cfg.update(kw)
    return cfg


def shapes(cfg):
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    bx, by, bz = (cfg["bc"][0] != "periodic", cfg["bc"][2] != "periodic", cfg["bc"][4] != "periodic")
    return {"u": (nz, ny, nx + bx), "v": (nz, ny + by, nx), "w": (nz + bz, ny, nx), "p": (nz, ny, nx)}


def coords(cfg):
    """Face and centre coordinates per direction (yf may be stretched)."""
    out = {}
    for d, (n, o, l) in enumerate(((cfg["nx"], cfg["x0"], cfg["lx"]), (cfg["ny"], cfg["y0"], cfg["ly"]),
                                    (cfg["nz"], cfg["z0"], cfg["lz"]))):
        f = o + (l / n) * np.arange(n + 1)
        if d == 1 and cfg.get("yf") is not None:
            f = np.asarray(cfg["yf"], dtype=np.float64)
        out["xyz"[d] + "f"] = f
        out["xyz"[d] + "c"] = 0.5 * (f[:-1] + f[1:])
    return out


# ---------------------------------------------------------------- c1: Taylor-Green vortex
def taylor_green(n=32, **kw):
    L = 2.0 * math.pi
    cfg = _base(name="c1_taylor_green", nx=n, ny=n, nz=n, lx=L, ly=L, lz=L, nu=0.01, dt=1e-3,
                rtol=1e-12, steps=10)
    cfg.update(kw)
    c = coords(cfg)
    xf, xc, yf, yc = c["xf"][:-1], c["xc"], c["yf"][:-1], c["yc"]
    u = np.sin(xf)[None, None, :] * np.cos(yc)[None, :, None] * np.ones((n, 1, 1))
    v = -np.cos(xc)[None, None, :] * np.sin(yf)[None, :, None] * np.ones((n, 1, 1))
    cfg["init"] = {"u": u, "v": v, "w": np.zeros((n, n, n))}
    return cfg


# ---------------------------------------------------------------- c2: turbulent-channel-shaped
def channel(n=128, beta=2.0, seed=12345, **kw):
    j = np.arange(n + 1)
    yf = np.tanh(beta * (2.0 * j / n - 1.0)) / math.tanh(beta)
    yf[0], yf[-1] = -1.0, 1.0
    cfg = _base(name="c2_channel", nx=n, ny=n, nz=n, lx=2 * math.pi, ly=2.0, lz=math.pi, y0=-1.0, yf=yf,
                nu=1.0 / 180.0, dt=2e-4, body_force=[1.0, 0.0, 0.0], steps=20, seed=seed)
    cfg["bc"] = ["periodic", "periodic", "noslip", "noslip", "periodic", "periodic"]
    cfg.update(kw)
    c = coords(cfg)
    sh = shapes(cfg)
    rng = np.random.Generator(np.random.Philox(key=seed))
    amp = 0.5 / cfg["nu"]                                  # g/(2 nu) = 90 for nu = 1/180
    prof_c = amp * (1.0 - c["yc"] ** 2)
    prof_f = amp * (1.0 - c["yf"] ** 2)
    u = prof_c[None, :, None] * (1.0 + 0.1 * (2.0 * rng.random(sh["u"]) - 1.0))
    v = prof_f[None, :, None] * 0.1 * (2.0 * rng.random(sh["v"]) - 1.0)
    w = prof_c[None, :, None] * 0.1 * (2.0 * rng.random(sh["w"]) - 1.0)
    v[:, 0, :] = 0.0
    v[:, -1, :] = 0.0
    cfg["init"] = {"u": u, "v": v, "w": w}
    return cfg


# ---------------------------------------------------------------- c3: fixed sphere
def fibonacci_sphere(n, radius, centre):
    i = np.arange(n) + 0.5
    z = 1.0 - 2.0 * i / n
    r = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    phi = i * math.pi * (3.0 - math.sqrt(5.0))
    pts = np.stack([r * np.cos(phi), r * np.sin(phi), z], axis=1) * radius
    return pts + np.asarray(centre)[None, :]


def sphere(scale=1, n_markers=None, **kw):
    """scale=1 is the full config (256x128x128, h=1/16); scale=2,4 shrink the box for quick parity."""
    nx, ny, nz = 256 // scale, 128 // scale, 128 // scale
    h = 1.0 / 16.0
    lx, ly, lz = nx * h, ny * h, nz * h
    cfg = _base(name="c3_sphere", nx=nx, ny=ny, nz=nz, lx=lx, ly=ly, lz=lz, nu=1.0 / 300.0, dt=5e-3, steps=20)
    cfg["bc"] = ["inflow", "outflow", "slip", "slip", "slip", "slip"]
    cfg["bc_vel"][0] = [1.0, 0.0, 0.0]
    cfg["bc_vel"][1] = [1.0, 0.0, 0.0]        # convective speed U_c
    cfg.update(kw)
    sh = shapes(cfg)
    cfg["init"] = {"u": np.ones(sh["u"]), "v": np.zeros(sh["v"]), "w": np.zeros(sh["w"])}
    D = 1.0
    nm = n_markers if n_markers is not None else 3200
    centre = (lx / 4.0, ly / 2.0, lz / 2.0)
    xyz = fibonacci_sphere(nm, D / 2.0, centre)
    dvol = np.full(nm, math.pi * D * D * h / nm)
    cfg["markers"] = (xyz, np.zeros_like(xyz), dvol)
    cfg["max_markers"] = nm
    return cfg


# ---------------------------------------------------------------- c4: elastically mounted cylinder
def cylinder_fsi(scale=1, per_ring=75, **kw):
    nx, ny, nz = 384 // scale, 256 // scale, 32
    h = 1.0 / 16.0
    lx, ly, lz = nx * h, ny * h, nz * h
    cfg = _base(name="c4_cylinder_fsi", nx=nx, ny=ny, nz=nz, lx=lx, ly=ly, lz=lz, nu=1.0 / 150.0, dt=5e-3,
                steps=50, seed=2024, inflow_noise=0.01)
    cfg["bc"] = ["inflow", "outflow", "slip", "slip", "periodic", "periodic"]
    cfg["bc_vel"][0] = [1.0, 0.0, 0.0]
    cfg["bc_vel"][1] = [1.0, 0.0, 0.0]
    cfg.update(kw)
    sh = shapes(cfg)
    cfg["init"] = {"u": np.ones(sh["u"]), "v": np.zeros(sh["v"]), "w": np.zeros(sh["w"])}
    D = 1.0
    cx, cy = lx / 3.0, ly / 2.0
    th = 2.0 * math.pi * np.arange(per_ring) / per_ring
    zc = (np.arange(nz) + 0.5) * h
    ring = np.stack([cx + 0.5 * D * np.cos(th), cy + 0.5 * D * np.sin(th)], axis=1)
    xyz = np.concatenate([np.concatenate([ring, np.full((per_ring, 1), z)], axis=1) for z in zc], axis=0)
    nm = xyz.shape[0]
    dvol = np.full(nm, math.pi * D * lz * h / nm)
    cfg["markers"] = (xyz, np.zeros_like(xyz), dvol)
    cfg["max_markers"] = nm
    m = 2.0 * 1.0 * math.pi * D * D / 4.0 * lz       # mass ratio 2
    fn = 1.0 / (5.0 * D)                             # reduced velocity 5
    cfg["body"] = (m, 0.0, m * (2.0 * math.pi * fn) ** 2, 2)   # dof mask: y only
    return cfg


# ---------------------------------------------------------------- flexible plate (third item)
def flexible_plate(scale=4, nodes=17, length=1.0, mass_ratio=10.0, ei=0.5, zeta=0.02, **kw):
    """A flexible plate clamped at its lower end in a cross flow, spanning the periodic z direction: the shape of the
    paper's wall-mounted flexible plate (section 3.3.1) on the c4 box.  `nodes` beam nodes along y,
    one marker per node and span plane; cfg["beam"] = (node_xy, marker_node, EI, mu_s, zeta_s) for set_beam."""
    nx, ny, nz = 384 // scale, 256 // scale, 32 // max(1, scale // 2)
    h = 1.0 / 16.0
    lx, ly, lz = nx * h, ny * h, nz * h
    cfg = _base(name="flexible_plate", nx=nx, ny=ny, nz=nz, lx=lx, ly=ly, lz=lz, nu=1.0 / 150.0, dt=5e-3, steps=20)
    cfg["bc"] = ["inflow", "outflow", "slip", "slip", "periodic", "periodic"]
    cfg["bc_vel"][0] = [1.0, 0.0, 0.0]
    cfg["bc_vel"][1] = [1.0, 0.0, 0.0]
    cfg.update(kw)
    sh = shapes(cfg)
    cfg["init"] = {"u": np.ones(sh["u"]), "v": np.zeros(sh["v"]), "w": np.zeros(sh["w"])}
    xp, y0 = lx / 3.0 + 0.013, 0.5 * (ly - length) + 0.007       # off the grid lines
    s = np.linspace(0.0, length, nodes)
    node_xy = np.stack([np.full(nodes, xp), y0 + s], axis=1)
    zc = (np.arange(nz) + 0.5) * h
    xyz = np.array([[node_xy[i, 0], node_xy[i, 1], z] for z in zc for i in range(nodes)])
    marker_node = np.array([i for _ in zc for i in range(nodes)], dtype=np.int32)
    ds = length / (nodes - 1)
    dvol = np.full(xyz.shape[0], ds * h * h)                    # shell of one grid spacing (L185)
    cfg["markers"] = (xyz, np.zeros_like(xyz), dvol)
    cfg["max_markers"] = xyz.shape[0]
    cfg["beam"] = (node_xy, marker_node, ei, mass_ratio * h * lz, zeta)   # mu_s = density ratio x thickness h x span
    return cfg


# ---------------------------------------------------------------- c5: decaying HIT
def hit(n=512, seed=777, dtype="f64", device="cpu", **kw):
    """Random-phase solenoidal field, E(k) ~ k^4 exp(-2 (k/4)^2), u_rms = 1.

    Harness-only spectral construction (torch FFT); the exact *discrete* projection with the
    staggered-grid modified wavenumbers makes the field solenoidal to rounding.
    """
    import torch
    L = 2.0 * math.pi
    cfg = _base(name="c5_hit", nx=n, ny=n, nz=n, lx=L, ly=L, lz=L, nu=1e-3, dt=5e-4, precond="gmg",
                rtol=1e-8, max_iter=200, steps=10, seed=seed, dtype=dtype)
    cfg.update(kw)
    h = L / n
    g = torch.Generator(device="cpu")
    g.manual_seed(seed)
    dev = torch.device(device)
    k1 = torch.fft.fftfreq(n, d=1.0 / n, dtype=torch.float64, device=dev)
    kr = torch.fft.rfftfreq(n, d=1.0 / n, dtype=torch.float64, device=dev)
    kz, ky, kx = k1[:, None, None], k1[None, :, None], kr[None, None, :]
    kk = torch.sqrt(kx * kx + ky * ky + kz * kz)
    shape_amp = torch.where(kk > 0, torch.sqrt(kk ** 4 * torch.exp(-2.0 * (kk / 4.0) ** 2)) /
                            torch.clamp(kk, min=1e-30), torch.zeros_like(kk))   # sqrt(E/(4 pi k^2)) up to a constant
    spec = []
    for _ in range(3):
        noise = torch.randn((n, n, n), generator=g, dtype=torch.float64).to(dev)
        f = torch.fft.rfftn(noise)
        del noise
        f = f / torch.clamp(f.abs(), min=1e-300) * shape_amp
        spec.append(f)
    # exact discrete projection: D_d = (e^{i k h} - 1)/h at centres, G_d = (1 - e^{-i k h})/h at faces
    ks = (kx, ky, kz)
    Dd = [(torch.exp(1j * k * h) - 1.0) / h for k in ks]
    Gd = [(1.0 - torch.exp(-1j * k * h)) / h for k in ks]
    div = Dd[0] * spec[0] + Dd[1] * spec[1] + Dd[2] * spec[2]
    lap = Dd[0] * Gd[0] + Dd[1] * Gd[1] + Dd[2] * Gd[2]
    lap = torch.where(lap.abs() > 0, lap, torch.ones_like(lap))
    phi = div / lap
    out = []
    for d in range(3):
        out.append(torch.fft.irfftn(spec[d] - Gd[d] * phi, s=(n, n, n)))
    del spec, div, phi
    rms = math.sqrt(float(sum((o * o).mean() for o in out)) / 3.0)
    tdt = torch.float64 if dtype == "f64" else torch.float32
    fields = {c: (o / rms).to(tdt).contiguous() for c, o in zip("uvw", out)}
    if device == "cpu":
        fields = {c: o.numpy() for c, o in fields.items()}
    cfg["init"] = fields
    return cfg


def hit_box(nx, ny, nz, seed=778, dtype="f64", **kw):
    """The c5 recipe on a non-cubic triply periodic box with isotropic spacing h = 2 pi / min(nx, ny, nz) (parity
    cases that need a particular extent, e.g. ny >= 384 for the 32-row V-cycle tiles): random phases, the same
    spectrum E(k) ~ k^4 exp(-2 (k/4)^2) in physical wavenumbers, exact discrete projection, u_rms = 1.  CPU only."""
    import torch
    nref = min(nx, ny, nz)
    h = 2.0 * math.pi / nref
    cfg = _base(name="c5_hit_box", nx=nx, ny=ny, nz=nz, lx=nx * h, ly=ny * h, lz=nz * h, nu=1e-3, dt=5e-4, precond="gmg",
                rtol=1e-8, max_iter=200, steps=10, seed=seed, dtype=dtype)
    cfg.update(kw)
    g = torch.Generator(device="cpu")
    g.manual_seed(seed)
    kz = (torch.fft.fftfreq(nz, d=1.0 / nz, dtype=torch.float64) * (nref / nz))[:, None, None]
    ky = (torch.fft.fftfreq(ny, d=1.0 / ny, dtype=torch.float64) * (nref / ny))[None, :, None]
    kx = (torch.fft.rfftfreq(nx, d=1.0 / nx, dtype=torch.float64) * (nref / nx))[None, None, :]
    kk = torch.sqrt(kx * kx + ky * ky + kz * kz)
    amp = torch.where(kk > 0, torch.sqrt(kk ** 4 * torch.exp(-2.0 * (kk / 4.0) ** 2)) / torch.clamp(kk, min=1e-30), torch.zeros_like(kk))
    spec = []
    for _ in range(3):
        f = torch.fft.rfftn(torch.randn((nz, ny, nx), generator=g, dtype=torch.float64))
        spec.append(f / torch.clamp(f.abs(), min=1e-300) * amp)
    ks = (kx, ky, kz)
    Dd = [(torch.exp(1j * k * h) - 1.0) / h for k in ks]
    Gd = [(1.0 - torch.exp(-1j * k * h)) / h for k in ks]
    div = Dd[0] * spec[0] + Dd[1] * spec[1] + Dd[2] * spec[2]
    lap = Dd[0] * Gd[0] + Dd[1] * Gd[1] + Dd[2] * Gd[2]
    lap = torch.where(lap.abs() > 0, lap, torch.ones_like(lap))
    phi = div / lap
    out = [torch.fft.irfftn(spec[d] - Gd[d] * phi, s=(nz, ny, nx)) for d in range(3)]
    rms = math.sqrt(float(sum((o * o).mean() for o in out)) / 3.0)
    cfg["init"] = {c: (o / rms).contiguous().numpy() for c, o in zip("uvw", out)}
    return cfg


def make(name, **kw):
    return {"c1": taylor_green, "c2": channel, "c3": sphere, "c4": cylinder_fsi, "c5": hit}[name](**kw)
