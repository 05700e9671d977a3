"""Seeded synthetic inputs for the five configurations of BASELINE.json (`configs[0..4]`).

This module serves BOTH the CPU oracle and the CUDA library: it produces plain numpy arrays
and a plain parameter dict and contains none of the method's arithmetic (no stencil of the
solver, no Poisson solve, no RK step).  It imports neither `oracle` nor the CUDA binding.

Recipes (restated in DESIGN.md "Input recipe"; values marked + are choices where
BASELINE.json fixes only a ratio or a non-dimensional number -- SURVEY.md 8(d)):

  every array has shape (nz, ny, nx), x fastest; u[k,j,i] on the x-face (x=(i+1)dx, y_j, zc_k),
  v on the y-face, w on the z-face zf[k+1].  rng = numpy default_rng(20250204 + index).

  * phase field: sum over droplets of 0.5*(1+tanh((R - r)/(2 eps))) (N21), r the minimum-image
    distance in the periodic directions; each droplet is added on a window of half-width
    R + 40 eps around it (beyond that its contribution is < 1e-17);  centres by sequential
    rejection with gap >= 2R + 6 eps between droplets and >= R + 6 eps from walls (clearance
    capped at 2R resp. R on coarse test grids).
  * solenoidal velocities are built as the discrete staggered curl of a vector potential, which
    is divergence-free to round-off by construction (no projection is needed).
  * dt (N16): 0.5*min(dt_adv, dt_visc, dt_sigma, dt_acdi), computed once from the initial fields.
"""
from __future__ import annotations

import math

import numpy as np

SEED0 = 20250204

NAMES = ["static_drop_32", "taylor_green_drops_128", "rising_bubbles_256", "hit_droplets_512",
         "channel_heat_1024x512x512"]

DEFAULT_GRIDS = [(32, 32, 32), (128, 128, 128), (256, 256, 256), (512, 512, 512), (1024, 512, 512)]
DEFAULT_STEPS = [10, 50, 100, 20, 20]


def _base(nx, ny, nz, lx, ly, lz):
    return dict(nx=int(nx), ny=int(ny), nz=int(nz), lx=float(lx), ly=float(ly), lz=float(lz), z_wall=0,
                rho1=1.0, rho2=1.0, mu1=1.0, mu2=1.0, k1=1.0, k2=1.0, cp1=1.0, cp2=1.0,
                sigma=0.0, eps=float(lx) / nx, delta=1e-100, gamma_rel=0.0, gamma_abs=0.0,
                gx=0.0, gy=0.0, gz=0.0, rho_ref=0.0, beta=0.0, t_ref=0.0, fx=0.0, fy=0.0, fz=0.0,
                a_lin=0.0, heat=0, t_bot=0.0, t_top=0.0)


def z_faces(cfg) -> np.ndarray:
    zf = cfg.get("zf")
    if zf is not None:
        return np.asarray(zf, dtype=np.float64)
    return np.linspace(0.0, cfg["lz"], cfg["nz"] + 1)


def cell_centres(cfg):
    nx, ny = cfg["nx"], cfg["ny"]
    dx, dy = cfg["lx"] / nx, cfg["ly"] / ny
    zf = z_faces(cfg)
    return (np.arange(nx) + 0.5) * dx, (np.arange(ny) + 0.5) * dy, 0.5 * (zf[1:] + zf[:-1])


def place_droplets(rng, cfg, count, radius, max_tries=200000):
    """Sequential rejection (N21): min-image gap >= 2R+6eps, wall gap >= R+6eps.  On the
    coarse grids of the small parity cases 6 eps can exceed the box, so the clearance is
    capped: min(6 eps, 2R) between droplets, min(6 eps, R) to a wall (inactive at full size)."""
    L = np.array([cfg["lx"], cfg["ly"], cfg["lz"]])
    eps = cfg["eps"]
    gap = 2 * radius + min(6 * eps, 2 * radius)
    wall = radius + min(6 * eps, radius)
    centres = []
    tries = 0
    while len(centres) < count:
        tries += 1
        if tries > max_tries:
            raise RuntimeError("could not place %d droplets" % count)
        c = rng.uniform(0.0, 1.0, 3) * L
        if cfg["z_wall"] and not (wall <= c[2] <= L[2] - wall):
            continue
        ok = True
        for o in centres:
            d = np.abs(c - o)
            d[0] = min(d[0], L[0] - d[0])
            d[1] = min(d[1], L[1] - d[1])
            if not cfg["z_wall"]:
                d[2] = min(d[2], L[2] - d[2])
            if math.sqrt(float(d @ d)) < gap:
                ok = False
                break
        if ok:
            centres.append(c)
    return np.array(centres)


def phase_field(cfg, centres, radius) -> np.ndarray:
    """Sum of tanh profiles, each added on a window of half-width R + 40 eps."""
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    lx, ly, lz = cfg["lx"], cfg["ly"], cfg["lz"]
    eps = cfg["eps"]
    xc, yc, zc = cell_centres(cfg)
    phi = np.zeros((nz, ny, nx))
    half = radius + 40.0 * eps

    def window(coord, c, length, periodic):
        d = coord - c
        if periodic:
            d = d - length * np.round(d / length)
        idx = np.nonzero(np.abs(d) <= half)[0]
        return idx, d[idx]

    for c in np.reshape(centres, (-1, 3)):
        ix, ddx = window(xc, c[0], lx, True)
        iy, ddy = window(yc, c[1], ly, True)
        iz, ddz = window(zc, c[2], lz, not cfg["z_wall"])
        r = np.sqrt(ddz[:, None, None] ** 2 + ddy[None, :, None] ** 2 + ddx[None, None, :] ** 2)
        phi[np.ix_(iz, iy, ix)] += 0.5 * (1.0 + np.tanh((radius - r) / (2.0 * eps)))
    return phi


def _smooth_potential(rng, shape, k0, lengths):
    """Three real random fields with Gaussian spectrum exp(-(|k|/k0)^2) via an inverse FFT
    (library routine); |k| is the physical wavenumber of a box with the given lengths."""
    try:
        from scipy import fft as sfft
        irfftn = lambda a, s: sfft.irfftn(a, s=s, workers=-1)
    except Exception:  # pragma: no cover
        irfftn = lambda a, s: np.fft.irfftn(a, s=s)
    nz, ny, nx = shape
    kz = 2 * np.pi * np.fft.fftfreq(nz, d=lengths[2] / nz)
    ky = 2 * np.pi * np.fft.fftfreq(ny, d=lengths[1] / ny)
    kx = 2 * np.pi * np.fft.rfftfreq(nx, d=lengths[0] / nx)
    k2 = kz[:, None, None] ** 2 + ky[None, :, None] ** 2 + kx[None, None, :] ** 2
    amp = np.exp(-k2 / (k0 * k0))
    amp[0, 0, 0] = 0.0
    out = []
    for _ in range(3):
        theta = rng.uniform(0.0, 2 * np.pi, amp.shape)
        out.append(irfftn(amp * np.exp(1j * theta), shape))
    return out


def staggered_curl(cfg, Ax, Ay, Az):
    """u = Dy(Az) - Dz(Ay), v = Dz(Ax) - Dx(Az), w = Dx(Ay) - Dy(Ax) with backward differences;
    Ax, Ay live on z-faces (index k <-> zf[k+1]), Az on cell-centre heights.  With walls the
    caller passes Ax, Ay that vanish on k = nz-1 (top wall); the bottom wall value is zero."""
    dx, dy = cfg["lx"] / cfg["nx"], cfg["ly"] / cfg["ny"]
    zf = z_faces(cfg)
    dzf = (zf[1:] - zf[:-1])[:, None, None]

    def dxm(f):
        return (f - np.roll(f, 1, axis=2)) / dx

    def dym(f):
        return (f - np.roll(f, 1, axis=1)) / dy

    def dzm(f):
        lo = np.roll(f, 1, axis=0)
        if cfg["z_wall"]:
            lo[0] = 0.0
        return (f - lo) / dzf

    u = dym(Az) - dzm(Ay)
    v = dzm(Ax) - dxm(Az)
    w = dxm(Ay) - dym(Ax)
    return u, v, w


def stable_dt(cfg, u, v, w) -> float:
    """N16: dt = 0.5*min(dt_adv, dt_visc, dt_sigma, dt_acdi), evaluated on the initial fields."""
    dx, dy = cfg["lx"] / cfg["nx"], cfg["ly"] / cfg["ny"]
    zf = z_faces(cfg)
    dzf = zf[1:] - zf[:-1]
    dzmin = float(dzf.min())
    cfl = np.abs(u) / dx + np.abs(v) / dy + np.abs(w) / dzf[:, None, None]
    adv = float(cfl.max())
    umax = max(float(np.abs(u).max()), float(np.abs(v).max()), float(np.abs(w).max()))
    gamma = cfg["gamma_rel"] * umax + cfg["gamma_abs"]
    S = 1.0 / dx ** 2 + 1.0 / dy ** 2 + 1.0 / dzmin ** 2
    nu_max = max(cfg["mu1"] / cfg["rho1"], cfg["mu2"] / cfg["rho2"])
    lims = []
    if adv > 0:
        lims.append(1.0 / adv)
    if nu_max > 0:
        lims.append(1.0 / (2.0 * nu_max * S))
    if cfg["sigma"] > 0:
        dmin = min(dx, dy, dzmin)
        lims.append(math.sqrt((cfg["rho1"] + cfg["rho2"]) * dmin ** 3 / (4.0 * math.pi * cfg["sigma"])))
    if gamma > 0:
        lims.append(1.0 / (2.0 * gamma * cfg["eps"] * S))
    if cfg["heat"]:
        a_max = max(cfg["k1"] / (cfg["rho1"] * cfg["cp1"]), cfg["k2"] / (cfg["rho2"] * cfg["cp2"]))
        lims.append(1.0 / (2.0 * a_max * S))
    return 0.5 * min(lims)


# Host memory a CPU comparison run of configs[4] at its own 1024x512x512 needs (about 40 ghost-padded fp64 arrays of
# 2.19 GB, a complex work array, the inputs and two sets of outputs).  Below it the full-size parity test falls back to
# 1024x512x256; `cfg5_parity_grid` is the one place that decides, so that the test and smoke() report the same branch.
CFG5_FULL_HOST_GB = 150.0


def cfg5_parity_grid(available_gb: float):
    """(grid, ndrops, label) of the configs[4] full-size parity case on a host with `available_gb` of free memory."""
    if available_gb >= CFG5_FULL_HOST_GB:
        return None, None, "1024x512x512"
    return (1024, 512, 256), 32, "1024x512x256"


def make(index: int, grid=None, ndrops=None, radius=None):
    """Build configuration `index` (0..4).  `grid=(nx,ny,nz)`, `ndrops`, `radius` override the
    BASELINE.json sizes for small parity cases (same recipe, same parameters).
    Returns (cfg, fields, dt, steps): cfg is a plain dict, fields a dict of numpy arrays
    u, v, w, p, phi and T (T only if cfg['heat'])."""
    rng = np.random.default_rng(SEED0 + index)
    nx, ny, nz = grid if grid is not None else DEFAULT_GRIDS[index]
    shape = (nz, ny, nx)
    steps = DEFAULT_STEPS[index]
    zeros = lambda: np.zeros(shape)

    if index == 0:  # static drop, BASELINE.json configs[0]
        cfg = _base(nx, ny, nz, 1.0, 1.0, 1.0)
        cfg.update(rho1=10.0, rho2=1.0, mu1=0.1, mu2=0.01, sigma=1.0, gamma_abs=1.0)
        R = 0.15 if radius is None else radius
        phi = phase_field(cfg, np.array([[0.5, 0.5, 0.5]]), R)
        u, v, w = zeros(), zeros(), zeros()
        dt = 1e-4
        cfg["radius"] = R

    elif index == 1:  # drops in a Taylor-Green field, configs[1]
        L = 2 * np.pi
        cfg = _base(nx, ny, nz, L, L, L)
        cfg.update(rho1=1.0, rho2=1.0, mu1=1e-3, mu2=1e-3, sigma=0.05, gamma_rel=1.2)
        R = 0.4 if radius is None else radius
        n = 4 if ndrops is None else ndrops
        xc, yc, zc = cell_centres(cfg)
        xf, yf = xc + 0.5 * L / nx, yc + 0.5 * L / ny
        u = np.sin(xf)[None, None, :] * np.cos(yc)[None, :, None] * np.cos(zc)[:, None, None]
        v = -np.cos(xc)[None, None, :] * np.sin(yf)[None, :, None] * np.cos(zc)[:, None, None]
        w = zeros()
        phi = phase_field(cfg, place_droplets(rng, cfg, n, R), R)
        dt = stable_dt(cfg, u, v, w)

    elif index == 2:  # rising bubble array, configs[2]
        cfg = _base(nx, ny, nz, 1.0, 1.0, 1.0)
        D = 0.2
        sigma = 1.0 * 1.0 * D * D / 10.0                 # Eo = rho_l g D^2 / sigma = 10
        mu_l = 1.0 * math.sqrt(1.0 * D) * D / 100.0      # Ga = rho_l sqrt(g D) D / mu_l = 100
        cfg.update(z_wall=1, rho1=1e-3, rho2=1.0, mu1=mu_l / 100.0, mu2=mu_l, sigma=sigma,
                   gz=-1.0, rho_ref=1.0, eps=0.75 * 1.0 / nx, gamma_rel=1.0, gamma_abs=0.1)
        R = 0.1 if radius is None else radius
        n = 8 if ndrops is None else ndrops
        u, v, w = zeros(), zeros(), zeros()
        phi = phase_field(cfg, place_droplets(rng, cfg, n, R), R)
        dt = stable_dt(cfg, u, v, w)

    elif index == 3:  # droplet-laden HIT, configs[3]
        L = 2 * np.pi
        cfg = _base(nx, ny, nz, L, L, L)
        R = 0.15 if radius is None else radius
        n = 200 if ndrops is None else ndrops
        cfg.update(rho1=1.0, rho2=1.0, mu1=1e-3, mu2=1e-3, sigma=1.0 * 1.0 * (2 * 0.15) / 5.0,
                   a_lin=0.02, gamma_rel=1.0)
        # |A_hat|^2 ~ E(k)/k^4 with E ~ k^4 exp(-2 (k/4)^2)  =>  |A_hat| ~ exp(-(k/4)^2)
        Ax, Ay, Az = _smooth_potential(rng, shape, 4.0, (L, L, L))
        u, v, w = staggered_curl(cfg, Ax, Ay, Az)
        del Ax, Ay, Az
        urms = math.sqrt(float((u * u).mean() + (v * v).mean() + (w * w).mean()) / 3.0)
        u /= urms; v /= urms; w /= urms
        phi = phase_field(cfg, place_droplets(rng, cfg, n, R), R)
        dt = stable_dt(cfg, u, v, w)

    elif index == 4:  # droplet-laden channel with heat transfer, configs[4]
        lx, ly, lz = 4 * np.pi, 2 * np.pi, 2.0
        cfg = _base(nx, ny, nz, lx, ly, lz)
        alpha = 2.0
        zf = 1.0 + np.tanh(alpha * (np.arange(nz + 1) / nz - 0.5)) / math.tanh(alpha / 2.0)
        zf[0], zf[-1] = 0.0, lz
        nu = 2.0 / 5600.0                                # Re_b = U_b 2h / nu = 5600, U_b = h = 1
        cfg.update(z_wall=1, zf=zf, rho1=10.0, rho2=1.0, mu1=10.0 * nu, mu2=nu, sigma=0.2,
                   k1=4.0 * nu, k2=nu, cp1=2.0, cp2=1.0, gz=-0.1, beta=1.0, t_ref=0.5,
                   t_bot=1.0, t_top=0.0, rho_ref=1.0, fx=3.0 * nu, heat=1, gamma_rel=1.0)
        R = 0.1 if radius is None else radius
        n = 64 if ndrops is None else ndrops
        xc, yc, zc = cell_centres(cfg)
        Ax, Ay, Az = _smooth_potential(rng, shape, 6.0, (lx, ly, lz))
        env_f = (zf[1:] * (lz - zf[1:]))[:, None, None]  # vanishes on the top wall face
        env_c = (zc * (lz - zc))[:, None, None]
        Ax *= env_f; Ay *= env_f; Az *= env_c
        u, v, w = staggered_curl(cfg, Ax, Ay, Az)
        del Ax, Ay, Az
        amp = 0.1 / max(float(np.abs(u).max()), float(np.abs(v).max()), float(np.abs(w).max()))
        u *= amp; v *= amp; w *= amp
        u += (6.0 * (zc / lz) * (1.0 - zc / lz))[:, None, None]
        w[-1] = 0.0
        phi = phase_field(cfg, place_droplets(rng, cfg, n, R), R)
        T = (1.0 - zc / lz)[:, None, None] + 0.01 * rng.uniform(-1.0, 1.0, shape)
        dt = stable_dt(cfg, u, v, w)
    else:
        raise ValueError("config index must be 0..4")

    cfg["name"] = NAMES[index]
    cfg["index"] = index
    fields = dict(u=np.ascontiguousarray(u), v=np.ascontiguousarray(v), w=np.ascontiguousarray(w),
                  p=zeros(), phi=np.ascontiguousarray(phi))
    if cfg["heat"]:
        fields["T"] = np.ascontiguousarray(T)
    return cfg, fields, float(dt), steps
