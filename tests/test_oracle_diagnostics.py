"""Pins of the oracle's run-time diagnostics against closed forms.

* Taylor-Green field u = sin x cos y cos z, v = -cos x sin y cos z on the staggered grid: the cell-centred mean
  of sin at the two faces of a cell is sin(x_c) cos(dx/2), and sums of sin^2 / cos^2 over whole periods are exactly
  n/2, so KE = (2 pi)^3 / 8 * cos^2(dx/2) to round-off; max|u| is the largest face value; D(u) = 0 (dx = dy).
* Diffuse sphere phi = 1/2 (1 + tanh((R - r)/(2 eps))): with the Fermi-Dirac integrals
  int phi dV = 4 pi/3 R^3 (1 + (pi eps/R)^2) and int |grad phi| dV = 4 pi (R^2 + (pi eps)^2 / 3), up to terms
  exp(-R/eps); the discrete sums carry the O(dx^2) quadrature / central-difference error.
* mean temperature of the linear conduction profile between walls at T = 1 and 0 is 1/2 on any z grid.
"""
import numpy as np

from paper_2502_04189_b200 import workloads as W


def test_taylor_green_kinetic_energy_closed_form(oracle_mod):
    n = 32
    cfg, f, dt, _ = W.make(1, grid=(n, n, n), ndrops=1)
    f["phi"][:] = 0.0
    o = oracle_mod.Oracle(cfg)
    o.set_fields(**f)
    d = o.diagnostics()
    dx = 2 * np.pi / n
    assert abs(d[1] - (2 * np.pi) ** 3 / 8 * np.cos(dx / 2) ** 2) <= 1e-12 * d[1]
    assert d[2] == max(np.abs(f["u"]).max(), np.abs(f["v"]).max())
    assert d[3] <= 1e-13
    assert d[0] == 0.0 and d[4] == 0.0 and d[5] == 0.0


def test_kinetic_energy_uses_the_mapped_density(oracle_mod):
    """phi = 1 everywhere with rho1 = 7: KE is 7 times the rho = 1 value (rho = rho2 + (rho1-rho2) clip(phi))."""
    n = 16
    cfg, f, dt, _ = W.make(1, grid=(n, n, n), ndrops=1)
    cfg.update(rho1=7.0)
    f["phi"][:] = 1.0
    o = oracle_mod.Oracle(cfg)
    o.set_fields(**f)
    d = o.diagnostics()
    dx = 2 * np.pi / n
    assert abs(d[1] - 7.0 * (2 * np.pi) ** 3 / 8 * np.cos(dx / 2) ** 2) <= 1e-12 * d[1]
    assert abs(d[0] - (2 * np.pi) ** 3) <= 1e-12 * d[0]


def test_diffuse_sphere_volume_and_area(oracle_mod):
    errs = []
    for n in (32, 64):
        cfg, f, dt, _ = W.make(0, grid=(n, n, n))
        cfg["eps"] = 1.0 / 32            # fixed interface thickness: only the grid is refined
        R, eps = cfg["radius"], cfg["eps"]
        f["phi"] = W.phase_field(cfg, np.array([[0.5, 0.5, 0.5]]), R)
        o = oracle_mod.Oracle(cfg)
        o.set_fields(**f)
        d = o.diagnostics()
        vol = 4 * np.pi / 3 * R ** 3 * (1 + (np.pi * eps / R) ** 2)
        area = 4 * np.pi * (R ** 2 + (np.pi * eps) ** 2 / 3)
        errs.append((abs(d[0] - vol) / vol, abs(d[4] - area) / area))
    assert errs[0][0] <= 1e-3 and errs[1][0] <= 1e-3          # the volume sum converges spectrally
    assert errs[0][1] <= 2e-2 and errs[1][1] <= errs[0][1] / 3  # central differences: second order


def test_mean_temperature_of_the_conduction_profile(oracle_mod):
    cfg, f, dt, _ = W.make(4, grid=(16, 8, 24), ndrops=1, radius=0.3)
    zc = W.cell_centres(cfg)[2]
    f["T"] = np.ascontiguousarray(np.broadcast_to((1.0 - zc / cfg["lz"])[:, None, None], f["T"].shape))
    o = oracle_mod.Oracle(cfg)
    o.set_fields(**f)
    assert abs(o.diagnostics()[5] - 0.5) <= 1e-12   # sum of 3072 terms


def test_nusselt_number_of_the_conduction_profile_is_one(oracle_mod):
    """Pure conduction between isothermal walls: -dT/dz = (t_bot - t_top)/lz everywhere, so Nu = 1 at both walls
    (closed form) -- exactly, also on the stretched grid, because the Dirichlet ghost 2 T_wall - T(0) is the linear
    extrapolation and the profile is linear.  Adding A sin(pi z/lz) changes the wall gradients by +A pi/lz at the
    bottom and -A pi/lz at the top: Nu = 1 -+ A pi/(t_bot - t_top)... with the sign of cos(pi z/lz) at each wall,
    approached at second order."""
    cfg, f, dt, _ = W.make(4, grid=(16, 8, 48), ndrops=1, radius=0.3)
    lz, tb, tt = cfg["lz"], cfg["t_bot"], cfg["t_top"]
    zc = W.cell_centres(cfg)[2]
    lin = tb + (tt - tb) * zc / lz
    f["T"] = np.ascontiguousarray(np.broadcast_to(lin[:, None, None], f["T"].shape))
    o = oracle_mod.Oracle(cfg)
    o.set_fields(**f)
    d = o.diagnostics()
    assert abs(d[6] - 1.0) <= 1e-12 and abs(d[7] - 1.0) <= 1e-12
    errs = []
    A = 0.2
    for nz in (24, 48, 96):
        cfg, f, dt, _ = W.make(4, grid=(16, 8, nz), ndrops=1, radius=0.3)
        zc = W.cell_centres(cfg)[2]
        prof = tb + (tt - tb) * zc / lz + A * np.sin(np.pi * zc / lz)
        f["T"] = np.ascontiguousarray(np.broadcast_to(prof[:, None, None], f["T"].shape))
        o = oracle_mod.Oracle(cfg)
        o.set_fields(**f)
        d = o.diagnostics()
        # -dT/dz = (tb - tt)/lz - A pi/lz cos(pi z/lz): bottom (cos = 1) and top (cos = -1)
        errs.append(max(abs(d[6] - (1.0 - A * np.pi / (tb - tt))), abs(d[7] - (1.0 + A * np.pi / (tb - tt)))))
    assert errs[0] < 2e-2 and errs[1] < errs[0] / 3.5 and errs[2] < errs[1] / 3.5, errs


def test_stable_dt_single_limits_in_closed_form_and_against_the_generator(oracle_mod):
    """N16.  Each limit alone, from numbers typed here (uniform velocity, one fluid), then every limit at once on a
    two-phase stretched channel against paper_2502_04189_b200.workloads.stable_dt (numpy; written for the input
    recipe, shares nothing with the oracle's C)."""
    n = 8
    base = dict(nx=n, ny=2 * n, nz=n, lx=1.0, ly=1.0, lz=2.0, z_wall=0, eps=0.1, rho1=1.0, rho2=1.0, mu1=0.0, mu2=0.0)
    one = np.ones((n, 2 * n, n))
    z = np.zeros_like(one)
    dx, dy, dz = 1.0 / n, 1.0 / (2 * n), 2.0 / n

    def dt_of(cfg, u=z, v=z, w=z, cfl=0.5):
        o = oracle_mod.Oracle(cfg)
        o.set_fields(u, v, w, z, z)
        return o.stable_dt(cfl)

    assert dt_of(base) == 0.0                                                   # nothing limits
    adv = dt_of(base, 0.3 * one, -0.2 * one, 0.5 * one, cfl=0.4)
    assert abs(adv - 0.4 / (0.3 / dx + 0.2 / dy + 0.5 / dz)) <= 1e-15
    S = 1 / dx ** 2 + 1 / dy ** 2 + 1 / dz ** 2
    assert abs(dt_of(dict(base, mu1=0.02, mu2=0.03, rho1=2.0)) - 0.5 / (2 * 0.03 * S)) <= 1e-15
    assert abs(dt_of(dict(base, sigma=0.7, rho1=3.0)) - 0.5 * np.sqrt(4.0 * dy ** 3 / (4 * np.pi * 0.7))) <= 1e-15
    acdi = dt_of(dict(base, gamma_rel=1.2, gamma_abs=0.1), 0.0 * one, -0.9 * one, 0.2 * one)
    assert abs(acdi - 0.5 * min(1.0 / (0.9 / dy + 0.2 / dz), 1.0 / (2 * (1.2 * 0.9 + 0.1) * 0.1 * S))) <= 1e-15
    heat = dict(base, heat=1, k1=0.4, k2=0.1, cp1=2.0, cp2=1.0, rho1=0.5)
    o = oracle_mod.Oracle(heat)
    o.set_fields(z, z, z, z, z, z)
    assert abs(o.stable_dt(0.5) - 0.5 / (2 * 0.4 * S)) <= 1e-15                 # a_max = 0.4/(0.5*2)
    for idx, grid in ((4, (16, 8, 24)), (2, (16, 16, 12)), (3, (16, 16, 16))):
        cfg, f, dt, _ = W.make(idx, grid=grid, ndrops=1, radius=0.3 if idx == 4 else (0.2 if idx == 2 else 0.5))
        o = oracle_mod.Oracle(cfg)
        o.set_fields(**f)
        assert abs(o.stable_dt(0.5) - dt) <= 1e-14 * dt, idx
