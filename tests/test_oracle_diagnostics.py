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
