"""Pins for the oracle's discrete operators (S1, S2b, S3) against things that are NOT the
oracle: continuous PDE right-hand sides derived with sympy (order of convergence), exact
discrete invariants (kinetic-energy conservation, flux-form conservation), exact steady
states (planar tanh equilibrium, conduction, hydrostatics) and symmetries.

Passages pinned: BASELINE.json:5 (i)-(iii); SURVEY.md 8(c) S1, S2, S2b, S3 and readings
N2-N5, N9-N14; PAPER.md:32 (one-fluid model, CSF, linear property map)
(2nd-order staggered finite differences, mass-momentum consistent flux)."""
import math

import numpy as np
import pytest

from paper_2502_04189_b200 import workloads as W
import mms_helper as mms

PRM = dict(rho1=3.0, rho2=1.0, mu1=0.05, mu2=0.02, k1=0.08, k2=0.03, cp1=2.0, cp2=1.0,
           sigma=0.7, gx=0.3, gy=-0.2, gz=-1.0, rho_ref=1.0, beta=0.6, t_ref=0.4,
           fx=0.11, fy=-0.07, fz=0.05, a_lin=0.13, heat=1, t_bot=1.0, t_top=0.0)


def _mms_errors(oracle_mod, n, stretched):
    lz = 2.0
    eps, gam = 0.35, 0.9          # fixed physical eps: the interface is resolved, errors are O(h^2)
    cfg = dict(nx=n, ny=n, nz=n, lx=2 * np.pi, ly=2 * np.pi, lz=lz, z_wall=1, eps=eps,
               delta=1e-100, gamma_rel=0.0, gamma_abs=gam, **PRM)
    if stretched:
        a = 1.2
        zf = lz * 0.5 * (1.0 + np.tanh(a * (np.arange(n + 1) / n - 0.5) * 2) / math.tanh(a))
        zf[0], zf[-1] = 0.0, lz
        cfg["zf"] = zf
    fn = mms.build(dict(PRM, eps=eps, gamma=gam), lz)
    xc, yc, zc = W.cell_centres(cfg)
    zf = W.z_faces(cfg)
    xf, yf, zfu = xc + 0.5 * cfg["lx"] / n, yc + 0.5 * cfg["ly"] / n, zf[1:]
    fields = dict(u=mms.sample(fn["u"], xf, yc, zc), v=mms.sample(fn["v"], xc, yf, zc),
                  w=mms.sample(fn["w"], xc, yc, zfu), p=np.zeros((n, n, n)),
                  phi=mms.sample(fn["phi"], xc, yc, zc), T=mms.sample(fn["T"], xc, yc, zc))
    fields["w"][-1] = 0.0
    o = oracle_mod.Oracle(cfg)
    o.set_fields(**fields)
    ru, rv, rw = o.momentum_rhs()
    got = dict(rhs_u=ru, rhs_v=rv, rhs_w=rw, rhs_phi=o.phi_rhs(gam), rhs_T=o.temperature_rhs(),
               kappa=o.intermediate("kappa"))
    ref = dict(rhs_u=mms.sample(fn["rhs_u"], xf, yc, zc), rhs_v=mms.sample(fn["rhs_v"], xc, yf, zc),
               rhs_w=mms.sample(fn["rhs_w"], xc, yc, zfu), rhs_phi=mms.sample(fn["rhs_phi"], xc, yc, zc),
               rhs_T=mms.sample(fn["rhs_T"], xc, yc, zc), kappa=mms.sample(fn["kappa"], xc, yc, zc))
    # the wall rows see the mirror/no-slip ghosts, which the smooth manufactured fields do not
    # satisfy: compare on the interior band 0.25 lz < z < 0.75 lz (same physical band at every n)
    band = (zc > 0.25 * lz) & (zc < 0.75 * lz)
    return {k: np.abs(got[k][band] - ref[k][band]).max() / np.abs(ref[k][band]).max() for k in got}


@pytest.mark.parametrize("stretched", [False, True])
def test_all_rhs_terms_converge_at_second_order_to_the_pde(oracle_mod, stretched):
    """Every term of S1, S2b and S3 (advection, variable-viscosity stress, CSF, the
    mass-consistent flux term, gravity, forcing, Boussinesq, ACDI regularisation, conduction)
    with all coefficients non-trivial: the discrete RHS must approach the sympy-derived
    continuous RHS with order ~2.  A dropped term, wrong sign, transposed index or wrong
    metric makes the error O(1) and fails."""
    e1 = _mms_errors(oracle_mod, 32, stretched)
    e2 = _mms_errors(oracle_mod, 64, stretched)
    for k in e1:
        order = math.log2(e1[k] / e2[k])
        assert e2[k] < 2e-2, (k, e2[k])
        assert order > 1.8, (k, e1[k], e2[k], order)


def _solenoidal(cfg, seed):
    rng = np.random.default_rng(seed)
    shape = (cfg["nz"], cfg["ny"], cfg["nx"])
    A = [rng.standard_normal(shape) for _ in range(3)]
    if cfg["z_wall"]:
        A[0][-1] = 0.0
        A[1][-1] = 0.0
    return W.staggered_curl(cfg, *A)


def test_advection_conserves_momentum_and_kinetic_energy(oracle_mod):
    """For a discretely solenoidal field on a uniform periodic grid the divergence-form,
    centred advective operator satisfies sum A_a = 0 and sum_a u_a A_a = 0 exactly
    (textbook property of the staggered 2nd-order scheme; SURVEY.md 8(c) pin 'S3 advection')."""
    n = 16
    cfg = dict(nx=n, ny=n, nz=n, lx=1.0, ly=1.3, lz=0.9, z_wall=0, eps=1.0 / n, rho1=1.0, rho2=1.0,
               mu1=0.0, mu2=0.0)
    u, v, w = _solenoidal(cfg, 1)
    o = oracle_mod.Oracle(cfg)
    o.set_fields(u, v, w, np.zeros_like(u), np.zeros_like(u))
    au, av, aw = o.momentum_rhs()
    scale = (np.abs(au).sum() + np.abs(av).sum() + np.abs(aw).sum())
    assert abs(au.sum()) + abs(av.sum()) + abs(aw.sum()) < 1e-12 * scale
    ke = (u * au).sum() + (v * av).sum() + (w * aw).sum()
    assert abs(ke) < 1e-13 * (np.abs(u * au).sum() + np.abs(v * av).sum() + np.abs(w * aw).sum())


def test_mass_consistent_term_exact_for_linear_velocity_and_zero_for_matched_density(oracle_mod):
    """N9: M_a = (rho1-rho2) (R . grad) u_a with central differences.  Between walls on a STRETCHED grid take
    u = a + b z, v = c + d z, w = e zf (linear in z, uniform in x, y): every central difference is exact, so
    on the rows whose stencil stays clear of the wall ghosts
        M_x = (rho1-rho2) b Rt_z,   M_y = (rho1-rho2) d Rt_z,   M_z = (rho1-rho2) e R_z
    where Rt_z is the mean of the four z-faces around the x- (y-) face -- the only part restated here; a
    wrong metric in a z-derivative (dzc for dzf, a missing factor 2) or a wrong sign fails.  M is isolated
    as RHS(rho1,rho2) - RHS(rho,rho) with mu = sigma = g = 0 (the advective part does not see rho), which
    also shows that it vanishes for matched densities whatever their common value."""
    nx, ny, nz, lz = 16, 16, 20, 1.0
    a_ = 1.1
    zf = lz * 0.5 * (1.0 + np.tanh(a_ * (np.arange(nz + 1) / nz - 0.5) * 2) / math.tanh(a_))
    zf[0], zf[-1] = 0.0, lz
    base = dict(nx=nx, ny=ny, nz=nz, lx=1.0, ly=1.0, lz=lz, z_wall=1, zf=zf, eps=1.5 / nx, mu1=0.0, mu2=0.0,
                gamma_abs=1.0)
    phi = W.phase_field(dict(base, rho1=1.0, rho2=1.0), np.array([[0.45, 0.55, 0.5]]), 0.25)
    zc = 0.5 * (zf[1:] + zf[:-1])
    ones = np.ones((nz, ny, nx))
    b, d, e = 0.7, -0.4, 0.3
    u = (0.3 + b * zc)[:, None, None] * ones
    v = (-0.2 + d * zc)[:, None, None] * ones
    w = (e * zf[1:])[:, None, None] * ones
    w[-1] = 0.0

    def run(rho1, rho2):
        o = oracle_mod.Oracle(dict(base, rho1=rho1, rho2=rho2))
        o.set_fields(u, v, w, np.zeros_like(u), phi)
        r = o.momentum_rhs()
        return r, o.intermediate("Rz"), o.intermediate("rho")

    r0, _, _ = run(1.0, 1.0)
    r0b, _, _ = run(2.5, 2.5)
    for q in range(3):
        assert np.array_equal(r0[q], r0b[q])          # matched densities: no M, no rho dependence at all
    r1, Rz, rho = run(3.0, 1.0)
    drho = 2.0
    sh = lambda f, dx=0, dy=0, dz=0: np.roll(f, (-dz, -dy, -dx), axis=(0, 1, 2))
    rows = slice(1, nz - 2)       # stencils clear of the wall ghosts and of the imposed w = 0 on the top face
    Rtz_x = 0.25 * (Rz + sh(Rz, dx=1) + sh(Rz, dz=-1) + sh(Rz, dx=1, dz=-1))
    Rtz_y = 0.25 * (Rz + sh(Rz, dy=1) + sh(Rz, dz=-1) + sh(Rz, dy=1, dz=-1))
    expect = [drho * b * Rtz_x / (0.5 * (rho + sh(rho, dx=1))),
              drho * d * Rtz_y / (0.5 * (rho + sh(rho, dy=1))),
              drho * e * Rz / (0.5 * (rho + sh(rho, dz=1)))]
    for q in range(3):
        got = (r1[q] - r0[q])[rows]
        scale = np.abs(expect[q][rows]).max()
        assert scale > 1e-3
        assert np.abs(got - expect[q][rows]).max() < 1e-12 * max(scale, np.abs(r0[q]).max()), q


def test_planar_tanh_profile_is_the_equilibrium_of_the_regularisation_flux(oracle_mod):
    """Jain (2022): phi = 0.5(1+tanh(d/2eps)) makes eps grad(phi) = phi(1-phi) n,
    so R = 0 in the continuum; the discrete residual near the interface must vanish at 2nd
    order for fixed eps (SURVEY.md 8(c) pin 'S1 regularisation operator')."""
    errs = []
    for n in (32, 64, 128):
        lz = 1.0
        cfg = dict(nx=8, ny=8, nz=n, lx=8.0 / n, ly=8.0 / n, lz=lz, z_wall=1, eps=lz / 16,
                   rho1=1.0, rho2=1.0, mu1=0.0, mu2=0.0)
        zc = (np.arange(n) + 0.5) * lz / n
        phi = np.broadcast_to((0.5 * (1 + np.tanh((zc - 0.47) / (2 * cfg["eps"]))))[:, None, None], (n, 8, 8)).copy()
        o = oracle_mod.Oracle(cfg)
        z = np.zeros_like(phi)
        o.set_fields(z, z, z, z, phi)
        r = o.phi_rhs(1.0)
        near = np.abs(zc - 0.47) < 3 * cfg["eps"]
        errs.append(np.abs(r[near]).max())
    assert math.log2(errs[0] / errs[1]) > 1.9 and math.log2(errs[1] / errs[2]) > 1.9, errs


def test_sphere_curvature(oracle_mod):
    """kappa = -div(n) of a sphere of radius R is 2/R on the interface, positive for phi=1
    inside (N5; Brackbill et al. 1992)."""
    n = 64
    cfg, f, _, _ = W.make(0, grid=(n, n, n), radius=0.25)
    cfg["eps"] = 2.0 / n
    f["phi"] = W.phase_field(cfg, np.array([[0.5, 0.5, 0.5]]), 0.25)
    o = oracle_mod.Oracle(cfg)
    o.set_fields(**f)
    o.phi_rhs(1.0)
    kap = o.intermediate("kappa")
    xc = (np.arange(n) + 0.5) / n
    r = np.sqrt((xc[:, None, None] - .5) ** 2 + (xc[None, :, None] - .5) ** 2 + (xc[None, None, :] - .5) ** 2)
    shell = np.abs(r - 0.25) < 0.5 / n
    assert abs(kap[shell].mean() - 8.0) < 0.05 * 8.0
    np.testing.assert_allclose(kap[shell] * r[shell], 2.0, rtol=0.05)


def test_phi_update_is_in_flux_form(oracle_mod):
    """sum(RHSphi * dzf) = 0 to round-off for arbitrary (non-solenoidal) velocity, walls and
    stretched grid: S1 is a divergence of face fluxes with zero wall flux."""
    cfg, f, dt, _ = W.make(4, grid=(16, 16, 24), ndrops=2, radius=0.3)
    rng = np.random.default_rng(3)
    for k in "uvw":
        f[k] = f[k] + 0.2 * rng.standard_normal(f[k].shape)
    f["w"][-1] = 0
    o = oracle_mod.Oracle(cfg)
    o.set_fields(**f)
    r = o.phi_rhs(0.8)
    dzf = np.diff(cfg["zf"])[:, None, None]
    assert abs((r * dzf).sum()) < 1e-13 * np.abs(r * dzf).sum()


def test_conduction_profile_is_an_exact_steady_state_on_the_stretched_grid(oracle_mod):
    """Linear T between isothermal walls, fluid at rest, no gravity: with the ghost rule
    T_ghost = 2 T_wall - T and centres at face midpoints, k_f dT/dz is the same on every face,
    so T must not change at all (SURVEY.md 8(c) pin 'S2b + walls')."""
    cfg, f, dt, _ = W.make(4, grid=(8, 8, 32), ndrops=0)
    cfg.update(gx=0.0, gy=0.0, gz=0.0, fx=0.0, sigma=0.0, k1=cfg["k2"], gamma_rel=0.0)
    zc = W.cell_centres(cfg)[2]
    T0 = np.broadcast_to((1.0 - zc / cfg["lz"])[:, None, None], f["phi"].shape).copy()
    z = np.zeros_like(T0)
    o = oracle_mod.Oracle(cfg)
    o.set_fields(z, z, z, z, z, T0)
    for _ in range(3):
        o.step(1e-2)
    g = o.get_fields()
    assert np.abs(g["T"] - T0).max() < 1e-13
    assert max(np.abs(g[k]).max() for k in "uvw") == 0.0


def test_hydrostatic_balance(oracle_mod):
    """Uniform fluid at rest under gravity with rho_ref = 0 (plain g): stays at rest and the
    pressure becomes hydrostatic, p(k+1)-p(k) = rho g (zc[k+1]-zc[k]) (N12); a horizontally
    stratified two-phase layer with rho_ref = rho2 also stays at rest."""
    cfg, f, dt, _ = W.make(2, grid=(8, 8, 32), ndrops=0)
    cfg.update(rho1=1.0, rho2=1.0, rho_ref=0.0, gz=-2.0, sigma=0.0, gamma_abs=0.0, gamma_rel=0.0)
    z = np.zeros_like(f["phi"])
    o = oracle_mod.Oracle(cfg)
    o.set_fields(z, z, z, z, z)
    for _ in range(2):
        o.step(1e-3)
    g = o.get_fields()
    assert max(np.abs(g[k]).max() for k in "uvw") < 1e-15
    dz = cfg["lz"] / cfg["nz"]
    np.testing.assert_allclose(np.diff(g["p"][:, 0, 0]), -2.0 * dz, rtol=1e-10)
    # stratified layer: light fluid (phi=1) on top, interface at z = 0.5, sigma != 0
    cfg.update(rho1=0.1, rho2=1.0, rho_ref=1.0, sigma=0.3, gamma_abs=1.0)
    zc = W.cell_centres(cfg)[2]
    phi = np.broadcast_to((0.5 * (1 + np.tanh((zc - 0.5) / (2 * cfg["eps"]))))[:, None, None], z.shape).copy()
    o = oracle_mod.Oracle(cfg)
    o.set_fields(z, z, z, z, phi)
    for _ in range(3):
        o.step(1e-3)
    g = o.get_fields()
    assert max(np.abs(g[k]).max() for k in "uvw") < 1e-13


def test_xy_transposition_symmetry_of_a_full_step(oracle_mod):
    """Swapping the roles of x and y (fields transposed, u<->v, parameters swapped) must give
    the transposed result: catches any single-axis index/metric slip in S1-S5."""
    cfg, f, dt, _ = W.make(1, grid=(16, 32, 16), ndrops=2, radius=0.7)
    cfg.update(rho1=2.0, mu1=5e-3, gx=0.3, gy=-0.1, fx=0.02, rho_ref=1.0)
    o = oracle_mod.Oracle(cfg)
    o.set_fields(**f)
    o.step(dt)
    a = o.get_fields()
    t = lambda q: np.ascontiguousarray(np.swapaxes(q, 1, 2))
    cfg2 = dict(cfg, nx=cfg["ny"], ny=cfg["nx"], lx=cfg["ly"], ly=cfg["lx"], gx=cfg["gy"], gy=cfg["gx"],
                fx=cfg["fy"], fy=cfg["fx"])
    o2 = oracle_mod.Oracle(cfg2)
    o2.set_fields(t(f["v"]), t(f["u"]), t(f["w"]), t(f["p"]), t(f["phi"]))
    o2.step(dt)
    b = o2.get_fields()
    for ka, kb in (("u", "v"), ("v", "u"), ("w", "w"), ("p", "p"), ("phi", "phi")):
        scale = max(np.abs(a[ka]).max(), 1e-300)
        assert np.abs(a[ka] - t(b[kb])).max() < 1e-12 * scale, (ka,)


def test_periodic_shift_invariance(oracle_mod):
    cfg, f, dt, _ = W.make(1, grid=(16, 16, 16), ndrops=2, radius=0.7)
    o = oracle_mod.Oracle(cfg)
    o.set_fields(**f)
    o.step(dt)
    a = o.get_fields()
    sh = lambda q: np.ascontiguousarray(np.roll(q, (3, 5, 7), axis=(0, 1, 2)))
    o2 = oracle_mod.Oracle(cfg)
    o2.set_fields(**{k: sh(q) for k, q in f.items()})
    o2.step(dt)
    b = o2.get_fields()
    for k in ("u", "v", "w", "p", "phi"):
        assert np.abs(sh(a[k]) - b[k]).max() < 1e-11 * max(np.abs(a[k]).max(), 1e-300), k
