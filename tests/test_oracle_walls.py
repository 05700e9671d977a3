"""Pins for the oracle's WALL rows (`fill_velocity_ghosts`, the k = 0 / k = nz-1 rows of
`momentum_rhs`, `phi_rhs`, `temperature_rhs`, `interface_quantities`, the Neumann rows of the Poisson
solve) and for `update_gamma` (S0) against things that are not the oracle:

  * plane Poiseuille flow: closed-form value of the viscous operator on interior AND wall rows
    (no-slip through the odd ghost, textbook), and the closed-form discrete steady state;
  * manufactured fields that satisfy the wall conditions exactly (sympy, tests/mms_helper.py):
    2nd-order convergence of every RHS on ALL rows, uniform and stretched;
  * the reflection principle: through its ghosts a row of the wall-bounded box reads what the same row
    reads in a z-periodic box of twice the height holding the evenly / oddly reflected fields, so the
    wall code path must reproduce the PERIODIC code path (pinned separately) to round-off, operator by
    operator, nhat-dependent terms included;
  * Gamma = gamma_rel * max(|u|,|v|,|w|) + gamma_abs exactly, with the maximum placed in each
    component in turn (N15).

Passages: SURVEY.md 8(c) "Walls" (ghost rules), S3, N10, N15, N17; PAPER.md:36 (2nd-order staggered
finite differences, pressure correction); BASELINE.json:9, :11 (no-slip walls, stretched z)."""
import math

import numpy as np
import pytest

from paper_2502_04189_b200 import workloads as W
import mms_helper as mms


def _tanh_faces(n, lz, a):
    zf = lz * 0.5 * (1.0 + np.tanh(a * (np.arange(n + 1) / n - 0.5) * 2) / math.tanh(a))
    zf[0], zf[-1] = 0.0, lz
    return zf


# ------------------------------------------------------------------ plane Poiseuille flow
def _channel_cfg(nz, lz, nu, stretched, **kw):
    cfg = dict(nx=8, ny=8, nz=nz, lx=1.0, ly=1.3, lz=lz, z_wall=1, eps=0.1, rho1=1.0, rho2=1.0,
               mu1=nu, mu2=nu, gamma_abs=0.0, gamma_rel=0.0)
    if stretched:
        cfg["zf"] = _tanh_faces(nz, lz, 1.1)
    cfg.update(kw)
    return cfg


@pytest.mark.parametrize("stretched", [False, True])
@pytest.mark.parametrize("axis", ["x", "y"])
def test_plane_poiseuille_viscous_operator_interior_and_wall_rows(oracle_mod, stretched, axis):
    """u = c z (lz - z), v = w = 0, one fluid.  Advection vanishes identically.  A divided difference of a
    parabola is its derivative at the midpoint, (u[k+1] - u[k])/dzc[k] = c (lz - zc[k] - zc[k+1]), so on
    interior rows RHS = f - nu c (zc[k+1] - zc[k-1])/dzf[k]  (= f - 2 nu c when uniform).  On the wall rows the odd ghost u(-1) = -u(0) at distance dzf[0] gives
        RHS = nu [ (u1 - u0)/dzc[0] - 2 u0/dzf[0] ] / dzf[0] + f
    (= nu (u1 - 3 u0)/dz^2 + f when uniform).  A mirrored (free-slip) ghost gives nu (u1 - u0)/dz^2 + f
    and a wrong dzc at the wall changes the 2 u0/dzf[0] term: both fail."""
    nz, lz, nu, c, f = 24, 2.0, 0.37, 0.8, 0.21
    cfg = _channel_cfg(nz, lz, nu, stretched, **({"fx": f} if axis == "x" else {"fy": f}))
    zc = W.cell_centres(cfg)[2]
    dzf = np.diff(W.z_faces(cfg))
    prof = c * zc * (lz - zc)
    z = np.zeros((nz, 8, 8))
    flow = np.broadcast_to(prof[:, None, None], z.shape).copy()
    o = oracle_mod.Oracle(cfg)
    o.set_fields(flow if axis == "x" else z, flow if axis == "y" else z, z, z, z)
    r = o.momentum_rhs()
    got = r[0] if axis == "x" else r[1]
    other = r[1] if axis == "x" else r[0]
    expect = np.full(nz, f - 2.0 * nu * c)
    expect[1:-1] = f - nu * c * (zc[2:] - zc[:-2]) / dzf[1:-1]
    dzc0, dzcn = 0.5 * (dzf[0] + dzf[1]), 0.5 * (dzf[-1] + dzf[-2])
    expect[0] = nu * ((prof[1] - prof[0]) / dzc0 - 2.0 * prof[0] / dzf[0]) / dzf[0] + f
    expect[-1] = nu * (-2.0 * prof[-1] / dzf[-1] - (prof[-1] - prof[-2]) / dzcn) / dzf[-1] + f
    if not stretched:
        dz = lz / nz
        assert abs(expect[0] - (nu * (prof[1] - 3.0 * prof[0]) / dz ** 2 + f)) < 1e-12
    assert np.abs(got - expect[:, None, None]).max() < 1e-11
    assert np.abs(other).max() == 0.0 and np.abs(r[2]).max() == 0.0
    # the wall rows really differ from what a free-slip ghost would give (the test has teeth)
    freeslip = nu * ((prof[1] - prof[0]) / dzc0) / dzf[0] + f
    assert abs(freeslip - expect[0]) > 0.1


def _steady_profile(oracle_mod, cfg, f):
    """Discrete steady state of du/dt = RHS(u) for u = u(z), v = w = 0: RHS is then affine in u (advection
    vanishes), so its matrix is read off by probing the oracle with unit profiles and solved directly."""
    nz = cfg["nz"]
    z = np.zeros((nz, cfg["ny"], cfg["nx"]))
    o = oracle_mod.Oracle(cfg)

    def rhs(prof):
        o.set_fields(np.broadcast_to(prof[:, None, None], z.shape).copy(), z, z, z, z)
        return o.momentum_rhs()[0][:, 0, 0].copy()

    r0 = rhs(np.zeros(nz))
    A = np.stack([rhs(np.eye(nz)[k]) - r0 for k in range(nz)], axis=1)
    assert np.allclose(r0, f)
    o.close()
    return np.linalg.solve(A, -r0)


def test_plane_poiseuille_discrete_steady_state(oracle_mod):
    """Forcing f = 2 nu c drives the parabola c z (lz - z).  Uniform grid: the parabola satisfies every
    interior row exactly and misses the wall rows by nu c / 2, so the discrete steady state is EXACTLY
    parabola + c dz^2 / 4 (closed form); stretched grid: 2nd-order convergence to the parabola.  The steady
    profile must then survive full RK3 steps of the oracle (S3 ghosts, Neumann Poisson rows, S5) unchanged."""
    lz, nu, c = 2.0, 0.5, 0.9
    f = 2.0 * nu * c
    for nz in (8, 16):
        cfg = _channel_cfg(nz, lz, nu, False, fx=f)
        zc = W.cell_centres(cfg)[2]
        us = _steady_profile(oracle_mod, cfg, f)
        assert np.abs(us - (c * zc * (lz - zc) + c * (lz / nz) ** 2 / 4.0)).max() < 1e-12
    errs = []
    for nz in (8, 16, 32):
        cfg = _channel_cfg(nz, lz, nu, True, fx=f)
        zc = W.cell_centres(cfg)[2]
        us = _steady_profile(oracle_mod, cfg, f)
        errs.append(np.abs(us - c * zc * (lz - zc)).max())
    assert math.log2(errs[0] / errs[1]) > 1.8 and math.log2(errs[1] / errs[2]) > 1.9, errs
    # time stepping keeps it (nz = 32, stretched)
    z = np.zeros((32, 8, 8))
    u0 = np.broadcast_to(us[:, None, None], z.shape).copy()
    o = oracle_mod.Oracle(cfg)
    o.set_fields(u0, z, z, z, z)
    for _ in range(3):
        o.step(1e-3)
    g = o.get_fields()
    assert np.abs(g["u"] - u0).max() < 1e-12
    assert np.abs(g["v"]).max() < 1e-14 and np.abs(g["w"]).max() < 1e-14


# ------------------------------------------------------------------ manufactured fields on the wall rows
PRM = dict(rho1=3.0, rho2=1.0, mu1=0.05, mu2=0.02, k1=0.08, k2=0.03, cp1=2.0, cp2=1.0,
           sigma=0.0, gx=0.3, gy=-0.2, gz=-1.0, rho_ref=1.0, beta=0.6, t_ref=0.4,
           fx=0.11, fy=-0.07, fz=0.05, a_lin=0.13, heat=1, t_bot=1.0, t_top=0.0)


def _wall_mms_errors(oracle_mod, n, stretched):
    lz, eps = 2.0, 0.35
    cfg = dict(nx=n, ny=n, nz=n, lx=2 * np.pi, ly=2 * np.pi, lz=lz, z_wall=1, eps=eps, delta=1e-100,
               gamma_rel=0.0, gamma_abs=0.0, **PRM)
    if stretched:
        cfg["zf"] = _tanh_faces(n, lz, 1.2)
    fn = mms.build(dict(PRM, eps=eps, gamma=0.0), lz, walls=True)
    xc, yc, zc = W.cell_centres(cfg)
    zf = W.z_faces(cfg)
    xf, yf, zfu = xc + 0.5 * cfg["lx"] / n, yc + 0.5 * cfg["ly"] / n, zf[1:]
    fields = dict(u=mms.sample(fn["u"], xf, yc, zc), v=mms.sample(fn["v"], xc, yf, zc),
                  w=mms.sample(fn["w"], xc, yc, zfu), p=np.zeros((n, n, n)),
                  phi=mms.sample(fn["phi"], xc, yc, zc), T=mms.sample(fn["T"], xc, yc, zc))
    assert np.abs(fields["w"][-1]).max() < 1e-15
    fields["w"][-1] = 0.0
    o = oracle_mod.Oracle(cfg)
    o.set_fields(**fields)
    ru, rv, rw = o.momentum_rhs()
    got = dict(rhs_u=ru, rhs_v=rv, rhs_w=rw[:-1], rhs_phi=o.phi_rhs(0.0), rhs_T=o.temperature_rhs())
    ref = dict(rhs_u=mms.sample(fn["rhs_u"], xf, yc, zc), rhs_v=mms.sample(fn["rhs_v"], xc, yf, zc),
               rhs_w=mms.sample(fn["rhs_w"], xc, yc, zfu)[:-1], rhs_phi=mms.sample(fn["rhs_phi"], xc, yc, zc),
               rhs_T=mms.sample(fn["rhs_T"], xc, yc, zc))
    whole = {k: np.abs(got[k] - ref[k]).max() / np.abs(ref[k]).max() for k in got}
    rows = {k: max(np.abs(got[k][q] - ref[k][q]).max() for q in (0, -1)) / np.abs(ref[k]).max() for k in got}
    return whole, rows


@pytest.mark.parametrize("stretched", [False, True])
def test_rhs_terms_converge_at_second_order_on_every_row_including_the_walls(oracle_mod, stretched):
    """Manufactured u, v, w (odd about both walls), phi (even), T (T - T_wall odd) satisfy the wall
    conditions exactly, so the ghost rules are exact and EVERY row -- k = 0 and k = nz-1 included, no band
    mask -- of the momentum (advection, variable-viscosity stress, gravity, Boussinesq, forcing, variable
    1/rho_f), phi-advection and temperature right-hand sides must converge at 2nd order.  Gamma = sigma = 0
    here: the terms that contain nhat are singular where grad(phi) vanishes, which on a wall is
    unavoidable; their wall rows are pinned by the mirror test below instead.  A free-slip u ghost, a
    mirrored w, a T ghost without the 2 T_wall or a wrong wall metric leaves an O(1) wall-row error."""
    w1, r1 = _wall_mms_errors(oracle_mod, 32, stretched)
    w2, r2 = _wall_mms_errors(oracle_mod, 64, stretched)
    for k in w1:
        assert w2[k] < 5e-3 and r2[k] < 1e-3, (k, w2[k], r2[k])
        assert math.log2(w1[k] / w2[k]) > 1.9, (k, w1[k], w2[k])
        assert math.log2(r1[k] / r2[k]) > 1.8, (k, r1[k], r2[k])


# ------------------------------------------------------------------ walls == mirror extension, periodic box
def _mirror_case(nz=12):
    """A wall-bounded two-phase case with every term on (rho, mu ratios, sigma, Gamma, heat with equal wall
    temperatures, horizontal gravity and forcing) and its mirror extension to a z-periodic box of height
    2 lz: cell-centred even fields concat(f[::-1], f), no-slip fields odd, w odd about the wall faces."""
    nx, ny, lz = 16, 8, 1.0
    zf = _tanh_faces(nz, lz, 0.9)
    cfg = dict(nx=nx, ny=ny, nz=nz, lx=1.6, ly=0.8, lz=lz, z_wall=1, zf=zf, eps=0.12, rho1=4.0, rho2=1.0,
               mu1=0.03, mu2=0.01, k1=0.05, k2=0.02, cp1=1.5, cp2=1.0, sigma=0.4, gamma_rel=0.5, gamma_abs=0.7,
               gx=0.3, gy=-0.2, gz=0.0, rho_ref=1.0, beta=0.5, t_ref=0.2, fx=0.05, fy=0.02, fz=0.0, a_lin=0.1,
               heat=1, t_bot=0.3, t_top=0.3)
    rng = np.random.default_rng(11)
    shape = (nz, ny, nx)
    phi = W.phase_field(cfg, np.array([[0.7, 0.4, 0.22]]), 0.3)      # a drop that touches the bottom rows
    u, v, w = (0.3 * rng.standard_normal(shape) for _ in range(3))
    w[-1] = 0.0
    T = 0.3 + 0.2 * rng.standard_normal(shape)
    p = 0.1 * rng.standard_normal(shape)
    f = dict(u=u, v=v, w=w, p=p, phi=phi, T=T)
    dzf = np.diff(zf)
    zf2 = np.concatenate([[0.0], np.cumsum(np.concatenate([dzf[::-1], dzf]))])
    cfg2 = dict(cfg, nz=2 * nz, lz=2 * lz, z_wall=0, zf=zf2)
    even = lambda a: np.concatenate([a[::-1], a])
    odd = lambda a: np.concatenate([-a[::-1], a])
    w2 = np.concatenate([-w[nz - 2::-1], np.zeros((1, ny, nx)), w])
    f2 = dict(u=odd(u), v=odd(v), w=w2, p=even(p), phi=even(phi), T=np.concatenate([2 * 0.3 - T[::-1], T]))
    return cfg, f, cfg2, f2


def test_wall_rules_equal_the_reflected_extension_in_a_periodic_box(oracle_mod):
    """SURVEY.md 8(c) "Walls": every ghost rule is the even or odd reflection of the interior (dzf mirrored
    too).  A row of the wall-bounded box therefore reads, through its ghosts, exactly what the same row
    reads in a z-periodic box of twice the height holding the reflected fields, and the oracle's wall code
    (ghost fills with BC_ODD / BC_WFACE / BC_EVEN / BC_TWALL, R_z = 0 and zero fluxes on wall faces, the
    wall metrics dzc[-1] = dzf[0]) must agree to round-off with its PERIODIC code (pinned separately by the
    MMS, conservation and symmetry tests) -- operator by operator, including kappa, R and the
    nhat-dependent CSF and mass-consistent terms on the rows k = 0 and k = nz-1 that no manufactured
    solution can reach (grad(phi) must vanish somewhere on a wall).  Only the w row ON the top wall face
    is left out: there the wall box imposes w = 0 while the periodic box has an equation.  The Neumann
    Poisson rows (a_0 = c_{nz-1} = 0) and the gauge are compared the same way: an even right-hand side in
    the doubled cyclic solve."""
    cfg, f, cfg2, f2 = _mirror_case()
    nz = cfg["nz"]
    ow, op = oracle_mod.Oracle(cfg), oracle_mod.Oracle(cfg2)
    ow.set_fields(**f)
    op.set_fields(**f2)
    ow.substep(0, 1e-12)          # latches Gamma from max|u| (N15); dt is too small to move anything
    op.substep(0, 1e-12)
    assert ow.gamma() == op.gamma() and ow.gamma() > 0.7
    ow.set_fields(**f)
    op.set_fields(**f2)
    gam = 0.9
    cmp = [("rhs_phi", ow.phi_rhs(gam), op.phi_rhs(gam))]
    for nm in ("kappa", "Rx", "Ry", "Rz", "nhz"):
        cmp.append((nm, ow.intermediate(nm), op.intermediate(nm)))
    for nm, a, b in zip(("rhs_u", "rhs_v", "rhs_w"), ow.momentum_rhs(), op.momentum_rhs()):
        cmp.append((nm, a, b))
    cmp.append(("rhs_T", ow.temperature_rhs(), op.temperature_rhs()))
    for nm, a, b in cmp:
        b = b[nz:]
        if nm in ("rhs_w", "Rz"):
            assert np.abs(a[-1]).max() == 0.0, nm       # imposed on the top wall face
            a, b = a[:-1], b[:-1]
        scale = np.abs(a).max()
        assert scale > 0, nm
        assert np.abs(a - b).max() <= 1e-12 * scale, (nm, np.abs(a - b).max() / scale)
        assert np.abs(a[0]).max() > 1e-3 * scale, nm    # the bottom row is active in every operator
    assert np.abs(cmp[1][1][0]).max() > 1.0     # the drop really reaches the bottom row: kappa is active there
    rhs = np.random.default_rng(5).standard_normal(f["p"].shape)
    dzf = np.diff(cfg["zf"])[:, None, None]
    rhs -= (rhs * dzf).sum() / (dzf.sum() * rhs[0].size)      # compatible: the gauge row then changes nothing
    pw, pp = ow.poisson_solve(rhs), op.poisson_solve(np.concatenate([rhs[::-1], rhs]))
    assert np.abs(pw - pp[nz:]).max() <= 1e-11 * np.abs(pw).max()


# ------------------------------------------------------------------ S0: Gamma
@pytest.mark.parametrize("which", ["u", "v", "w"])
def test_update_gamma_takes_the_max_over_all_three_components(oracle_mod, which):
    """N15: Gamma = gamma_rel * max over faces of max(|u|, |v|, |w|) + gamma_abs, latched at stage 0.  The
    largest magnitude (negative, so that dropping the |.| fails too) is planted in each component in turn;
    a max that forgets one component, uses u^2 or a vector magnitude gives a different number."""
    n = 8
    cfg = dict(nx=n, ny=n, nz=n, lx=1.0, ly=1.0, lz=1.0, z_wall=0, eps=0.2, rho1=1.0, rho2=1.0, mu1=0.01,
               mu2=0.01, gamma_rel=1.2, gamma_abs=0.1)
    rng = np.random.default_rng(3)
    f = {k: rng.uniform(-0.5, 0.5, (n, n, n)) for k in "uvw"}
    f[which][3, 5, 2] = -0.9
    z = np.zeros((n, n, n))
    o = oracle_mod.Oracle(cfg)
    o.set_fields(f["u"], f["v"], f["w"], z, z)
    assert o.gamma() == 0.1                       # before the first stage-0 latch: gamma_abs
    o.substep(0, 1e-6)
    assert o.gamma() == 1.2 * 0.9 + 0.1
    latched = o.gamma()
    o.substep(1, 1e-6)                            # stages 1, 2 keep the latched value
    o.substep(2, 1e-6)
    assert o.gamma() == latched
