"""Pins of oracle/varcoef.py (the variable-coefficient pressure Poisson problem)
against things other than itself: an entry-by-entry dense assembly written with explicit loops, the constant-density
limit (the independent plain-C FFT/tridiagonal oracle), the structure of the operator (null vectors, symmetry after
volume weighting) and a manufactured solution with a smooth variable density at second-order convergence."""
import numpy as np
import pytest

from oracle import varcoef as V
from paper_2502_04189_b200 import workloads as W


def _cfg(nx, ny, nz, walls, stretched=False, rho=(3.0, 1.0), box=(1.0, 1.5, 2.0)):
    cfg = W._base(nx, ny, nz, *box)
    cfg.update(rho1=rho[0], rho2=rho[1], z_wall=1 if walls else 0)
    if stretched:
        cfg["zf"] = W.tanh_faces(nz, box[2], 2.0) if hasattr(W, "tanh_faces") else None
        if cfg["zf"] is None:
            k = np.arange(nz + 1) / nz
            cfg["zf"] = box[2] * 0.5 * (1.0 + np.tanh(2.0 * (k - 0.5)) / np.tanh(1.0))
            cfg["zf"][0], cfg["zf"][-1] = 0.0, box[2]
    return cfg


def _dense_by_loops(cfg, phi):
    """Third, deliberately pedestrian coding of the operator: one Python loop over cells, six neighbours each."""
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    dx, dy = cfg["lx"] / nx, cfg["ly"] / ny
    zf = np.asarray(cfg["zf"]) if cfg.get("zf") is not None else np.linspace(0, cfg["lz"], nz + 1)
    zc = 0.5 * (zf[1:] + zf[:-1])
    wall = bool(cfg["z_wall"])
    rho = cfg["rho2"] + (cfg["rho1"] - cfg["rho2"]) * np.minimum(np.maximum(phi, 0.0), 1.0)
    N = nx * ny * nz
    A = np.zeros((N, N))
    at = lambda i, j, k: (i % nx) + nx * ((j % ny) + ny * (k % nz))
    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                r = at(i, j, k)
                for (di, dj, dk, h2) in ((1, 0, 0, dx * dx), (-1, 0, 0, dx * dx), (0, 1, 0, dy * dy), (0, -1, 0, dy * dy)):
                    beta = 2.0 / (rho[k, j, i] + rho[k, (j + dj) % ny, (i + di) % nx])
                    A[r, at(i + di, j + dj, k)] += beta / h2
                    A[r, r] -= beta / h2
                for dk in (1, -1):
                    kn = k + dk
                    if wall and (kn < 0 or kn >= nz):
                        continue                       # no flux through a wall face
                    knw = kn % nz
                    if 0 <= kn < nz:
                        hc = abs(zc[kn] - zc[k])
                    else:                              # periodic wrap: the ghost centre lies half a cell beyond the box
                        hc = 0.5 * (zf[k + 1] - zf[k]) + 0.5 * (zf[knw + 1] - zf[knw])
                    beta = 2.0 / (rho[k, j, i] + rho[knw, j, i])
                    A[r, at(i, j, kn)] += beta / (hc * (zf[k + 1] - zf[k]))
                    A[r, r] -= beta / (hc * (zf[k + 1] - zf[k]))
    return A


@pytest.mark.parametrize("walls,stretched", [(False, False), (True, False), (True, True)])
def test_assembly_entry_by_entry_and_against_array_differences(walls, stretched):
    cfg = _cfg(4, 6, 5, walls, stretched)
    rng = np.random.default_rng(1)
    phi = rng.uniform(-0.1, 1.1, (5, 6, 4))          # exercises the clip
    A = V.assemble(cfg, phi).toarray()
    assert np.abs(A - _dense_by_loops(cfg, phi)).max() <= 1e-12 * np.abs(A).max()
    p = rng.standard_normal((5, 6, 4))
    assert np.abs(A @ p.ravel() - V.apply(cfg, phi, p).ravel()).max() <= 1e-11 * np.abs(A).max()


@pytest.mark.parametrize("walls,stretched", [(False, False), (True, False), (True, True)])
def test_operator_structure(walls, stretched):
    """Constants are the null space, dzf the left null vector, diag(dzf) A is symmetric negative semi-definite."""
    cfg = _cfg(4, 4, 6, walls, stretched)
    phi = np.random.default_rng(2).uniform(0, 1, (6, 4, 4))
    A = V.assemble(cfg, phi).toarray()
    dzf, _ = V.z_metrics(cfg)
    w = np.repeat(dzf, 16)
    assert np.abs(A @ np.ones(96)).max() <= 1e-12 * np.abs(A).max()
    assert np.abs(w @ A).max() <= 1e-12 * np.abs(A).max()
    S = w[:, None] * A
    assert np.abs(S - S.T).max() <= 1e-12 * np.abs(S).max()
    ev = np.linalg.eigvalsh(0.5 * (S + S.T))
    assert ev.max() <= 1e-10 * np.abs(ev).max() and (np.abs(ev) < 1e-10 * np.abs(ev).max()).sum() == 1


@pytest.mark.parametrize("walls,stretched", [(False, False), (True, False), (True, True)])
def test_solution_satisfies_the_system_and_the_gauge(walls, stretched):
    cfg = _cfg(8, 4, 6, walls, stretched, rho=(1e-3, 1.0))
    rng = np.random.default_rng(3)
    phi = rng.uniform(0, 1, (6, 4, 8))
    rhs = rng.standard_normal((6, 4, 8))             # incompatible on purpose
    p = V.solve(cfg, phi, rhs)
    dzf, _ = V.z_metrics(cfg)
    wmean = lambda f: (f * dzf[:, None, None]).sum() / (dzf.sum() * 32)
    assert abs(wmean(p)) <= 1e-12 * np.abs(p).max()
    res = V.apply(cfg, phi, p) - (rhs - wmean(rhs))
    assert np.abs(res).max() <= 1e-9 * np.abs(rhs).max()
    pb = V.solve_bordered(cfg, phi, rhs)             # the bordered system as it stands gives the same solution
    assert np.abs(pb - p).max() <= 1e-10 * np.abs(p).max()


@pytest.mark.parametrize("kind", ["periodic", "walls", "stretched"])
def test_constant_density_limit_is_the_fft_tridiagonal_oracle(oracle_mod, kind):
    """rho1 = rho2 = rho_c: p = rho_c * (solution of the constant-coefficient problem by the plain-C oracle)."""
    nx, ny, nz = 16, 8, 12
    cfg = _cfg(nx, ny, nz, kind != "periodic", kind == "stretched", rho=(2.5, 2.5))
    o = oracle_mod.Oracle(cfg)
    rng = np.random.default_rng(4)
    rhs = rng.standard_normal(o.shape)
    dzf, _ = V.z_metrics(cfg)
    rhs -= (rhs * dzf[:, None, None]).sum() / (dzf.sum() * nx * ny)
    ref = 2.5 * o.poisson_solve(rhs)
    p = V.solve(cfg, rng.uniform(0, 1, o.shape), rhs)
    assert np.abs(p - ref).max() <= 1e-10 * np.abs(ref).max()
    o.close()


def test_manufactured_solution_second_order():
    """p = cos(2 pi x/lx) cos(2 pi y/ly) cos(pi z/lz) (Neumann at the walls), rho = 1 + 2 phi with a smooth phi:
    rhs = div((1/rho) grad p) from sympy; the discrete solution converges at second order on the stretched grid."""
    import sympy as sy
    x, y, z = sy.symbols("x y z")
    lx, ly, lz = 1.0, 1.5, 2.0
    pe = sy.cos(2 * sy.pi * x / lx) * sy.cos(2 * sy.pi * y / ly) * sy.cos(sy.pi * z / lz)
    ph = sy.Rational(1, 2) + sy.Rational(2, 5) * sy.sin(2 * sy.pi * x / lx) * sy.cos(2 * sy.pi * y / ly) * sy.cos(2 * sy.pi * z / lz)
    rho = 1 + 2 * ph
    rhs_e = sum(sy.diff(sy.diff(pe, s) / rho, s) for s in (x, y, z))
    f_p, f_ph, f_rhs = (sy.lambdify((x, y, z), e, "numpy") for e in (pe, ph, rhs_e))
    errs = []
    sizes = (8, 12, 16, 24)                          # a sparse direct solve of 32^3 unknowns takes a minute
    for n in sizes:
        cfg = _cfg(n, n, n, True, True, rho=(3.0, 1.0), box=(lx, ly, lz))
        zf = np.asarray(cfg["zf"])
        zc = 0.5 * (zf[1:] + zf[:-1])
        X = (np.arange(n) + 0.5) * lx / n
        Y = (np.arange(n) + 0.5) * ly / n
        Z3, Y3, X3 = np.meshgrid(zc, Y, X, indexing="ij")
        p = V.solve(cfg, f_ph(X3, Y3, Z3), f_rhs(X3, Y3, Z3))
        ex = f_p(X3, Y3, Z3)
        dzf = np.diff(zf)
        ex = ex - (ex * dzf[:, None, None]).sum() / (dzf.sum() * n * n)
        errs.append(np.abs(p - ex).max())
    orders = [np.log(errs[q] / errs[q + 1]) / np.log(sizes[q + 1] / sizes[q]) for q in range(3)]
    assert orders[2] > 1.8 and orders[1] > 1.7, (errs, orders)


# ---------------------------------------------------------------------------------------------------------------
# the plain-C oracle's own variable-coefficient path (orc_varcoef_solve, orc_substep with solver = 1)

@pytest.mark.parametrize("index,grid", [(0, (16, 16, 12)), (2, (16, 16, 12)), (4, (16, 8, 12))])
def test_c_oracle_cg_solve_matches_the_sparse_direct_solve(oracle_mod, index, grid):
    """Unpreconditioned CG in C (an iteration) against the bordered sparse direct solve (the definition): periodic ratio
    10, walls ratio 1000, stretched walls ratio 10."""
    cfg, f, dt, _ = W.make(index, grid=grid, ndrops=1, radius=0.2 if index else None)
    o = oracle_mod.Oracle(cfg)
    o.set_fields(**f)
    rhs = np.random.default_rng(9).standard_normal(o.shape)
    pc = o.varcoef_solve(rhs)
    pd = V.solve(cfg, f["phi"], rhs)
    assert np.abs(pc - pd).max() <= 1e-9 * np.abs(pd).max(), o.varcoef_iterations
    o.close()


def test_substep_with_the_variable_coefficient_solver_equals_the_splitting_for_matched_densities(oracle_mod):
    """rho1 = rho2: the splitting is exact (its p_hat terms vanish), so both pressure paths give the same step."""
    cfg, f, dt, _ = W.make(1, grid=(16, 16, 16), ndrops=1)
    a, b = oracle_mod.Oracle(cfg), oracle_mod.Oracle(cfg)
    b.set_solver(1)
    for o in (a, b):
        o.set_fields(**f)
        o.step(dt)
    fa, fb = a.get_fields(), b.get_fields()
    for k in fa:
        m = np.abs(fa[k]).max()
        assert np.abs(fa[k] - fb[k]).max() <= 1e-10 * max(m, 1e-300), k
    a.close(); b.close()


def test_substep_with_the_variable_coefficient_solver_projects_exactly_at_ratio_1000(oracle_mod):
    """D(u) after the correction = (residual of the solve) * a dt: divergence-free to the CG tolerance, walls, ratio 1000;
    and the step differs from the splitting's (which extrapolates p_hat) only at the order of the splitting error."""
    cfg, f, dt, _ = W.make(2, grid=(16, 16, 16), ndrops=1, radius=0.2)
    o = oracle_mod.Oracle(cfg)
    o.set_solver(1)
    o.set_fields(**f)
    for s in range(3):
        o.substep(s, dt)
    u = o.get_fields()
    dx = cfg["lx"] / cfg["nx"]
    div = (u["u"] - np.roll(u["u"], 1, 2)) / dx + (u["v"] - np.roll(u["v"], 1, 1)) / dx
    wz = np.concatenate([np.zeros((1,) + u["w"].shape[1:]), u["w"]])[:-1]          # w below the first cell: the wall
    div += (u["w"] - wz) / (cfg["lz"] / cfg["nz"])
    umax = max(np.abs(u[k]).max() for k in "uvw")
    assert np.abs(div).max() * dx / max(umax, 1.0) <= 1e-10
    o.close()
