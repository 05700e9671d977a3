"""Continuous right-hand sides of the governing equations, derived symbolically (sympy) from
the PDEs of PAPER.md:32 / BASELINE.json:5(i)-(iii) -- NOT from the discrete formulas of the
oracle.  Used to pin the oracle's discrete operators by their order of convergence."""
import numpy as np
import sympy as sp

x, y, z = sp.symbols("x y z", real=True)
X = (x, y, z)


def grad(f):
    return [sp.diff(f, s) for s in X]


def div(F):
    return sum(sp.diff(F[a], X[a]) for a in range(3))


def build(prm, lz, walls=False):
    """Smooth manufactured fields on a box periodic in x,y (2 pi) with z in (0, lz).
    walls=False: generic fields (phi monotone in z so that grad(psi) never vanishes); they do not
    satisfy the wall conditions, so only rows away from the walls can be compared.
    walls=True: fields that satisfy the wall conditions of SURVEY.md 8(c) "Walls" EXACTLY and are odd /
    even about both walls, so that the oracle's ghost rules (no-slip: u, v odd; w = 0 on the wall faces
    and odd beyond; phi mirrored; T - T_wall odd) hold to all orders and every row, including k = 0 and
    k = nz-1, must converge at 2nd order.  grad(phi) then necessarily vanishes at isolated points of the
    walls (a periodic function on a torus has critical points): `gradpsi` is returned so that the caller
    can leave those neighbourhoods out of the terms that contain nhat.
    Returns dict of lambdified functions: fields u,v,w,phi,T and the continuous RHS rhs_phi, rhs_T,
    rhs_u, rhs_v, rhs_w, kappa, gradpsi = |grad psi|."""
    s = z / lz
    if walls:
        phi = 0.5 + 0.22 * sp.cos(sp.pi * s) + 0.1 * sp.sin(x) * sp.cos(y) * (1 + 0.5 * sp.cos(2 * sp.pi * s))
        u = [(0.7 * sp.sin(x) * sp.cos(y) + 0.3) * sp.sin(sp.pi * s) * (1 + 0.3 * sp.cos(sp.pi * s)),
             (-0.4 * sp.cos(x + 0.3) * sp.sin(y) + 0.1 * sp.cos(2 * y) + 0.2) * sp.sin(sp.pi * s),
             0.5 * sp.sin(x + y) * sp.sin(sp.pi * s) * (1 + 0.4 * sp.cos(sp.pi * s))]
        T = prm["t_bot"] + (prm["t_top"] - prm["t_bot"]) * s + \
            (0.3 * sp.cos(x) * sp.sin(y + 0.4) + 0.15) * sp.sin(sp.pi * s) + 0.05 * sp.sin(2 * sp.pi * s)
    else:
        phi = 0.25 + 0.5 * s + 0.04 * sp.sin(x) * sp.cos(y) * sp.sin(sp.pi * s)
        u = [0.7 * sp.sin(x) * sp.cos(y) * sp.cos(2 * s) + 0.3,
             -0.4 * sp.cos(x + 0.3) * sp.sin(y) * sp.sin(1.5 * s + 0.2) + 0.1 * sp.cos(2 * y),
             0.5 * sp.sin(x + y) * sp.sin(sp.pi * s) * sp.cos(s)]
        T = 0.5 + 0.3 * sp.cos(x) * sp.sin(y + 0.4) * sp.cos(1.3 * s) + 0.2 * s

    eps, gam = prm["eps"], prm["gamma"]
    psi = eps * sp.log(phi / (1 - phi))
    gpsi = grad(psi)
    mag = sp.sqrt(sum(g * g for g in gpsi))
    nh = [g / mag for g in gpsi]
    sharp = sp.Rational(1, 4) * (1 - sp.tanh(psi / (2 * eps)) ** 2)
    gphi = grad(phi)
    R = [gam * (eps * gphi[a] - sharp * nh[a]) for a in range(3)]
    kappa = -div(nh)

    rho = prm["rho2"] + (prm["rho1"] - prm["rho2"]) * phi
    mu = prm["mu2"] + (prm["mu1"] - prm["mu2"]) * phi
    kth = prm["k2"] + (prm["k1"] - prm["k2"]) * phi
    cp = prm["cp2"] + (prm["cp1"] - prm["cp2"]) * phi
    g = [prm["gx"], prm["gy"], prm["gz"]]
    f = [prm["fx"], prm["fy"], prm["fz"]]

    rhs_phi = -div([u[a] * phi for a in range(3)]) + div(R)
    rhs_T = -div([u[a] * T for a in range(3)]) + div([kth * d for d in grad(T)]) / (rho * cp)
    rhs_u = []
    for a in range(3):
        adv = -div([u[t] * u[a] for t in range(3)])                    # divergence form
        visc = div([mu * (sp.diff(u[a], X[t]) + sp.diff(u[t], X[a])) for t in range(3)])
        surf = prm["sigma"] * kappa * gphi[a]
        mass = (prm["rho1"] - prm["rho2"]) * sum(R[t] * sp.diff(u[a], X[t]) for t in range(3))
        body = g[a] * (1 - prm["rho_ref"] / rho) + f[a] + prm["a_lin"] * u[a] \
            - g[a] * prm["beta"] * (T - prm["t_ref"])
        rhs_u.append(adv + (visc + surf + mass) / rho + body)

    exprs = dict(phi=phi, u=u[0], v=u[1], w=u[2], T=T, rhs_phi=rhs_phi, rhs_T=rhs_T,
                 rhs_u=rhs_u[0], rhs_v=rhs_u[1], rhs_w=rhs_u[2], kappa=kappa, gradpsi=mag)
    return {k: sp.lambdify((x, y, z), e, "numpy") for k, e in exprs.items()}


def sample(fn, xs, ys, zs):
    out = fn(xs[None, None, :], ys[None, :, None], zs[:, None, None])
    return np.broadcast_to(out, (len(zs), len(ys), len(xs))).astype(np.float64).copy()
