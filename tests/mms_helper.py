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


def build(prm, lz):
    """Smooth manufactured fields on a box periodic in x,y (2 pi) with z in (0, lz);
    phi is monotone in z so that grad(psi) never vanishes.  Returns dict of lambdified
    functions: fields u,v,w,phi,T and the continuous RHS rhs_phi, rhs_T, rhs_u, rhs_v, rhs_w."""
    s = z / lz
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
                 rhs_u=rhs_u[0], rhs_v=rhs_u[1], rhs_w=rhs_u[2], kappa=kappa)
    return {k: sp.lambdify((x, y, z), e, "numpy") for k, e in exprs.items()}


def sample(fn, xs, ys, zs):
    out = fn(xs[None, None, :], ys[None, :, None], zs[:, None, None])
    return np.broadcast_to(out, (len(zs), len(ys), len(xs))).astype(np.float64).copy()
