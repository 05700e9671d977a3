"""CPU ORACLE (TEST INFRASTRUCTURE, NOT THE PRODUCT) -- the variable-coefficient pressure Poisson problem.

PAPER.md:36: "Fizzy also allows for solving the conventional variable-coefficients problem using a geometric multigrid
method" -- i.e. instead of the constant-coefficient splitting, solve directly

    D( (1/rho_f) d_a p ) = rhs                                  (operators of DESIGN.md section 2)

on the staggered grid: D the cell divergence of a face vector, d_a the face gradient, rho_f = 1/2 (rho + rho(+1_a))
the arithmetic face density (N11) of the linear map rho = rho2 + (rho1 - rho2) clip(phi, 0, 1) (N2), periodic x and y,
periodic or wall (homogeneous Neumann: no flux through the wall faces) z, possibly stretched in z.

The result has a plain definition -- the solution of a linear system -- so this oracle IS that definition written out:
the matrix is assembled entry by entry (scipy.sparse, one loop per axis, no stencil tricks) and handed to a sparse direct
solver (a library primitive).  The operator is singular (constants) and, because row k carries 1/dzf[k], its left null
vector is w = dzf: the system is bordered with that vector,

    [ A   1 ] [ p      ]   [ rhs ]
    [ w^T 0 ] [ lambda ] = [ 0   ],

which makes the solution unique (sum_k dzf[k] p = 0: the gauge of N17) and absorbs an incompatible right-hand side
(lambda = its dzf-weighted mean); `solve_bordered` factorises exactly this matrix (small grids), `solve` reduces it by hand.  Nothing here is shared with the CUDA path; only tests/ may import it.
"""
from __future__ import annotations

import numpy as np
import scipy.sparse as sp
import scipy.sparse.linalg as spla


def z_metrics(cfg):
    """dzf[k] (cell heights) and dzc[k] (centre spacing at face k+1/2; the periodic wrap at k = nz-1)."""
    nz = cfg["nz"]
    zf = np.asarray(cfg["zf"], dtype=np.float64) if cfg.get("zf") is not None else np.linspace(0.0, cfg["lz"], nz + 1)
    dzf = np.diff(zf)
    dzc = 0.5 * (dzf + np.roll(dzf, -1))   # N10: centres are face midpoints
    return dzf, dzc


def face_coefficients(cfg, phi):
    """beta_a = 1/rho_f on the '+' face of every cell, a = x, y, z; beta_z = 0 on a wall face (no flux)."""
    rho = cfg["rho2"] + (cfg["rho1"] - cfg["rho2"]) * np.clip(phi, 0.0, 1.0)
    bx = 1.0 / (0.5 * (rho + np.roll(rho, -1, axis=2)))
    by = 1.0 / (0.5 * (rho + np.roll(rho, -1, axis=1)))
    bz = 1.0 / (0.5 * (rho + np.roll(rho, -1, axis=0)))
    if cfg.get("z_wall", 0):
        bz[-1, :, :] = 0.0
    return bx, by, bz


def assemble(cfg, phi):
    """The matrix of p -> D(beta d p), rows and columns in the flat order i + nx (j + ny k)."""
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    dx, dy = cfg["lx"] / nx, cfg["ly"] / ny
    dzf, dzc = z_metrics(cfg)
    bx, by, bz = face_coefficients(cfg, phi)
    N = nx * ny * nz
    idx = np.arange(N).reshape(nz, ny, nx)
    rows, cols, vals = [], [], []

    def add(r, c, v):
        rows.append(r.ravel()); cols.append(c.ravel()); vals.append(v.ravel())

    # x: face between i and i+1 (periodic).  Flux F = beta (p(i+1) - p(i))/dx enters cell i with +1/dx, cell i+1 with -1/dx
    ip = np.roll(idx, -1, axis=2)
    cx = bx / (dx * dx)
    add(idx, ip, cx); add(idx, idx, -cx); add(ip, idx, cx); add(ip, ip, -cx)
    # y
    jp = np.roll(idx, -1, axis=1)
    cy = by / (dy * dy)
    add(idx, jp, cy); add(idx, idx, -cy); add(jp, idx, cy); add(jp, jp, -cy)
    # z: face k+1/2 between k and k+1, spacing dzc[k]; divided by the height of the cell it enters
    kp = np.roll(idx, -1, axis=0)
    f = bz / dzc[:, None, None]
    lo = f / dzf[:, None, None]                       # contribution to cell k
    hi = f / np.roll(dzf, -1)[:, None, None]          # contribution to cell k+1
    add(idx, kp, lo); add(idx, idx, -lo); add(kp, idx, hi); add(kp, kp, -hi)
    A = sp.csr_matrix((np.concatenate(vals), (np.concatenate(rows), np.concatenate(cols))), shape=(N, N))
    return A


def solve(cfg, phi, rhs):
    """The zero-(dzf-weighted)-mean solution of D(beta d p) = rhs - (weighted mean of rhs); arrays (nz, ny, nx).
    The bordered system of the module header, reduced by hand so that the sparse factorisation stays sparse: lambda is the
    dzf-weighted mean of rhs (multiply the first block row by w^T: w^T A = 0), the consistent singular system is solved
    with the first unknown pinned to zero, and the constant that restores w^T p = 0 is subtracted."""
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    N = nx * ny * nz
    dzf, _ = z_metrics(cfg)
    A = assemble(cfg, np.asarray(phi, dtype=np.float64)).tocsc()
    w = np.repeat(dzf, nx * ny)
    b = np.asarray(rhs, dtype=np.float64).ravel()
    b = b - (w @ b) / w.sum()
    x = np.zeros(N)
    x[1:] = spla.spsolve(A[1:, 1:], b[1:])
    x -= (w @ x) / w.sum()
    return x.reshape(nz, ny, nx)


def solve_bordered(cfg, phi, rhs):
    """The bordered system factorised as it stands (dense border: small grids only)."""
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    N = nx * ny * nz
    dzf, _ = z_metrics(cfg)
    A = assemble(cfg, np.asarray(phi, dtype=np.float64))
    w = np.repeat(dzf, nx * ny)
    K = sp.bmat([[A, sp.csr_matrix(np.ones((N, 1)))], [sp.csr_matrix(w[None, :]), None]], format="csc")
    x = spla.spsolve(K, np.concatenate([np.asarray(rhs, dtype=np.float64).ravel(), [0.0]]))
    return x[:N].reshape(nz, ny, nx)


def apply(cfg, phi, p):
    """D(beta d p) by plain array differences (independent of `assemble`; used to pin it)."""
    nx, ny = cfg["nx"], cfg["ny"]
    dx, dy = cfg["lx"] / nx, cfg["ly"] / ny
    dzf, dzc = z_metrics(cfg)
    bx, by, bz = face_coefficients(cfg, phi)
    fx = bx * (np.roll(p, -1, axis=2) - p) / dx
    fy = by * (np.roll(p, -1, axis=1) - p) / dy
    fz = bz * (np.roll(p, -1, axis=0) - p) / dzc[:, None, None]
    return ((fx - np.roll(fx, 1, axis=2)) / dx + (fy - np.roll(fy, 1, axis=1)) / dy +
            (fz - np.roll(fz, 1, axis=0)) / dzf[:, None, None])
