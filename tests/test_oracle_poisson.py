"""Pins for the oracle's FFT and Poisson solver (S4): naive DFT, dense direct solve on tiny
grids, manufactured solution at second order, gauge.  Passages: PAPER.md:36 ("fast direct
FFT solver of the CaNS code"), BASELINE.json:5 (iv) ("FFTs in the periodic x and y directions
and a per-wavenumber tridiagonal solve in z"), SURVEY.md 8(c) S4 and N17, N18."""
import math

import numpy as np
import pytest

from paper_2502_04189_b200 import workloads as W


@pytest.mark.parametrize("n", [2, 4, 8, 16, 32, 64])
def test_fft_matches_naive_dft(oracle_mod, n):
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    jk = np.outer(np.arange(n), np.arange(n))
    for sign in (-1, +1):
        F = np.exp(sign * 2j * np.pi * jk / n)       # the definition, O(n^2)
        np.testing.assert_allclose(oracle_mod.fft(x, sign), F @ x, rtol=0, atol=1e-12 * n)


def _grid_cfg(kind, nx, ny, nz):
    cfg = dict(nx=nx, ny=ny, nz=nz, lx=1.3, ly=0.9, lz=1.1, z_wall=0, eps=0.1, rho1=1.0, rho2=1.0,
               mu1=0.0, mu2=0.0)
    if kind != "periodic":
        cfg["z_wall"] = 1
    if kind == "stretched":
        a = 2.0
        zf = cfg["lz"] * 0.5 * (1.0 + np.tanh(a * (np.arange(nz + 1) / nz - 0.5)) / math.tanh(a / 2))
        zf[0], zf[-1] = 0.0, cfg["lz"]
        cfg["zf"] = zf
    return cfg


def _dense_laplacian(cfg):
    """L = D(delta .) assembled entry by entry from its definition: sum over the six faces of
    (p_nb - p_c)/hc/hf, periodic wrap in x,y(,z), no flux through walls."""
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    dx, dy = cfg["lx"] / nx, cfg["ly"] / ny
    zf = W.z_faces(cfg)
    dzf = np.diff(zf)
    zc = 0.5 * (zf[1:] + zf[:-1])
    N = nx * ny * nz
    L = np.zeros((N, N))
    idx = lambda i, j, k: (i % nx) + nx * ((j % ny) + ny * (k % nz))
    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                c = idx(i, j, k)
                for (di, dj, h) in ((1, 0, dx), (-1, 0, dx), (0, 1, dy), (0, -1, dy)):
                    L[c, idx(i + di, j + dj, k)] += 1.0 / (h * h)
                    L[c, c] -= 1.0 / (h * h)
                for dk in (1, -1):
                    kk = k + dk
                    if cfg["z_wall"] and (kk < 0 or kk >= nz):
                        continue                      # wall face: zero gradient
                    hc = abs(zc[kk] - zc[k]) if 0 <= kk < nz else dzf[0]
                    L[c, idx(i, j, kk)] += 1.0 / (hc * dzf[k])
                    L[c, c] -= 1.0 / (hc * dzf[k])
    return L, dzf


@pytest.mark.parametrize("kind", ["periodic", "walls", "stretched"])
def test_poisson_matches_dense_direct_solve(oracle_mod, kind):
    cfg = _grid_cfg(kind, 8, 4, 6)
    L, dzf = _dense_laplacian(cfg)
    rng = np.random.default_rng(7)
    shape = (cfg["nz"], cfg["ny"], cfg["nx"])
    wgt = np.broadcast_to(dzf[:, None, None], shape)
    rhs = rng.standard_normal(shape)
    rhs -= (rhs * wgt).sum() / wgt.sum()               # compatible right-hand side
    o = oracle_mod.Oracle(cfg)
    p = o.poisson_solve(rhs)
    # residual with the independently assembled operator
    assert np.abs(L @ p.ravel() - rhs.ravel()).max() < 1e-11 * np.abs(rhs).max()
    # dense solve with the gauge sum(p dzf) = 0 appended as a Lagrange row
    N = L.shape[0]
    A = np.zeros((N + 1, N + 1))
    A[:N, :N] = L
    A[:N, N] = 1.0
    A[N, :N] = wgt.ravel()
    sol = np.linalg.solve(A, np.concatenate([rhs.ravel(), [0.0]]))[:N]
    np.testing.assert_allclose(p.ravel(), sol, rtol=0, atol=1e-12 * np.abs(sol).max())
    assert abs((p * wgt).sum()) < 1e-13 * np.abs(p * wgt).sum()


@pytest.mark.parametrize("kind", ["periodic", "walls", "stretched"])
def test_poisson_manufactured_solution_second_order(oracle_mod, kind):
    errs = []
    for n in (16, 32, 64):
        cfg = _grid_cfg(kind, n, n, n)
        xc, yc, zc = W.cell_centres(cfg)
        kx, ky = 2 * np.pi / cfg["lx"], 4 * np.pi / cfg["ly"]
        kz = (2 * np.pi if kind == "periodic" else np.pi) / cfg["lz"]
        pex = np.cos(kx * xc)[None, None, :] * np.cos(ky * yc + 0.3)[None, :, None] * np.cos(kz * zc)[:, None, None]
        rhs = -(kx * kx + ky * ky + kz * kz) * pex
        p = oracle_mod.Oracle(cfg).poisson_solve(rhs)
        dzf = np.diff(W.z_faces(cfg))[:, None, None]
        pex = pex - (pex * dzf).sum() / (dzf.sum() * n * n)
        errs.append(np.abs(p - pex).max())
    o1, o2 = math.log2(errs[0] / errs[1]), math.log2(errs[1] / errs[2])
    assert o1 > 1.8 and o2 > 1.9, (errs, o1, o2)
