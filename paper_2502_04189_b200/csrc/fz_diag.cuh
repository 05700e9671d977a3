// fz_diag.cuh -- run-time diagnostics of the current state:
//   [0] sum phi dV   [1] 1/2 sum rho(phi) |u_c|^2 dV   [2] max over faces of max(|u|,|v|,|w|)
//   [3] max |D(u)|   [4] sum |grad phi| dV (central differences)   [5] sum T dV / sum dV (heat on)
// One grid-stride pass over the cells (every prognostic array read once, neighbours from L1/L2),
// fixed-order two-stage reduction: block partials in `part`, one CTA folds them -> deterministic.
#pragma once
#include "fz_common.cuh"

#define FZ_DIAG_BLOCKS (148 * 8)
#define FZ_DIAG_NV 7   // vol1, ke, umax, dmax, area, tsum, vsum

__device__ __forceinline__ void fz_diag_fold(double (&a)[FZ_DIAG_NV], const double (&b)[FZ_DIAG_NV])
{
    a[0] += b[0]; a[1] += b[1]; a[2] = fmax(a[2], b[2]); a[3] = fmax(a[3], b[3]);
    a[4] += b[4]; a[5] += b[5]; a[6] += b[6];
}

// block-level fold of acc; thread 0 ends up with the block result
__device__ __forceinline__ void fz_diag_block(double (&acc)[FZ_DIAG_NV])
{
    __shared__ double red[8][FZ_DIAG_NV];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        double b[FZ_DIAG_NV];
#pragma unroll
        for (int q = 0; q < FZ_DIAG_NV; ++q) b[q] = __shfl_down_sync(0xffffffffu, acc[q], o);
        fz_diag_fold(acc, b);
    }
    const int w = threadIdx.x >> 5, nw = blockDim.x >> 5;
    if ((threadIdx.x & 31) == 0)
        for (int q = 0; q < FZ_DIAG_NV; ++q) red[w][q] = acc[q];
    __syncthreads();
    if (threadIdx.x == 0)
        for (int ww = 1; ww < nw; ++ww) {
            double b[FZ_DIAG_NV];
            for (int q = 0; q < FZ_DIAG_NV; ++q) b[q] = red[ww][q];
            fz_diag_fold(acc, b);
        }
}

__global__ void __launch_bounds__(256)
k_diag(FzP P, const double *__restrict__ u, const double *__restrict__ v, const double *__restrict__ w,
       const double *__restrict__ phi, const double *__restrict__ T, double *__restrict__ part)
{
    const int lgx = __ffs(P.nx) - 1, lgy = __ffs(P.ny) - 1;
    const unsigned nx = P.nx, sxy = (unsigned)P.sxy;
    double acc[FZ_DIAG_NV] = {0, 0, 0, 0, 0, 0, 0};
    for (unsigned c = blockIdx.x * blockDim.x + threadIdx.x; c < (unsigned)P.N; c += gridDim.x * blockDim.x) {
        const int i = c & (P.nx - 1), j = (c >> lgx) & (P.ny - 1), k = c >> (lgx + lgy);
        const FzZ z = fz_zn(P, k);
        const unsigned pl = (unsigned)k * sxy, row = pl + nx * j;
        const unsigned xm = row + fz_im(i, P.nx), xp = row + fz_ip(i, P.nx);
        const unsigned ym = pl + nx * fz_im(j, P.ny) + i, yp = pl + nx * fz_ip(j, P.ny) + i;
        const unsigned zm = (unsigned)z.km * sxy + nx * j + i, zp = (unsigned)z.kp * sxy + nx * j + i;
        const double dV = P.dx * P.dy * P.dzf[k];
        const double u0 = u[c], v0 = v[c], w0 = w[c], um = u[xm], vm = v[ym];
        const double wm = z.gm ? 0.0 : w[zm];   // bottom wall face
        const double ph = phi[c], rho = P.rho2 + P.drho * fz_clip01(ph);
        const double uc = 0.5 * (u0 + um), vc = 0.5 * (v0 + vm), wc = 0.5 * (w0 + wm);
        const double div = (u0 - um) * P.idx + (v0 - vm) * P.idy + (w0 - wm) * P.idzf[k];
        const double gx = (phi[xp] - phi[xm]) * (0.5 * P.idx), gy = (phi[yp] - phi[ym]) * (0.5 * P.idy);
        const double gz = (phi[zp] - phi[zm]) * P.igz[k];   // mirror ghosts at walls
        double b[FZ_DIAG_NV];
        b[0] = ph * dV;
        b[1] = 0.5 * rho * (uc * uc + vc * vc + wc * wc) * dV;
        b[2] = fmax(fabs(u0), fmax(fabs(v0), fabs(w0)));
        b[3] = fabs(div);
        b[4] = sqrt(gx * gx + gy * gy + gz * gz) * dV;
        b[5] = P.heat ? T[c] * dV : 0.0;
        b[6] = dV;
        fz_diag_fold(acc, b);
    }
    fz_diag_block(acc);
    if (threadIdx.x == 0)
        for (int q = 0; q < FZ_DIAG_NV; ++q) part[blockIdx.x * FZ_DIAG_NV + q] = acc[q];
}

// one CTA: fold the block partials in a fixed order, write the six diagnostics
__global__ void __launch_bounds__(256)
k_diag_final(FzP P, const double *__restrict__ part, int nblocks, double *__restrict__ out)
{
    double acc[FZ_DIAG_NV] = {0, 0, 0, 0, 0, 0, 0};
    for (int b = threadIdx.x; b < nblocks; b += blockDim.x) {
        double t[FZ_DIAG_NV];
        for (int q = 0; q < FZ_DIAG_NV; ++q) t[q] = part[b * FZ_DIAG_NV + q];
        fz_diag_fold(acc, t);
    }
    fz_diag_block(acc);
    if (threadIdx.x == 0) {
        out[0] = acc[0]; out[1] = acc[1]; out[2] = acc[2]; out[3] = acc[3]; out[4] = acc[4];
        out[5] = P.heat ? acc[5] / acc[6] : 0.0;
    }
}
