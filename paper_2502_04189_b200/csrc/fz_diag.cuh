// fz_diag.cuh -- run-time diagnostics of the current state:
//   [0] sum phi dV   [1] 1/2 sum rho(phi) |u_c|^2 dV   [2] max over faces of max(|u|,|v|,|w|)
//   [3] max |D(u)|   [4] sum |grad phi| dV (central differences)   [5] sum T dV / sum dV (heat on)
//   [6], [7] Nusselt number at the bottom / top wall: <-dT/dz>_wall lz/(t_bot - t_top), the wall gradient
//            through the Dirichlet ghost 2 T_wall - T (heat on, walls, t_bot != t_top; else 0)
// One grid-stride pass over the cells (every prognostic array read once, neighbours from L1/L2),
// fixed-order two-stage reduction: block partials in `part`, one CTA folds them -> deterministic.
#pragma once
#include "fz_common.cuh"

#define FZ_DIAG_BLOCKS (148 * 8)
#define FZ_DIAG_NV 9   // vol1, ke, umax, dmax, area, tsum, vsum, sum of T on plane 0, on plane nz-1

__device__ __forceinline__ void fz_diag_fold(double (&a)[FZ_DIAG_NV], const double (&b)[FZ_DIAG_NV])
{
    a[0] += b[0]; a[1] += b[1]; a[2] = fmax(a[2], b[2]); a[3] = fmax(a[3], b[3]);
    a[4] += b[4]; a[5] += b[5]; a[6] += b[6]; a[7] += b[7]; a[8] += b[8];
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
    double acc[FZ_DIAG_NV] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
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
        const double tc = P.heat ? T[c] : 0.0;
        b[5] = tc * dV;
        b[6] = dV;
        b[7] = k == 0 ? tc : 0.0;
        b[8] = k == P.nz - 1 ? tc : 0.0;
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
    double acc[FZ_DIAG_NV] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
    for (int b = threadIdx.x; b < nblocks; b += blockDim.x) {
        double t[FZ_DIAG_NV];
        for (int q = 0; q < FZ_DIAG_NV; ++q) t[q] = part[b * FZ_DIAG_NV + q];
        fz_diag_fold(acc, t);
    }
    fz_diag_block(acc);
    if (threadIdx.x == 0) {
        out[0] = acc[0]; out[1] = acc[1]; out[2] = acc[2]; out[3] = acc[3]; out[4] = acc[4];
        out[5] = P.heat ? acc[5] / acc[6] : 0.0;
        out[6] = out[7] = 0.0;
        if (P.heat && P.z_wall && P.t_bot != P.t_top) {
            // mean over the wall of -(T(0) - T(-1))/dzc[-1] with T(-1) = 2 t_bot - T(0), dzc[-1] = dzf[0]; top alike
            const double inv = 1.0 / (double)P.sxy, scale = 1.0 / (P.t_bot - P.t_top);
            out[6] = 2.0 * (P.t_bot - acc[7] * inv) * P.idzf[0] * P.lz * scale;
            out[7] = 2.0 * (acc[8] * inv - P.t_top) * P.idzf[P.nz - 1] * P.lz * scale;
        }
    }
}

// ---------------------------------------------------------------- stable time step (N16): the two maxima
// red[0] = max over cells of |u|/dx + |v|/dy + |w|/dzf[k], red[1] = max(|u|,|v|,|w|); red zeroed by the caller.
__global__ void __launch_bounds__(256)
k_dt_reduce(FzP P, const double *__restrict__ u, const double *__restrict__ v, const double *__restrict__ w,
            double *__restrict__ red)
{
    const int lgxy = __ffs(P.nx) - 1 + __ffs(P.ny) - 1;
    double adv = 0.0, um = 0.0;
    for (unsigned c = blockIdx.x * blockDim.x + threadIdx.x; c < (unsigned)P.N; c += gridDim.x * blockDim.x) {
        const double a = fabs(u[c]), b = fabs(v[c]), d = fabs(w[c]);
        adv = fmax(adv, a * P.idx + b * P.idy + d * P.idzf[c >> lgxy]);
        um = fmax(um, fmax(a, fmax(b, d)));
    }
    for (int o = 16; o > 0; o >>= 1) {
        adv = fmax(adv, __shfl_xor_sync(0xffffffffu, adv, o));
        um = fmax(um, __shfl_xor_sync(0xffffffffu, um, o));
    }
    if ((threadIdx.x & 31) == 0) { fz_atomic_max_nonneg(red, adv); fz_atomic_max_nonneg(red + 1, um); }
}

// ---------------------------------------------------------------- number of non-finite values in up to six fields
__global__ void __launch_bounds__(256)
k_count_nonfinite(long long N, const double *f0, const double *f1, const double *f2, const double *f3,
                  const double *f4, const double *f5, unsigned long long *count)
{
    const double *f[6] = {f0, f1, f2, f3, f4, f5};
    unsigned long long bad = 0;
    for (long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x; c < N; c += (long long)gridDim.x * blockDim.x)
#pragma unroll
        for (int q = 0; q < 6; ++q)
            if (f[q] && !isfinite(f[q][c])) ++bad;
    bad = __reduce_add_sync(0xffffffffu, (unsigned)bad);
    if ((threadIdx.x & 31) == 0 && bad) atomicAdd(count, bad);
}
