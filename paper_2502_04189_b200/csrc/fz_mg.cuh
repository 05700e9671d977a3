// fz_mg.cuh -- SURVEY.md 8(f)-4: the variable-coefficient pressure Poisson problem
//     D( (1/rho_f) d_a p ) = rhs          ("the conventional variable-coefficients problem [solved with] a
//                                           geometric multigrid method"; Hypre in the paper, hand-written here)
// by conjugate gradients preconditioned with one geometric multigrid V-cycle.  rho_f = 1/2 (rho + rho(+1_a)) with
// rho = rho2 + (rho1-rho2) clip(phi) (N2, N11), periodic x and y, periodic or wall z (no flux through the wall faces),
// stretched z allowed.  Row k of the operator carries 1/dzf[k], so A is self-adjoint and negative semi-definite in the
// dzf-weighted inner product <u,v> = sum dzf[k] u v; constants span its null space (gauge N17: <1,p> = 0, and the
// dzf-weighted mean of rhs is removed first).  Every ingredient keeps that symmetry, which CG needs:
//   * smoother: red-black Gauss-Seidel, colours in the order R,B before and B,R after the coarse-grid correction
//     (zebra z-line Gauss-Seidel instead on wall-bounded grids with flat cells, see k_mg_zline);
//   * restriction: volume-weighted mean of the 8 children; prolongation: piecewise constant (its weighted adjoint);
//   * coarse operators: the same discretisation on the coarse grid, face coefficient = mean of the 4 fine faces that
//     tile the coarse face; levels halve nx, ny, nz together while all three stay even and >= 4;
//   * coarsest level: many symmetric Gauss-Seidel sweeps.
// All kernels are one thread per cell (the solver is HBM-bound: 7-point stencils over 4-5 arrays).
#pragma once
#include "fz_common.cuh"

#define FZ_MG_MAXLEV 10
#define FZ_MG_NU 2          // red-black sweeps before and after the coarse-grid correction
#define FZ_MG_COARSE 24     // symmetric sweeps on the coarsest level
#define FZ_MG_RBLOCKS 1184  // partial sums of the reductions (148 x 8)

struct FzMgLevel {
    int nx, ny, nz, z_wall;
    double cx, cy;              // 1/dx^2, 1/dy^2
    const double *czh, *czl;    // per k: 1/(dzc[k] dzf[k]) (face k+1/2 seen from cell k), 1/(dzc[k-1] dzf[k]) (face k-1/2; 0 at a wall)
    const double *wz;           // dzf[k]
    double *x, *b, *r;          // iterate, right-hand side, residual / scratch
    double *bx, *by, *bz;       // 1/rho_f on the "+" faces; bz = 0 on a wall face
};

#define FZ_MG_CELL                                                   \
    const int i = blockIdx.x * blockDim.x + threadIdx.x;             \
    const int j = blockIdx.y * blockDim.y + threadIdx.y;             \
    const int k = blockIdx.z;                                        \
    if (i >= L.nx || j >= L.ny) return;                              \
    const int sxy = L.nx * L.ny, c = i + L.nx * (j + L.ny * k);      \
    const int im = c - i + (i == 0 ? L.nx - 1 : i - 1), ip = c - i + (i + 1 == L.nx ? 0 : i + 1);                    \
    const int jm = c + ((j == 0 ? L.ny - 1 : j - 1) - j) * L.nx, jp = c + ((j + 1 == L.ny ? 0 : j + 1) - j) * L.nx;  \
    const int km = c + ((k == 0 ? L.nz - 1 : k - 1) - k) * sxy, kp = c + ((k + 1 == L.nz ? 0 : k + 1) - k) * sxy;

// the six off-diagonal coefficients of row c (the diagonal is minus their sum)
#define FZ_MG_COEF                                                                       \
    const double axp = L.cx * L.bx[c], axm = L.cx * L.bx[im];                            \
    const double ayp = L.cy * L.by[c], aym = L.cy * L.by[jm];                            \
    const double azp = L.czh[k] * L.bz[c], azm = L.czl[k] * L.bz[km];

// 1/rho_f on the faces of the finest level from the phase field
__global__ void k_mg_beta(FzMgLevel L, const double *__restrict__ phi, double rho2, double drho)
{
    FZ_MG_CELL
    (void)im; (void)jm; (void)km;
    const double r0 = rho2 + drho * fz_clip01(phi[c]);
    L.bx[c] = 1.0 / (0.5 * (r0 + rho2 + drho * fz_clip01(phi[ip])));
    L.by[c] = 1.0 / (0.5 * (r0 + rho2 + drho * fz_clip01(phi[jp])));
    L.bz[c] = (L.z_wall && k == L.nz - 1) ? 0.0 : 1.0 / (0.5 * (r0 + rho2 + drho * fz_clip01(phi[kp])));
}

// coarse face coefficient = mean of the four fine faces that tile it (L = coarse level, F = fine level)
__global__ void k_mg_coarsen_beta(FzMgLevel L, FzMgLevel F)
{
    FZ_MG_CELL
    (void)im; (void)ip; (void)jm; (void)jp; (void)km; (void)kp;
    const int fs = F.nx * F.ny;
    const int f0 = 2 * i + F.nx * (2 * j + F.ny * 2 * k);   // child (0,0,0)
    L.bx[c] = 0.25 * (F.bx[f0 + 1] + F.bx[f0 + 1 + F.nx] + F.bx[f0 + 1 + fs] + F.bx[f0 + 1 + F.nx + fs]);
    L.by[c] = 0.25 * (F.by[f0 + F.nx] + F.by[f0 + F.nx + 1] + F.by[f0 + F.nx + fs] + F.by[f0 + F.nx + 1 + fs]);
    L.bz[c] = 0.25 * (F.bz[f0 + fs] + F.bz[f0 + fs + 1] + F.bz[f0 + fs + F.nx] + F.bz[f0 + fs + F.nx + 1]);
}

// y = A x (out may not alias x)
__global__ void k_mg_apply(FzMgLevel L, const double *__restrict__ x, double *__restrict__ out)
{
    FZ_MG_CELL
    FZ_MG_COEF
    const double xc = x[c];
    out[c] = axp * (x[ip] - xc) + axm * (x[im] - xc) + ayp * (x[jp] - xc) + aym * (x[jm] - xc) +
             azp * (x[kp] - xc) + azm * (x[km] - xc);
}

// r = b - A x
__global__ void k_mg_residual(FzMgLevel L)
{
    FZ_MG_CELL
    FZ_MG_COEF
    const double xc = L.x[c];
    L.r[c] = L.b[c] - (axp * (L.x[ip] - xc) + axm * (L.x[im] - xc) + ayp * (L.x[jp] - xc) + aym * (L.x[jm] - xc) +
                       azp * (L.x[kp] - xc) + azm * (L.x[km] - xc));
}

// one colour of a Gauss-Seidel sweep: x_c = (sum_n a_n x_n - b_c) / sum_n a_n for the cells with (i+j+k) & 1 == colour
__global__ void k_mg_gs(FzMgLevel L, int colour)
{
    FZ_MG_CELL
    if (((i + j + k) & 1) != colour) return;
    FZ_MG_COEF
    const double s = axp * L.x[ip] + axm * L.x[im] + ayp * L.x[jp] + aym * L.x[jm] + azp * L.x[kp] + azm * L.x[km];
    L.x[c] = (s - L.b[c]) / (axp + axm + ayp + aym + azp + azm);
}

// z-line ("zebra") Gauss-Seidel for wall-bounded z: one thread per column (i, j) with (i + j) & 1 == colour solves the
// tridiagonal system of its nz unknowns exactly (Thomas; the x and y neighbours belong to the other colour and are
// frozen).  On the stretched wall grids the z coupling is 6-30 times the x, y coupling near the walls and point
// relaxation stalls (71 CG iterations at 512 x 256 x 256 of config 5); relaxing whole z lines restores the textbook
// rate.  Scratch: L.r holds the eliminated super-diagonal, L.x the modified right-hand side, then the solution.
__global__ void k_mg_zline(FzMgLevel L, int colour)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= L.nx || j >= L.ny || (((i + j) & 1) != colour)) return;
    const int sxy = L.nx * L.ny, c0 = i + L.nx * j;
    const int im = c0 - i + (i == 0 ? L.nx - 1 : i - 1), ip = c0 - i + (i + 1 == L.nx ? 0 : i + 1);
    const int jm = c0 + ((j == 0 ? L.ny - 1 : j - 1) - j) * L.nx, jp = c0 + ((j + 1 == L.ny ? 0 : j + 1) - j) * L.nx;
    double cp = 0.0, dp = 0.0, bzm = 0.0;   // c'_{k-1}, d'_{k-1}, bz of the face below (no flux through the bottom wall)
    for (int k = 0; k < L.nz; ++k) {
        const int o = k * sxy, c = c0 + o;
        const double axp = L.cx * L.bx[c], axm = L.cx * L.bx[im + o], ayp = L.cy * L.by[c], aym = L.cy * L.by[jm + o];
        const double bzc = L.bz[c];
        const double azp = L.czh[k] * bzc, azm = L.czl[k] * bzm;
        const double diag = -(axp + axm + ayp + aym + azp + azm);
        const double rhs = L.b[c] - (axp * L.x[ip + o] + axm * L.x[im + o] + ayp * L.x[jp + o] + aym * L.x[jm + o]);
        const double inv = 1.0 / (diag - azm * cp);
        cp = azp * inv;
        dp = (rhs - azm * dp) * inv;
        L.r[c] = cp;
        L.x[c] = dp;
        bzm = bzc;
    }
    double xn = 0.0;
    for (int k = L.nz - 1; k >= 0; --k) {
        const int c = c0 + k * sxy;
        xn = L.x[c] - L.r[c] * xn;
        L.x[c] = xn;
    }
}

// b_coarse = volume-weighted mean of the residual of the 8 children; x_coarse = 0   (L = coarse, F = fine)
__global__ void k_mg_restrict(FzMgLevel L, FzMgLevel F)
{
    FZ_MG_CELL
    (void)im; (void)ip; (void)jm; (void)jp; (void)km; (void)kp;
    const int fs = F.nx * F.ny;
    const int f0 = 2 * i + F.nx * (2 * j + F.ny * 2 * k);
    const double lo = F.r[f0] + F.r[f0 + 1] + F.r[f0 + F.nx] + F.r[f0 + F.nx + 1];
    const double hi = F.r[f0 + fs] + F.r[f0 + fs + 1] + F.r[f0 + fs + F.nx] + F.r[f0 + fs + F.nx + 1];
    const double w0 = F.wz[2 * k], w1 = F.wz[2 * k + 1];
    L.b[c] = 0.25 * (w0 * lo + w1 * hi) / (w0 + w1);
    L.x[c] = 0.0;
}

// x_fine += x_coarse(parent)   (L = fine, C = coarse)
__global__ void k_mg_prolong(FzMgLevel L, FzMgLevel C)
{
    FZ_MG_CELL
    (void)im; (void)ip; (void)jm; (void)jp; (void)km; (void)kp;
    L.x[c] += C.x[(i >> 1) + C.nx * ((j >> 1) + C.ny * (k >> 1))];
}

// ---- vector helpers of the CG loop (n = cells of the finest level; plane = nx*ny selects dzf[k])
__global__ void k_mg_fill(double *x, double v, int n)
{
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < n; c += gridDim.x * blockDim.x) x[c] = v;
}
// y = a x + s y
__global__ void k_mg_axpby(double *__restrict__ y, const double *__restrict__ x, double a, double s, int n)
{
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < n; c += gridDim.x * blockDim.x) y[c] = a * x[c] + s * y[c];
}
// y = x + shift
__global__ void k_mg_shift(double *__restrict__ y, const double *__restrict__ x, double shift, int n)
{
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < n; c += gridDim.x * blockDim.x) y[c] = x[c] + shift;
}
// partial[b] = sum over the block's cells of dzf[k] a[c] b[c]  (bvec == NULL: b = 1); fixed order: deterministic
__global__ void k_mg_dot(const double *__restrict__ a, const double *__restrict__ bvec, const double *__restrict__ wz,
                         int plane, int n, double *__restrict__ partial)
{
    __shared__ double sh[256];
    double s = 0.0;
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < n; c += gridDim.x * blockDim.x)
        s += wz[c / plane] * a[c] * (bvec ? bvec[c] : 1.0);
    sh[threadIdx.x] = s;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}
__global__ void k_mg_dot_final(const double *__restrict__ partial, int nb, double *__restrict__ out)
{
    __shared__ double sh[256];
    double s = 0.0;
    for (int q = threadIdx.x; q < nb; q += 256) s += partial[q];
    sh[threadIdx.x] = s;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = sh[0];
}
