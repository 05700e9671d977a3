// fz_tridiag.cuh -- S4c: per-wavenumber tridiagonal solve in z (kernel group (d)),
// BASELINE.json:5(iv); SURVEY/DESIGN readings N17 (gauge) and N18 (periodic z = cyclic system).
//
// For each retained mode t = l + nxh*m (lam = lam_x(l) + lam_y(m)):
//   a_k x_{k-1} + (b_k + lam) x_k + c_k x_{k+1} = d_k,   a_k = 1/(dzf[k] dzc[k-1]),
//   c_k = 1/(dzf[k] dzc[k]), b_k = -(a_k + c_k);  walls: a_0 = c_{nz-1} = 0; periodic: cyclic.
// The matrix is real and depends on the grid only, so its elimination is done ONCE at
// fizzy_create (k_tri_tables) and stored as tables; a solve is then two division-free sweeps
// that are coalesced along t (threads) and sequential along k:
//   forward   d'_k = (d_k - a_k d'_{k-1}) * INV[k][t]                    (+ h += F[k][t] d'_k, cyclic)
//   backward  x_k  = d'_k - c_k INV[k][t] x_{k+1}  (- E[k][t] X, cyclic, X = x_{nz-1})
// Cyclic systems are reduced with the last unknown X as a separator (T):
// rows 0..nz-2 are eliminated carrying the fill-in column E (coefficient of X), the last row is
// reduced alongside (coefficients F, pivot g -> GINV = 1/g), X = (d_{nz-1} - h) * GINV.
// The singular mode t = 0 gets GINV = 0 (cyclic) or INV[nz-1] = 0 (walls), i.e. x_{nz-1} = 0 (N17).
#pragma once
#include "fz_common.cuh"

struct FzTri {
    const double *a, *c;        // nz each (1-D)
    const double *lamx, *lamy;  // nxh, ny
    double *inv, *e, *f, *ginv; // [nz][M], [nz][M], [nz][M], [M];  M = nxh*ny
    long long M;
    int cyclic;
};

__global__ void k_tri_tables(FzP P, FzTri Tt)
{
    const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t >= Tt.M) return;
    const int l = (int)(t % P.nxh), m = (int)(t / P.nxh);
    const double lam = Tt.lamx[l] + Tt.lamy[m];
    const int n = P.nz;
    if (!Tt.cyclic) {
        double cp = 0.0;
        for (int k = 0; k < n; ++k) {
            const double a = Tt.a[k], c = Tt.c[k];
            const double den = -(a + c) + lam - a * cp;
            double inv = 1.0 / den;
            if (t == 0 && k == n - 1) inv = 0.0;  // N17: x_{nz-1} = 0 for the singular mode
            Tt.inv[(long long)k * Tt.M + t] = inv;
            cp = c * inv;
        }
    } else {
        // rows 0..n-2 with fill-in column e (coefficient of X = x_{n-1}); last row reduced alongside
        double cp = 0.0, e = 0.0;
        double f = Tt.c[n - 1];                       // coefficient of x_0 in the last row
        double g = -(Tt.a[n - 1] + Tt.c[n - 1]) + lam; // coefficient of X in the last row
        for (int k = 0; k <= n - 2; ++k) {
            const double a = Tt.a[k];
            const double c = (k == n - 2) ? 0.0 : Tt.c[k];
            const double den = -(Tt.a[k] + Tt.c[k]) + lam - a * cp;
            const double inv = 1.0 / den;
            double ek;
            if (k == 0) ek = a * inv;
            else ek = -a * e * inv;
            if (k == n - 2) ek += Tt.c[k] * inv;   // c_{n-2} multiplies X as well
            const double fk = (k == n - 2) ? f + Tt.a[n - 1] : f;
            Tt.inv[(long long)k * Tt.M + t] = inv;
            Tt.e[(long long)k * Tt.M + t] = ek;
            Tt.f[(long long)k * Tt.M + t] = fk;
            g -= fk * ek;
            cp = c * inv;
            f = -fk * cp;
            e = ek;
        }
        Tt.inv[(long long)(n - 1) * Tt.M + t] = 0.0;
        Tt.e[(long long)(n - 1) * Tt.M + t] = 0.0;
        Tt.f[(long long)(n - 1) * Tt.M + t] = 0.0;
        Tt.ginv[t] = (t == 0) ? 0.0 : 1.0 / g;  // N17
    }
}

#define FZ_TRI_U 8
template <bool CYCLIC>
__global__ void __launch_bounds__(128)
k_tridiag(FzP P, FzTri Tt, double2 *__restrict__ spec)
{
    const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t >= Tt.M) return;
    const long long M = Tt.M;
    const int n = P.nz;
    const int nrow = CYCLIC ? n - 1 : n;   // rows swept by the recurrences
    double2 dp = make_double2(0, 0), h = make_double2(0, 0);
    // forward sweep, loads batched FZ_TRI_U deep so the dependent chain never waits on HBM
    int k = 0;
    for (; k + FZ_TRI_U <= nrow; k += FZ_TRI_U) {
        double2 d[FZ_TRI_U];
        double iv[FZ_TRI_U], ff[FZ_TRI_U];
#pragma unroll
        for (int q = 0; q < FZ_TRI_U; ++q) {
            d[q] = spec[(long long)(k + q) * M + t];
            iv[q] = Tt.inv[(long long)(k + q) * M + t];
            if (CYCLIC) ff[q] = Tt.f[(long long)(k + q) * M + t];
        }
#pragma unroll
        for (int q = 0; q < FZ_TRI_U; ++q) {
            const double a = Tt.a[k + q];
            dp.x = (d[q].x - a * dp.x) * iv[q];
            dp.y = (d[q].y - a * dp.y) * iv[q];
            if (CYCLIC) { h.x += ff[q] * dp.x; h.y += ff[q] * dp.y; }
            spec[(long long)(k + q) * M + t] = dp;
        }
    }
    for (; k < nrow; ++k) {
        const double2 d = spec[(long long)k * M + t];
        const double iv = Tt.inv[(long long)k * M + t];
        const double a = Tt.a[k];
        dp.x = (d.x - a * dp.x) * iv;
        dp.y = (d.y - a * dp.y) * iv;
        if (CYCLIC) { const double ff = Tt.f[(long long)k * M + t]; h.x += ff * dp.x; h.y += ff * dp.y; }
        spec[(long long)k * M + t] = dp;
    }
    double2 X = make_double2(0, 0);
    if (CYCLIC) {
        const double2 dl = spec[(long long)(n - 1) * M + t];
        const double gi = Tt.ginv[t];
        X = make_double2((dl.x - h.x) * gi, (dl.y - h.y) * gi);
        spec[(long long)(n - 1) * M + t] = X;
    }
    // backward sweep: x_k = d'_k - c_k INV_k x_{k+1} - E_k X   (row nrow-1 has no x_{k+1} term)
    double2 xn = make_double2(0, 0);
    k = nrow - 1;
    for (; k - FZ_TRI_U + 1 >= 0; k -= FZ_TRI_U) {
        double2 d[FZ_TRI_U];
        double iv[FZ_TRI_U], ee[FZ_TRI_U];
#pragma unroll
        for (int q = 0; q < FZ_TRI_U; ++q) {
            d[q] = spec[(long long)(k - q) * M + t];
            iv[q] = Tt.inv[(long long)(k - q) * M + t];
            if (CYCLIC) ee[q] = Tt.e[(long long)(k - q) * M + t];
        }
#pragma unroll
        for (int q = 0; q < FZ_TRI_U; ++q) {
            const double cc = (k - q == nrow - 1) ? 0.0 : Tt.c[k - q] * iv[q];
            xn.x = d[q].x - cc * xn.x;
            xn.y = d[q].y - cc * xn.y;
            if (CYCLIC) { xn.x -= ee[q] * X.x; xn.y -= ee[q] * X.y; }
            spec[(long long)(k - q) * M + t] = xn;
        }
    }
    for (; k >= 0; --k) {
        const double2 d = spec[(long long)k * M + t];
        const double iv = Tt.inv[(long long)k * M + t];
        const double cc = (k == nrow - 1) ? 0.0 : Tt.c[k] * iv;
        xn.x = d.x - cc * xn.x;
        xn.y = d.y - cc * xn.y;
        if (CYCLIC) { const double ee = Tt.e[(long long)k * M + t]; xn.x -= ee * X.x; xn.y -= ee * X.y; }
        spec[(long long)k * M + t] = xn;
    }
}

// N17 gauge: remove the dzf-weighted mean of p, i.e. of mode (0,0): one CTA.
__global__ void k_gauge(FzP P, double2 *__restrict__ spec, long long M)
{
    __shared__ double red[256];
    double s = 0.0, vol = 0.0;
    for (int k = threadIdx.x; k < P.nz; k += blockDim.x) {
        s += spec[(long long)k * M].x * P.dzf[k];
        vol += P.dzf[k];
    }
    red[threadIdx.x] = s;
    __syncthreads();
    for (int o = blockDim.x / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    const double tot = red[0];
    __syncthreads();
    red[threadIdx.x] = vol;
    __syncthreads();
    for (int o = blockDim.x / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    const double mean = tot / red[0];
    for (int k = threadIdx.x; k < P.nz; k += blockDim.x) spec[(long long)k * M].x -= mean;
}
