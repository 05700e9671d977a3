// fz_spectral.cuh -- S4b-d fused: complex FFT along y and the per-wavenumber tridiagonal solve in z
// in ONE pass over the half-spectrum per direction (kernel groups (c)+(d) of BASELINE.json:5;
// PAPER.md:36 "fast direct FFT solver"; readings N17 gauge, N18 periodic z = cyclic system).
//
// Spectrum layout: spec[(k*nxh + l)*ny + m] (double2), m fastest: every y line is ny contiguous
// complex numbers.  One CTA owns one x-mode l and ALL of its (m, k): it marches over the planes k,
//   forward  (k_spec_fwd): line k arrives by cp.async -> FFT_y in shared memory -> forward
//            elimination step of the ny tridiagonal systems (each thread owns 8 of them, state in
//            registers) -> d'_k written back in place;
//   backward (k_spec_bwd): k descending: d'_k arrives -> back substitution step -> inverse FFT_y in
//            shared memory -> line k of the solution written back in place.
// HBM sees one read and one write of the spectrum per direction (plus the elimination tables),
// instead of the six reads/writes of separate FFT_y, Thomas (two sweeps) and inverse FFT_y kernels.
//
// Tridiagonal system of mode (l, m), lam = lam_x(l) + lam_y(m):
//   a_k x_{k-1} + (b_k + lam) x_k + c_k x_{k+1} = d_k,  a_k = 1/(dzf[k] dzc[k-1]), c_k = 1/(dzf[k] dzc[k]),
//   b_k = -(a_k + c_k);  walls: a_0 = c_{nz-1} = 0;  periodic z: cyclic.
// The matrix is real and fixed, so its elimination is done once at fizzy_create (k_tri_tables):
//   INV[k] = 1/(pivot_k);  forward d'_k = (d_k - a_k d'_{k-1}) INV[k];  backward x_k = d'_k - c_k INV[k] x_{k+1}.
// Cyclic systems use the last unknown X = x_{nz-1} as separator: rows 0..nz-2 are eliminated carrying
// the fill-in column E[k] (coefficient of X), the last row is reduced alongside (running coefficient
// f, pivot g -> GINV): X = (d_{nz-1} - sum_k f_k d'_k) GINV, x_k = d'_k - c_k INV[k] x_{k+1} - E[k] X.
// The singular mode (0,0) gets GINV = 0 (cyclic) or INV[nz-1] = 0 (walls): x_{nz-1} = 0 (N17); the
// dzf-weighted mean of that mode is accumulated by the thread that owns it and written to
// scal[2], and k_fftx_inv subtracts it in physical space.
#pragma once
#include "fz_common.cuh"
#include "fz_fft.cuh"
#include "fz_linefft.cuh"

struct FzTri {
    const double *a, *c;        // nz each (1-D)
    const double *lamx, *lamy;  // nxh, ny
    double *inv, *e;            // [nz][nxh][ny]  (e: cyclic only)
    double *ginv;               // [nxh][ny]      (cyclic only)
    int cyclic;
};

#define SPEC_RING 4
// padded position of element i of a line (one double2 of padding per 8 elements)
#define SPEC_PADI(i_) ((i_) + ((i_) >> 3))
#define SPEC_LINE(n_) ((n_) + ((n_) >> 3))

// pivot of row k: b_k + lam - a_k c'_{k-1}, b_k = -(a_k + c_k); one spelling for the table and the kernels
__device__ __forceinline__ double fz_tri_den(double a, double c, double lam, double cp)
{
    return fma(-a, cp, lam - (a + c));
}

__global__ void k_tri_tables(FzP P, FzTri Tt)
{
    const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    const long long M = (long long)P.nxh * P.ny;
    if (t >= M) return;
    const int m = (int)(t % P.ny), l = (int)(t / P.ny);
    const double lam = Tt.lamx[l] + Tt.lamy[m];
    const int n = P.nz;
    if (!Tt.cyclic) {
        double cp = 0.0;
        for (int k = 0; k < n; ++k) {
            const double a = Tt.a[k], c = Tt.c[k];
            const double den = fz_tri_den(a, c, lam, cp);
            double inv = fz_rcp_signed(den);      // the same pivot, bit for bit, that k_spec_fwd recomputes
            if (t == 0 && k == n - 1) inv = 0.0;  // N17: x_{nz-1} = 0 for the singular mode
            Tt.inv[(long long)k * M + t] = inv;
            cp = c * inv;
        }
    } else {
        double cp = 0.0, e = 0.0;
        double f = Tt.c[n - 1];                        // coefficient of x_0 in the last row
        double g = -(Tt.a[n - 1] + Tt.c[n - 1]) + lam;  // coefficient of X in the last row
        for (int k = 0; k <= n - 2; ++k) {
            const double a = Tt.a[k];
            const double c = (k == n - 2) ? 0.0 : Tt.c[k];
            const double den = fz_tri_den(a, Tt.c[k], lam, cp);
            const double inv = fz_rcp_signed(den);
            double ek = (k == 0) ? a * inv : -a * e * inv;
            if (k == n - 2) ek += Tt.c[k] * inv;   // c_{n-2} multiplies X as well
            const double fk = (k == n - 2) ? f + Tt.a[n - 1] : f;
            Tt.inv[(long long)k * M + t] = inv;
            Tt.e[(long long)k * M + t] = ek;
            g -= fk * ek;
            cp = c * inv;
            f = -fk * cp;
            e = ek;
        }
        Tt.inv[(long long)(n - 1) * M + t] = 0.0;
        Tt.e[(long long)(n - 1) * M + t] = 0.0;
        Tt.ginv[t] = (t == 0) ? 0.0 : 1.0 / g;  // N17
    }
}

// shared memory: scratch line | ring of SPEC_RING padded lines | `tables` rings of coefficient rows
// (forward sweep: none; backward: INV, and E when z is periodic)
__host__ __device__ inline size_t fz_spec_smem(int n, int tables)
{
    return (size_t)SPEC_LINE(n) * 16 + (size_t)SPEC_RING * ((size_t)SPEC_LINE(n) * 16 + (size_t)n * 8 * tables);
}

// ---------------------------------------------------------------- forward: FFT_y + elimination
// grid = nxh CTAs (one x-mode each), block = ny/8 threads; thread jt owns the systems m = jt + q*ny/8.
template <bool CYCLIC, int LOG2N>
__global__ void __launch_bounds__(128)
k_spec_fwd(FzP P, FzTri Tt, double2 *__restrict__ spec, const double2 *__restrict__ tw)
{
    extern __shared__ __align__(16) double2 sms[];
    constexpr int n = 1 << LOG2N, nt = n / 8, LN = SPEC_LINE(n);
    const int jt = threadIdx.x, nz = P.nz;
    double2 *scratch = sms, *lines = sms + LN;
    FzLineFFT<LOG2N, -1> fft;
    fft.init(tw, jt);
    const long long M = (long long)P.nxh * n, base = (long long)blockIdx.x * n;
    auto issue = [&](int k) {
        if (k < nz) {
            const int slot = k & (SPEC_RING - 1);
            const double2 *g = spec + (long long)k * M + base;
            double2 *d = lines + slot * LN;
#pragma unroll
            for (int q = 0; q < 8; ++q) { const int i = jt + q * nt; fz_cp_async16(d + SPEC_PADI(i), g + i); }
        }
    };
    for (int p = 0; p < SPEC_RING - 1; ++p) { issue(p); fz_cp_async_commit(); }
    double2 dp[8], h[8], v[8];
    double f[8], lam[8], cp[8];   // the pivots are recomputed on the fly (c' carried): the forward sweep reads no table
    const double c_last = Tt.c[nz - 1], a_last = Tt.a[nz - 1];
    const double lamx = Tt.lamx[blockIdx.x];
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        dp[q] = make_double2(0, 0); h[q] = make_double2(0, 0); f[q] = c_last;
        lam[q] = lamx + Tt.lamy[jt + q * nt]; cp[q] = 0.0;
    }
    for (int k = 0; k < nz; ++k) {
        fz_cp_async_wait<SPEC_RING - 2>();
        __syncthreads();
        issue(k + SPEC_RING - 1);
        fz_cp_async_commit();
        fft.smem_to_regs(jt, lines + (k & (SPEC_RING - 1)) * LN, scratch, v);
        double2 *out = spec + (long long)k * M + base;
        const double a = Tt.a[k], cfull = Tt.c[k];
        if (!CYCLIC || k < nz - 1) {
            const bool pen = CYCLIC && k == nz - 2;       // row nz-2 of a cyclic system
            const double ck = pen ? 0.0 : cfull, fadd = pen ? a_last : 0.0;
            // N17: x_{nz-1} = 0 for the singular mode (walls); its thread is (l, m) = (0, 0), q = 0
            const bool sing = !CYCLIC && k == nz - 1 && blockIdx.x == 0 && jt == 0;
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const int m = jt + q * nt;
                double inv = fz_rcp_signed(fz_tri_den(a, cfull, lam[q], cp[q]));
                if (q == 0 && sing) inv = 0.0;
                cp[q] = ck * inv;
                dp[q].x = (v[q].x - a * dp[q].x) * inv;
                dp[q].y = (v[q].y - a * dp[q].y) * inv;
                if (CYCLIC) {
                    const double fk = f[q] + fadd;
                    h[q].x += fk * dp[q].x;
                    h[q].y += fk * dp[q].y;
                    f[q] = -fk * (ck * inv);
                }
                out[m] = dp[q];
            }
        } else {   // last row of a cyclic system: the separator X
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const int m = jt + q * nt;
                const double gi = Tt.ginv[base + m];
                out[m] = make_double2((v[q].x - h[q].x) * gi, (v[q].y - h[q].y) * gi);
            }
        }
    }
    fz_cp_async_wait<0>();
}

// ---------------------------------------------------------------- backward: substitution + inverse FFT_y
// k descends from nz-1 to 0.  scal[2] receives the dzf-weighted mean of mode (0,0) (gauge, N17).
template <bool CYCLIC, int LOG2N>
__global__ void __launch_bounds__(128)
k_spec_bwd(FzP P, FzTri Tt, double2 *__restrict__ spec, const double2 *__restrict__ tw,
           double *__restrict__ scal)
{
    extern __shared__ __align__(16) double2 sms[];
    constexpr int n = 1 << LOG2N, nt = n / 8, LN = SPEC_LINE(n);
    const int jt = threadIdx.x, nz = P.nz;
    double2 *scratch = sms, *lines = sms + LN;
    double *invs = reinterpret_cast<double *>(lines + SPEC_RING * LN);
    double *es = invs + SPEC_RING * n;   // cyclic only
    FzLineFFT<LOG2N, +1> fft;
    fft.init(tw, jt);
    const long long M = (long long)P.nxh * n, base = (long long)blockIdx.x * n;
    auto issue = [&](int s) {   // step s handles plane k = nz-1-s
        if (s < nz) {
            const int slot = s & (SPEC_RING - 1), k = nz - 1 - s;
            const double2 *g = spec + (long long)k * M + base;
            double2 *d = lines + slot * LN;
#pragma unroll
            for (int q = 0; q < 8; ++q) { const int i = jt + q * nt; fz_cp_async16(d + SPEC_PADI(i), g + i); }
            const double *gi = Tt.inv + (long long)k * M + base;
            const double *ge = Tt.e + (long long)k * M + base;
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int i = 2 * (jt + q * nt);
                fz_cp_async16(invs + slot * n + i, gi + i);
                if (CYCLIC) fz_cp_async16(es + slot * n + i, ge + i);
            }
        }
    };
    for (int p = 0; p < SPEC_RING - 1; ++p) { issue(p); fz_cp_async_commit(); }
    double2 xn[8], X[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) { xn[q] = make_double2(0, 0); X[q] = make_double2(0, 0); }
    const int nrow = CYCLIC ? nz - 1 : nz;
    const bool gauge = blockIdx.x == 0 && jt == 0;   // owner of mode (l, m) = (0, 0)
    double acc = 0.0, vol = 0.0;
    for (int s = 0; s < nz; ++s) {
        const int k = nz - 1 - s;
        fz_cp_async_wait<SPEC_RING - 2>();
        __syncthreads();
        issue(s + SPEC_RING - 1);
        fz_cp_async_commit();
        double2 *ln = lines + (s & (SPEC_RING - 1)) * LN;
        const double *iv = invs + (s & (SPEC_RING - 1)) * n, *ev = es + (s & (SPEC_RING - 1)) * n;
        const double ck = (k == nrow - 1) ? 0.0 : Tt.c[k];
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const int m = jt + q * nt;
            const double2 d = ln[SPEC_PADI(m)];
            const double cc = ck * iv[m];
            double2 x = make_double2(d.x - cc * xn[q].x, d.y - cc * xn[q].y);
            if (CYCLIC) {
                const double e = ev[m];
                x.x -= e * X[q].x;
                x.y -= e * X[q].y;
                if (k == nz - 1) X[q] = x;   // row nz-1 holds the separator itself (cc = e = 0)
            }
            xn[q] = x;
        }
        if (gauge) { acc += xn[0].x * P.dzf[k]; vol += P.dzf[k]; }
        double2 v[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) v[q] = xn[q];
        const double2 *res = fft.regs_to_smem(jt, ln, scratch, v);
        double2 *out = spec + (long long)k * M + base;
#pragma unroll
        for (int q = 0; q < 8; ++q) { const int m = jt + q * nt; out[m] = res[SPEC_PADI(m)]; }
    }
    if (gauge) scal[2] = acc / vol;
    fz_cp_async_wait<0>();
}

// ---------------------------------------------------------------- host-side dispatch over log2(ny)
// which: 0 forward sweep, 1 backward sweep, < 0: shared-memory opt-in of both kernels (once, at fizzy_create)
template <bool CYCLIC, int LOG2N>
cudaError_t fz_spec_launch_one(int which, const FzP &P, const FzTri &Tt, double2 *spec, const double2 *tw,
                               double *scal, cudaStream_t st)
{
    const int n = 1 << LOG2N;
    const size_t sf = fz_spec_smem(n, 0), sb = fz_spec_smem(n, CYCLIC ? 2 : 1);
    if (which < 0) {
        cudaError_t e = cudaFuncSetAttribute(k_spec_fwd<CYCLIC, LOG2N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sf);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_spec_bwd<CYCLIC, LOG2N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sb);
        return e;
    }
    if (which == 0) k_spec_fwd<CYCLIC, LOG2N><<<P.nxh, n / 8, sf, st>>>(P, Tt, spec, tw);
    else k_spec_bwd<CYCLIC, LOG2N><<<P.nxh, n / 8, sb, st>>>(P, Tt, spec, tw, scal);
    return cudaSuccess;
}

template <bool CYCLIC>
cudaError_t fz_spec_launch(int which, int log2n, const FzP &P, const FzTri &Tt, double2 *spec, const double2 *tw,
                           double *scal, cudaStream_t st)
{
    switch (log2n) {
#define FZ_CASE(L_) case L_: return fz_spec_launch_one<CYCLIC, L_>(which, P, Tt, spec, tw, scal, st);
        FZ_CASE(3) FZ_CASE(4) FZ_CASE(5) FZ_CASE(6) FZ_CASE(7) FZ_CASE(8) FZ_CASE(9) FZ_CASE(10)
#undef FZ_CASE
    }
    return cudaErrorInvalidValue;
}
