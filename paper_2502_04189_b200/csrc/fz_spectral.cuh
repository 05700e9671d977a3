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

// ---------------------------------------------------------------- marching kernels, G line transforms in flight
// One CTA per x-mode.  A plane-step is a long dependent chain (three shared-memory FFT passes, then the recurrence),
// and there are only nxh independent x-modes, so with one transform per CTA an SM holds a warp or two and sits idle
// most of the time.  The CTA therefore runs G groups of ny/8 threads (blockDim = (ny/8, G)): group g owns the
// planes k = g, g+G, ...; it stages and transforms ITS plane on its own (cp.async one own-plane ahead, L2 prefetch
// two ahead, its own named barrier inside FzLineFFT), and only the recurrence itself is serial: its state -- d', c'
// (and the running f, h of a cyclic system), resp. x_{k+1} (and the separator X) -- lives in shared memory and is
// handed from the group of plane k to the group of plane k+1 through a named barrier (producer bar.arrive, consumer
// bar.sync).  Throughput per plane is then (FFT + recurrence)/G instead of their sum, until HBM binds.
// Per group: three padded lines (current | being prefetched | scratch, rotating), backward also two rows of INV (E).
// G = 1 (ny < 256: a group must be whole warps; ny = 1024: shared memory) degenerates to the single-transform kernel.
// G = 4 at ny = 256, where one transform per CTA leaves an SM with less than one warp (129 CTAs of 32 threads):
// measured 2.1x (0.209 -> 0.094 ms forward, 0.205 -> 0.100 ms backward at 256^3).  G = 1 at ny = 512: there two
// single-transform CTAs per SM already load the shared-memory pipe to ~40-50 %, and G = 2 or 3 (with the twiddles
// in registers, in L1 or in shared memory) measured 0.65-0.95 ms against 0.56-0.60 ms -- the handoff traffic and
// the table reads make that pipe the limiter.  G must keep groups whole warps (ny >= 256).
#define SPEC_FL 5    // lines per group: one fixed scratch line + a ring of SPEC_FL-1 (current | SPEC_FL-2 being prefetched by
                     // cp.async); backward: also SPEC_FL-1 rows of INV (E)
__host__ __device__ constexpr int spec_groups(int log2n) { return log2n == 8 ? 4 : 1; }

__host__ __device__ inline size_t fz_spec_smem(int log2n, bool fwd, bool cyclic)
{
    const int n = 1 << log2n, nt = n / 8, G = spec_groups(log2n);
    const size_t lines = (size_t)G * SPEC_FL * SPEC_LINE(n) * 16;
    const size_t state = G > 1 ? 1 : 0;   // the handoff buffers exist only when there is somebody to hand over to
    if (fwd) return lines + state * nt * 8 * (cyclic ? 48 : 24);
    return lines + (size_t)G * (SPEC_FL - 1) * n * 8 * (cyclic ? 2 : 1) + state * nt * 8 * 16 * (cyclic ? 2 : 1) + 16;
}

__device__ __forceinline__ void fz_bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void fz_bar_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }

// ---------------------------------------------------------------- forward: FFT_y + elimination
// thread jt of a group owns the systems m = jt + q*ny/8.  The pivots are recomputed on the fly (c' carried): the
// forward sweep reads no table.
template <bool CYCLIC, int LOG2N, int G>
__global__ void __launch_bounds__(G * ((1 << LOG2N) / 8), ((1 << LOG2N) >= 512 ? 2 : 1))
k_spec_fwd(FzP P, FzTri Tt, double2 *__restrict__ spec, const double2 *__restrict__ tw)
{
    extern __shared__ __align__(16) double2 sms[];
    constexpr int n = 1 << LOG2N, nt = n / 8, LN = SPEC_LINE(n);
    const int jt = threadIdx.x, g = threadIdx.y, nz = P.nz;
    double2 *scratch = sms + g * SPEC_FL * LN, *lines = scratch + LN;   // ring of RL = SPEC_FL-1 lines
    double2 *st_dp = sms + G * SPEC_FL * LN;                              // [q][jt]
    double *st_cp = reinterpret_cast<double *>(st_dp + 8 * nt);
    double2 *st_h = reinterpret_cast<double2 *>(st_cp + 8 * nt);   // cyclic only
    double *st_f = reinterpret_cast<double *>(st_h + 8 * nt);
    FzLineFFT<LOG2N, -1> fft;
    fft.init(tw, jt);
    if (G > 1) { fft.bar_id = 1 + G + g; fft.bar_n = nt; }
    const long long M = (long long)P.nxh * n, base = (long long)blockIdx.x * n;
    auto issue = [&](int k, int slot) {
        if (k < nz) {
            const double2 *gp = spec + (long long)k * M + base;
            double2 *d = lines + slot * LN;
#pragma unroll
            for (int q = 0; q < 8; ++q) { const int i = jt + q * nt; fz_cp_async16(d + SPEC_PADI(i), gp + i); }
        }
    };
#pragma unroll
    for (int d = 0; d < SPEC_FL - 2; ++d) { issue(g + d * G, d); fz_cp_async_commit(); }
    double lam[8];
    const double c_last = Tt.c[nz - 1], a_last = Tt.a[nz - 1];
    const double lamx = Tt.lamx[blockIdx.x];
#pragma unroll
    for (int q = 0; q < 8; ++q) lam[q] = lamx + Tt.lamy[jt + q * nt];
    double2 dp[8], h[8];
    double f[8], cp[8];
    int cur = 0;
    for (int k = g; k < nz; k += G) {
        // ring slots: cur | cur+1 .. cur+RL-2 in flight | cur-1 = the slot the previous plane left, issued now
        constexpr int RL = SPEC_FL - 1;
        const int nxt = cur + 1 == RL ? 0 : cur + 1, tgt = cur == 0 ? RL - 1 : cur - 1;
        fz_cp_async_wait<SPEC_FL - 3>();
        fft.sync();
        issue(k + (SPEC_FL - 2) * G, tgt);
        fz_cp_async_commit();
        double2 v[8];
        fft.smem_to_regs(jt, lines + cur * LN, scratch, v);
        // the recurrence state of plane k-1 (token from its group)
        if (k == 0) {
#pragma unroll
            for (int q = 0; q < 8; ++q) { dp[q] = make_double2(0, 0); h[q] = make_double2(0, 0); f[q] = c_last; cp[q] = 0.0; }
        } else if (G > 1) {
            fz_bar_sync(1 + g, 2 * nt);
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                dp[q] = st_dp[q * nt + jt]; cp[q] = st_cp[q * nt + jt];
                if (CYCLIC) { h[q] = st_h[q * nt + jt]; f[q] = st_f[q * nt + jt]; }
            }
        }
        double2 *out = spec + (long long)k * M + base;
        const double a = Tt.a[k], cfull = Tt.c[k];
        if (!CYCLIC || k < nz - 1) {
            const bool pen = CYCLIC && k == nz - 2;       // row nz-2 of a cyclic system
            const double ck = pen ? 0.0 : cfull, fadd = pen ? a_last : 0.0;
            // N17: x_{nz-1} = 0 for the singular mode (walls); its thread is (l, m) = (0, 0), q = 0
            const bool sing = !CYCLIC && k == nz - 1 && blockIdx.x == 0 && jt == 0;
#pragma unroll
            for (int q = 0; q < 8; ++q) {
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
            }
            if (G > 1 && k < nz - 1) {   // hand the state to the group of plane k+1
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    st_dp[q * nt + jt] = dp[q]; st_cp[q * nt + jt] = cp[q];
                    if (CYCLIC) { st_h[q * nt + jt] = h[q]; st_f[q * nt + jt] = f[q]; }
                }
                fz_bar_arrive(1 + (g + 1 == G ? 0 : g + 1), 2 * nt);
            }
#pragma unroll
            for (int q = 0; q < 8; ++q) out[jt + q * nt] = dp[q];
        } else {   // last row of a cyclic system: the separator X
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const int m = jt + q * nt;
                const double gi = Tt.ginv[base + m];
                out[m] = make_double2((v[q].x - h[q].x) * gi, (v[q].y - h[q].y) * gi);
            }
        }
        cur = nxt;
    }
    fz_cp_async_wait<0>();
}

// ---------------------------------------------------------------- backward: substitution + inverse FFT_y
// k descends from nz-1 to 0 (step s = nz-1-k; group g owns the steps s = g, g+G, ...).  scal[2] receives the
// dzf-weighted mean of mode (0,0) (gauge, N17), accumulated in plane order under the token.
template <bool CYCLIC, int LOG2N, int G>
__global__ void __launch_bounds__(G * ((1 << LOG2N) / 8), ((1 << LOG2N) >= 512 ? 2 : 1))
k_spec_bwd(FzP P, FzTri Tt, double2 *__restrict__ spec, const double2 *__restrict__ tw,
           double *__restrict__ scal)
{
    extern __shared__ __align__(16) double2 sms[];
    constexpr int n = 1 << LOG2N, nt = n / 8, LN = SPEC_LINE(n), NT = CYCLIC ? 2 : 1;
    const int jt = threadIdx.x, g = threadIdx.y, nz = P.nz;
    constexpr int RR = SPEC_FL - 1;                                 // ring of coefficient rows: current + in flight
    double2 *scratch = sms + g * SPEC_FL * LN, *lines = scratch + LN;   // ring of RR lines
    double *rows0 = reinterpret_cast<double *>(sms + G * SPEC_FL * LN);
    double *rows = rows0 + g * RR * n * NT;                         // [slot][INV | E][n]
    double2 *st_x = reinterpret_cast<double2 *>(rows0 + G * RR * n * NT);   // [q][jt]
    double2 *st_X = st_x + 8 * nt;                                  // cyclic only
    double *st_acc = reinterpret_cast<double *>(st_x + (G > 1 ? 8 * nt * NT : 0));   // G = 1: no handoff buffers
    FzLineFFT<LOG2N, +1> fft;
    fft.init(tw, jt);
    if (G > 1) { fft.bar_id = 1 + G + g; fft.bar_n = nt; }
    const long long M = (long long)P.nxh * n, base = (long long)blockIdx.x * n;
    auto issue = [&](int s, int slot, int rslot) {   // step s handles plane k = nz-1-s
        if (s < nz) {
            const int k = nz - 1 - s;
            const double2 *gp = spec + (long long)k * M + base;
            double2 *d = lines + slot * LN;
#pragma unroll
            for (int q = 0; q < 8; ++q) { const int i = jt + q * nt; fz_cp_async16(d + SPEC_PADI(i), gp + i); }
            const double *gi = Tt.inv + (long long)k * M + base;
            const double *ge = Tt.e + (long long)k * M + base;
            double *dr = rows + rslot * n * NT;
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int i = 2 * (jt + q * nt);
                fz_cp_async16(dr + i, gi + i);
                if (CYCLIC) fz_cp_async16(dr + n + i, ge + i);
            }
        }
    };
#pragma unroll
    for (int d = 0; d < SPEC_FL - 2; ++d) { issue(g + d * G, d, d); fz_cp_async_commit(); }
    double2 xn[8], X[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) { xn[q] = make_double2(0, 0); X[q] = make_double2(0, 0); }
    const int nrow = CYCLIC ? nz - 1 : nz;
    const bool gauge = blockIdx.x == 0 && jt == 0;   // owner of mode (l, m) = (0, 0)
    int cur = 0;
    bool first = true;
    for (int s = g; s < nz; s += G) {
        const int k = nz - 1 - s;
        const int nxt = cur + 1 == RR ? 0 : cur + 1, tgt = cur == 0 ? RR - 1 : cur - 1;   // lines and rows rotate together
        fz_cp_async_wait<SPEC_FL - 3>();
        fft.sync();
        issue(s + (SPEC_FL - 2) * G, tgt, tgt);
        fz_cp_async_commit();
        double2 *ln = lines + cur * LN;
        const double *iv = rows + cur * n * NT, *ev = iv + n;
        if (G > 1 && s > 0) {   // x_{k+1} (and, once, the separator) from the group of plane k+1
            fz_bar_sync(1 + g, 2 * nt);
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                xn[q] = st_x[q * nt + jt];
                if (CYCLIC && first) X[q] = st_X[q * nt + jt];
            }
        }
        first = false;
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
        if (gauge) {
            double acc = s == 0 ? 0.0 : st_acc[0], vol = s == 0 ? 0.0 : st_acc[1];
            acc += xn[0].x * P.dzf[k];
            vol += P.dzf[k];
            st_acc[0] = acc; st_acc[1] = vol;
            if (s == nz - 1) scal[2] = acc / vol;
        }
        if (G > 1 && s < nz - 1) {
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                st_x[q * nt + jt] = xn[q];
                if (CYCLIC && s == 0) st_X[q * nt + jt] = X[q];
            }
            fz_bar_arrive(1 + (g + 1 == G ? 0 : g + 1), 2 * nt);
        }
        double2 v[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) v[q] = xn[q];
        const double2 *res = fft.regs_to_smem(jt, ln, scratch, v);
        double2 *out = spec + (long long)k * M + base;
#pragma unroll
        for (int q = 0; q < 8; ++q) { const int m = jt + q * nt; out[m] = res[SPEC_PADI(m)]; }
        cur = nxt;
    }
    fz_cp_async_wait<0>();
}

// ---------------------------------------------------------------- host-side dispatch over log2(ny)
// which: 0 forward sweep, 1 backward sweep, < 0: shared-memory opt-in of both kernels (once, at fizzy_create)
template <bool CYCLIC, int LOG2N>
cudaError_t fz_spec_launch_one(int which, const FzP &P, const FzTri &Tt, double2 *spec, const double2 *tw,
                               double *scal, cudaStream_t st)
{
    constexpr int n = 1 << LOG2N, GF = spec_groups(LOG2N), GB = spec_groups(LOG2N);
    const size_t sf = fz_spec_smem(LOG2N, true, CYCLIC), sb = fz_spec_smem(LOG2N, false, CYCLIC);
    if (which < 0) {
        cudaError_t e = cudaFuncSetAttribute(k_spec_fwd<CYCLIC, LOG2N, GF>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sf);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_spec_bwd<CYCLIC, LOG2N, GB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sb);
        return e;
    }
    if (which == 0) k_spec_fwd<CYCLIC, LOG2N, GF><<<P.nxh, dim3(n / 8, GF), sf, st>>>(P, Tt, spec, tw);
    else k_spec_bwd<CYCLIC, LOG2N, GB><<<P.nxh, dim3(n / 8, GB), sb, st>>>(P, Tt, spec, tw, scal);
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
