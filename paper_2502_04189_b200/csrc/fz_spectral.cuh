// fz_spectral.cuh -- S4b-d fused: complex FFT along y and the per-wavenumber tridiagonal solve in z
// in ONE pass over the half-spectrum per direction (kernel groups (c)+(d) of BASELINE.json:5;
// PAPER.md:36 "fast direct FFT solver"; readings N17 gauge, N18 periodic z = cyclic system).
//
// Spectrum layout: spec[(k*nxh + l)*ny + m] (double2), m fastest: every y line is ny contiguous
// complex numbers.  A CTA owns one x-mode l, ALL of its m and HALF of the planes k; it marches over them,
//   forward  (k_spec_fwd): line k arrives by cp.async -> FFT_y in shared memory -> elimination step of the
//            ny tridiagonal systems (each thread owns 8 of them, state in registers) -> d'_k written back in place;
//   backward (k_spec_bwd): d'_k arrives -> substitution step -> inverse FFT_y in shared memory -> line k of
//            the solution written back in place.
// HBM sees one read and one write of the spectrum per direction (plus the elimination tables),
// instead of the six reads/writes of separate FFT_y, Thomas (two sweeps) and inverse FFT_y kernels.
//
// Tridiagonal system of mode (l, m), lam = lam_x(l) + lam_y(m):
//   a_k x_{k-1} + (b_k + lam) x_k + c_k x_{k+1} = d_k,  a_k = 1/(dzf[k] dzc[k-1]), c_k = 1/(dzf[k] dzc[k]),
//   b_k = -(a_k + c_k);  walls: a_0 = c_{nz-1} = 0;  periodic z: cyclic.
//
// TWO-SIDED ("twisted") elimination.  A plane step is a long dependent chain (three shared-memory FFT passes, then
// the recurrence) and there are only nxh independent x-modes, so a single sweep over all nz planes leaves an SM
// with a warp or two and a serial path of nz steps.  The chain of unknowns is therefore eliminated from BOTH ends
// towards a middle row mid = (nz-1)/2 by two independent CTAs per x-mode (blockIdx.y = half): twice the warps,
// half the serial path.  With lo/hi = the coefficient towards the previous/next row IN SWEEP ORDER
// (top half, rows 0 .. mid-1 ascending: lo = a, hi = c; bottom half, rows kb .. mid+1 descending: lo = c, hi = a;
// kb = nz-1 with walls, nz-2 if cyclic) both halves run the same recurrence
//   pivot_s = b + lam - lo_s hi'_{s-1},  INV = 1/pivot,  hi'_s = hi_s INV,  d'_s = (d_s - lo_s d'_{s-1}) INV
// and leave  x_k + hi'_k x_next + e_k X = d'_k.  The middle row then reads  Pm x_mid + Q X = r1,
//   Pm = b_mid + lam - a_mid hi'_top - c_mid hi'_bot,   r1 = d_mid - a_mid d'_top - c_mid d'_bot,
// and the substitution runs from the middle outwards, again as two independent halves:
//   x_k = d'_k - hi'_k x_(towards the middle) - e_k X.
// Cyclic systems keep the last unknown X = x_{nz-1} as separator: the first row of either half couples to it
// (e_0 = lo_0 INV_0, e_s = -lo_s e_{s-1} INV_s) and the last row c x_0 + a x_{nz-2} + (b + lam) X = d_{nz-1} is reduced
// alongside by both halves (running coefficient f on the next unknown, f_0 = hi_{nz-1}; h = sum f_s d'_s;
// g = b + lam - sum f_s e_s), which leaves  F x_mid + g X = r2 = d_{nz-1} - h_top - h_bot,  F = f_top + f_bot.
// Everything that depends on the matrix only is set up once by k_tri_tables: INV[k], E[k] and the inverse of the
// 2x2 middle system per mode (MID).  The forward sweep recomputes its pivots (hi' carried in registers) and
// reads no table; it hands the two halves' contributions to r1, r2 over in SIDE (four lines per x-mode), since
// the backward CTAs of the two halves overwrite each other's input planes.
// The singular mode (0,0) gets X = 0 (cyclic) or INV[nz-1] = 0 (walls): x_{nz-1} = 0 (N17); the dzf-weighted mean
// of that mode is accumulated by the thread that owns it, one partial per half -> scal[2], scal[6], and
// k_fftx_inv subtracts their sum in physical space.
#pragma once
#include "fz_common.cuh"
#include "fz_fft.cuh"
#include "fz_linefft.cuh"

struct FzTri {
    const double *a, *c;        // nz each (1-D)
    const double *lamx, *lamy;  // nxh, ny
    double *inv, *e;            // [nz][nxh][ny]  (e: cyclic only)
    double *mid;                // walls: [nxh][ny] 1/Pm;  cyclic: [4][nxh][ny] inverse of the 2x2 middle system
    double2 *side;              // [4][nxh][ny]: r1 (top), r2 (top), r1 (bottom), r2 (bottom); r2: cyclic only
    int cyclic;
};

// padded position of element i of a line (one double2 of padding per 8 elements)
#define SPEC_PADI(i_) ((i_) + ((i_) >> 3))
#define SPEC_LINE(n_) ((n_) + ((n_) >> 3))

// pivot of a row: b + lam - lo hi'_{prev}, b = -(lo + hi); one spelling for the table and the kernels
__device__ __forceinline__ double fz_tri_den(double lo, double hi, double lam, double hp)
{
    return fma(-lo, hp, lam - (lo + hi));
}

// the rows of one half in sweep order
struct FzHalf {
    int S;          // eliminated rows
    int kfirst, dk; // row of step s: kfirst + dk*s
    const double *LO, *HI;
};
__device__ __forceinline__ int fz_tri_mid(int nz) { return (nz - 1) / 2; }
__device__ __forceinline__ FzHalf fz_tri_half(const FzTri &Tt, int nz, int half)
{
    const int mid = fz_tri_mid(nz), kb = Tt.cyclic ? nz - 2 : nz - 1;
    FzHalf H;
    H.S = half == 0 ? mid : kb - mid;
    H.kfirst = half == 0 ? 0 : kb;
    H.dk = half == 0 ? 1 : -1;
    H.LO = half == 0 ? Tt.a : Tt.c;
    H.HI = half == 0 ? Tt.c : Tt.a;
    return H;
}

__global__ void k_tri_tables(FzP P, FzTri Tt)
{
    const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    const long long M = (long long)P.nxh * P.ny;
    if (t >= M) return;
    const int m = (int)(t % P.ny), l = (int)(t / P.ny);
    const double lam = Tt.lamx[l] + Tt.lamy[m];
    const int n = P.nz, mid = fz_tri_mid(n);
    double hpl[2], el[2], fl[2], gsum = 0.0;
    for (int half = 0; half < 2; ++half) {
        const FzHalf H = fz_tri_half(Tt, n, half);
        double hp = 0.0, e = 0.0, f = Tt.cyclic ? H.HI[n - 1] : 0.0;
        for (int s = 0; s < H.S; ++s) {
            const int k = H.kfirst + H.dk * s;
            const double lo = H.LO[k], hi = H.HI[k];
            double inv = fz_rcp_signed(fz_tri_den(lo, hi, lam, hp));   // the same pivot, bit for bit, that k_spec_fwd recomputes
            if (!Tt.cyclic && half == 1 && s == 0 && t == 0) inv = 0.0;   // N17: x_{nz-1} = 0 for the singular mode
            Tt.inv[(long long)k * M + t] = inv;
            hp = hi * inv;
            if (Tt.cyclic) {
                e = (s == 0) ? lo * inv : -lo * e * inv;
                Tt.e[(long long)k * M + t] = e;
                gsum += f * e;
                f = -f * hp;
            }
        }
        hpl[half] = hp; el[half] = e; fl[half] = f;
    }
    const double am = Tt.a[mid], cm = Tt.c[mid];
    const double Pm = (lam - (am + cm)) - am * hpl[0] - cm * hpl[1];
    if (!Tt.cyclic) {
        Tt.mid[t] = 1.0 / Pm;
    } else {
        const double Q = -(am * el[0] + cm * el[1]), F = fl[0] + fl[1];
        const double g = (lam - (Tt.a[n - 1] + Tt.c[n - 1])) - gsum;
        const double det = Pm * g - Q * F;
        const bool sing = t == 0;   // N17: X = 0, the (redundant) last row is dropped
        Tt.mid[t] = sing ? 1.0 / Pm : g / det;
        Tt.mid[M + t] = sing ? 0.0 : -Q / det;
        Tt.mid[2 * M + t] = sing ? 0.0 : -F / det;
        Tt.mid[3 * M + t] = sing ? 0.0 : Pm / det;
    }
}

// ---------------------------------------------------------------- marching kernels, G line transforms in flight
// One CTA per x-mode and half.  The CTA runs G groups of ny/8 threads (blockDim = (ny/8, G)): group g owns the
// steps s = g, g+G, ... of its half; it stages and transforms ITS plane on its own (cp.async own-planes ahead, its own
// named barrier inside FzLineFFT), and only the recurrence itself is serial: its state -- d', hi' (and the running
// f, h of a cyclic system), resp. the previous x -- lives in shared memory and is handed from the group of step s to
// the group of step s+1 through a named barrier (producer bar.arrive, consumer bar.sync).  Throughput per plane is
// then (FFT + recurrence)/G instead of their sum, until HBM binds.
// G = 1 (ny < 256: a group must be whole warps; ny >= 512: shared memory) degenerates to the single-transform kernel.
// G = 4 at ny = 256, where one transform per CTA leaves an SM with about a warp: measured 2.1x in round 2.
// G = 1 at ny = 512: there four single-transform CTAs share an SM (56 KB of shared memory each at most).
#define SPEC_FL 5    // forward, lines per group: one fixed scratch line + a ring of SPEC_FL-1 (current | SPEC_FL-2 in flight)
#define SPEC_FLB 4   // backward: scratch + ring of 3 lines (current | 2 in flight) and a ring of 2 rows of INV (E)
__host__ __device__ constexpr int spec_groups(int log2n) { return log2n <= 8 ? 4 : 1; }
__host__ __device__ constexpr int spec_minb(int log2n) { return log2n == 9 ? 4 : (log2n >= 8 ? 2 : 1); }
// Short lines (ny < 256: fewer than 32 threads per transform): a group is still one whole warp and transforms
// MPG = 32/(ny/8) x-modes side by side, so that the named barriers see whole warps and a 128^3 grid is not solved by 130
// half-warps.  GT = threads per group.
__host__ __device__ constexpr int spec_mpg(int log2n) { return log2n >= 8 ? 1 : 32 / ((1 << log2n) / 8); }
__host__ __device__ constexpr int spec_gt(int log2n) { return log2n >= 8 ? (1 << log2n) / 8 : 32; }

__host__ __device__ inline size_t fz_spec_smem(int log2n, bool fwd, bool cyclic)
{
    const int n = 1 << log2n, G = spec_groups(log2n), MPG = spec_mpg(log2n), GT = spec_gt(log2n);
    const size_t state = G > 1 ? 1 : 0;   // the handoff buffers exist only when there is somebody to hand over to
    if (fwd) return (size_t)G * MPG * SPEC_FL * SPEC_LINE(n) * 16 + state * GT * 8 * (cyclic ? 48 : 24);
    return (size_t)G * MPG * SPEC_FLB * SPEC_LINE(n) * 16 + (size_t)G * MPG * 2 * n * 8 * (cyclic ? 2 : 1) + state * GT * 8 * 16 + 16;
}

__device__ __forceinline__ void fz_bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void fz_bar_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }

// ---------------------------------------------------------------- forward: FFT_y + elimination
// thread jt of a group owns the systems m = jt + q*ny/8.  Steps s = 0 .. S-1 eliminate the rows of the half; the
// tail step (the top half: row mid; the bottom half of a cyclic system: row nz-1) only transforms its plane and
// forms the half's contribution to r1 (and r2) in SIDE.
template <bool CYCLIC, int LOG2N, int G>
__global__ void __launch_bounds__(G * spec_gt(LOG2N), spec_minb(LOG2N))
k_spec_fwd(FzP P, FzTri Tt, double2 *__restrict__ spec, const double2 *__restrict__ tw)
{
    extern __shared__ __align__(16) double2 sms[];
    constexpr int n = 1 << LOG2N, nt = n / 8, LN = SPEC_LINE(n), MPG = spec_mpg(LOG2N), GT = spec_gt(LOG2N), SL = MPG * LN;
    const int tx = threadIdx.x, jt = tx & (nt - 1), ms = tx / nt, g = threadIdx.y, nz = P.nz, half = blockIdx.y;
    // x-mode of this thread; a CTA past the last mode repeats it without storing (its threads still meet the barriers)
    const bool live = (int)blockIdx.x * MPG + ms < P.nxh;
    const int l = live ? (int)blockIdx.x * MPG + ms : P.nxh - 1;
    double2 *scratch = sms + (g * SPEC_FL * MPG + ms) * LN, *lines = scratch + SL;   // ring of RL = SPEC_FL-1 slots of MPG lines
    double2 *st_dp = sms + G * SPEC_FL * SL;                                          // [q][tx]
    double *st_hp = reinterpret_cast<double *>(st_dp + 8 * GT);
    double2 *st_h = reinterpret_cast<double2 *>(st_hp + 8 * GT);   // cyclic only
    double *st_f = reinterpret_cast<double *>(st_h + 8 * GT);
    FzLineFFT<LOG2N, -1> fft;
    fft.init(tw, jt);
    if (G > 1) { fft.bar_id = 1 + G + g; fft.bar_n = GT; }
    const FzHalf H = fz_tri_half(Tt, nz, half);
    const int mid = fz_tri_mid(nz);
    const bool has_tail = CYCLIC || half == 0;
    const int NS = H.S + (has_tail ? 1 : 0), ktail = half == 0 ? mid : nz - 1;
    const long long M = (long long)P.nxh * n, base = (long long)l * n;
    auto issue = [&](int s, int slot) {
        if (s < NS) {
            const int k = s < H.S ? H.kfirst + H.dk * s : ktail;
            const double2 *gp = spec + (long long)k * M + base;
            double2 *d = lines + slot * SL;
#pragma unroll
            for (int q = 0; q < 8; ++q) { const int i = jt + q * nt; fz_cp_async16(d + SPEC_PADI(i), gp + i); }
        }
    };
#pragma unroll
    for (int d = 0; d < SPEC_FL - 2; ++d) { issue(g + d * G, d); fz_cp_async_commit(); }
    double lam[8];
    const double f0 = H.HI[nz - 1], lom = H.LO[mid];
    const double lamx = Tt.lamx[l];
#pragma unroll
    for (int q = 0; q < 8; ++q) lam[q] = lamx + Tt.lamy[jt + q * nt];
    double2 dp[8], h[8];
    double f[8], hp[8];
    int cur = 0;
    for (int s = g; s < NS; s += G) {
        // ring slots: cur | cur+1 .. cur+RL-2 in flight | cur-1 = the slot the previous plane left, issued now
        constexpr int RL = SPEC_FL - 1;
        const int nxt = cur + 1 == RL ? 0 : cur + 1, tgt = cur == 0 ? RL - 1 : cur - 1;
        fz_cp_async_wait<SPEC_FL - 3>();
        fft.sync();
        issue(s + (SPEC_FL - 2) * G, tgt);
        fz_cp_async_commit();
        double2 v[8];
        fft.smem_to_regs(jt, lines + cur * SL, scratch, v);
        // the recurrence state of step s-1 (token from its group)
        if (s == 0) {
#pragma unroll
            for (int q = 0; q < 8; ++q) { dp[q] = make_double2(0, 0); h[q] = make_double2(0, 0); f[q] = f0; hp[q] = 0.0; }
        } else if (G > 1) {
            fz_bar_sync(1 + g, 2 * GT);
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                dp[q] = st_dp[q * GT + tx]; hp[q] = st_hp[q * GT + tx];
                if (CYCLIC) { h[q] = st_h[q * GT + tx]; f[q] = st_f[q * GT + tx]; }
            }
        }
        if (s < H.S) {
            const int k = H.kfirst + H.dk * s;
            double2 *out = spec + (long long)k * M + base;
            const double lo = H.LO[k], hi = H.HI[k];
            // N17: x_{nz-1} = 0 for the singular mode (walls): first row of the bottom half; its thread is (l, m) = (0, 0), q = 0
            const bool sing = !CYCLIC && half == 1 && s == 0 && l == 0 && jt == 0;
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                double inv = fz_rcp_signed(fz_tri_den(lo, hi, lam[q], hp[q]));
                if (q == 0 && sing) inv = 0.0;
                hp[q] = hi * inv;
                dp[q].x = (v[q].x - lo * dp[q].x) * inv;
                dp[q].y = (v[q].y - lo * dp[q].y) * inv;
                if (CYCLIC) {
                    h[q].x += f[q] * dp[q].x;
                    h[q].y += f[q] * dp[q].y;
                    f[q] = -f[q] * hp[q];
                }
            }
            if (G > 1 && s < NS - 1) {   // hand the state to the group of step s+1
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    st_dp[q * GT + tx] = dp[q]; st_hp[q * GT + tx] = hp[q];
                    if (CYCLIC) { st_h[q * GT + tx] = h[q]; st_f[q * GT + tx] = f[q]; }
                }
                fz_bar_arrive(1 + (g + 1 == G ? 0 : g + 1), 2 * GT);
            }
            if (live) {
#pragma unroll
                for (int q = 0; q < 8; ++q) out[jt + q * nt] = dp[q];
            }
            if (live && !has_tail && s == H.S - 1) {   // bottom half, walls: r1 contribution -c_mid d'_bot
                double2 *sd = Tt.side + 2 * M + base;
#pragma unroll
                for (int q = 0; q < 8; ++q) sd[jt + q * nt] = make_double2(-lom * dp[q].x, -lom * dp[q].y);
            }
        } else if (live) {   // tail: v = transformed row mid (top) / row nz-1 (bottom, cyclic)
            double2 *s1 = Tt.side + (half == 0 ? 0 : 2 * M) + base, *s2 = s1 + M;
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const int m = jt + q * nt;
                if (half == 0) {
                    s1[m] = make_double2(v[q].x - lom * dp[q].x, v[q].y - lom * dp[q].y);
                    if (CYCLIC) s2[m] = make_double2(-h[q].x, -h[q].y);
                } else {
                    s1[m] = make_double2(-lom * dp[q].x, -lom * dp[q].y);
                    s2[m] = make_double2(v[q].x - h[q].x, v[q].y - h[q].y);
                }
            }
        }
        cur = nxt;
    }
    fz_cp_async_wait<0>();
}

// ---------------------------------------------------------------- backward: substitution + inverse FFT_y
// From the middle outwards.  Top half: step 0 is row mid itself (x_mid from the middle system, no plane to load), step t
// handles row mid-t.  Bottom half: step t handles row mid+1+t; a cyclic system ends with the separator row nz-1 (X, no
// plane to load).  scal[2] / scal[6] receive the halves' parts of the dzf-weighted mean of mode (0,0) (gauge, N17),
// accumulated in plane order under the token.
template <bool CYCLIC, int LOG2N, int G>
__global__ void __launch_bounds__(G * spec_gt(LOG2N), spec_minb(LOG2N))
k_spec_bwd(FzP P, FzTri Tt, double2 *__restrict__ spec, const double2 *__restrict__ tw,
           double *__restrict__ scal)
{
    extern __shared__ __align__(16) double2 sms[];
    constexpr int n = 1 << LOG2N, nt = n / 8, LN = SPEC_LINE(n), NT = CYCLIC ? 2 : 1;
    constexpr int MPG = spec_mpg(LOG2N), GT = spec_gt(LOG2N), SL = MPG * LN, SR = MPG * n * NT;
    constexpr int RL = SPEC_FLB - 1;                                    // ring of lines: current + 2 in flight
    const int tx = threadIdx.x, jt = tx & (nt - 1), ms = tx / nt, g = threadIdx.y, nz = P.nz, half = blockIdx.y;
    const bool live = (int)blockIdx.x * MPG + ms < P.nxh;               // see k_spec_fwd
    const int l = live ? (int)blockIdx.x * MPG + ms : P.nxh - 1;
    double2 *scratch = sms + (g * SPEC_FLB * MPG + ms) * LN, *lines = scratch + SL;
    double *rows0 = reinterpret_cast<double *>(sms + G * SPEC_FLB * SL);
    double *rows = rows0 + (g * 2 * MPG + ms) * n * NT;                 // [slot: current | next][mode][INV | E][n]
    double2 *st_x = reinterpret_cast<double2 *>(rows0 + G * 2 * SR);    // [q][tx]
    double *st_acc = reinterpret_cast<double *>(st_x + (G > 1 ? 8 * GT : 0));   // G = 1: no handoff buffer
    FzLineFFT<LOG2N, +1> fft;
    fft.init(tw, jt);
    if (G > 1) { fft.bar_id = 1 + G + g; fft.bar_n = GT; }
    const FzHalf H = fz_tri_half(Tt, nz, half);
    const int mid = fz_tri_mid(nz);
    const int NSTEP = half == 0 ? mid + 1 : H.S + (CYCLIC ? 1 : 0);
    const long long M = (long long)P.nxh * n, base = (long long)l * n;
    // step t: a row with a plane to load (regular), or x_mid / X (special)
    auto special = [&](int t) { return half == 0 ? t == 0 : t == H.S; };
    auto plane = [&](int t) { return half == 0 ? mid - t : (t < H.S ? mid + 1 + t : nz - 1); };
    auto issue_rows = [&](int t, int rslot) {
        if (t < NSTEP && !special(t)) {
            const int k = plane(t);
            const double *gi = Tt.inv + (long long)k * M + base;
            const double *ge = Tt.e + (long long)k * M + base;
            double *dr = rows + rslot * SR;
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int i = 2 * (jt + q * nt);
                fz_cp_async16(dr + i, gi + i);
                if (CYCLIC) fz_cp_async16(dr + n + i, ge + i);
            }
        }
    };
    auto issue_line = [&](int t, int slot) {
        if (t < NSTEP && !special(t)) {
            const double2 *gp = spec + (long long)plane(t) * M + base;
            double2 *d = lines + slot * SL;
#pragma unroll
            for (int q = 0; q < 8; ++q) { const int i = jt + q * nt; fz_cp_async16(d + SPEC_PADI(i), gp + i); }
        }
    };
    // cp.async groups: a step first commits the rows of the group's NEXT step, then the line of the one after: with at
    // most ONE group pending (the line of the next step) both the line and the rows of the current step have landed
    issue_rows(g, 0); issue_line(g, 0); fz_cp_async_commit();
    issue_line(g + G, 1); fz_cp_async_commit();
    // the middle system: x_mid (and X) of the thread's 8 modes, from the halves' contributions in SIDE
    double2 xn[8], X[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const long long i = base + jt + q * nt;
        const double2 a1 = Tt.side[i], b1 = Tt.side[2 * M + i];
        const double2 r1 = make_double2(a1.x + b1.x, a1.y + b1.y);
        if (CYCLIC) {
            const double2 a2 = Tt.side[M + i], b2 = Tt.side[3 * M + i];
            const double2 r2 = make_double2(a2.x + b2.x, a2.y + b2.y);
            const double m11 = Tt.mid[i], m12 = Tt.mid[M + i], m21 = Tt.mid[2 * M + i], m22 = Tt.mid[3 * M + i];
            xn[q] = make_double2(m11 * r1.x + m12 * r2.x, m11 * r1.y + m12 * r2.y);
            X[q] = make_double2(m21 * r1.x + m22 * r2.x, m21 * r1.y + m22 * r2.y);
        } else {
            const double pi = Tt.mid[i];
            xn[q] = make_double2(r1.x * pi, r1.y * pi);
            X[q] = make_double2(0, 0);
        }
    }
    const bool gauge = l == 0 && jt == 0;   // owner of mode (l, m) = (0, 0)
    int cur = 0, rcur = 0;
    for (int t = g; t < NSTEP; t += G) {
        const int nxt = cur + 1 == RL ? 0 : cur + 1, tgt = cur == 0 ? RL - 1 : cur - 1;
        fz_cp_async_wait<1>();
        fft.sync();
        issue_rows(t + G, rcur ^ 1);
        fz_cp_async_commit();
        issue_line(t + 2 * G, tgt);
        fz_cp_async_commit();
        double2 *ln = lines + cur * SL;
        const double *iv = rows + rcur * SR, *ev = iv + n;
        if (G > 1 && t > 0) {   // the previous x from the group of step t-1
            fz_bar_sync(1 + g, 2 * GT);
#pragma unroll
            for (int q = 0; q < 8; ++q) xn[q] = st_x[q * GT + tx];
        }
        const int k = plane(t);
        if (!special(t)) {
            const double hi = H.HI[k];
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const int m = jt + q * nt;
                const double2 d = ln[SPEC_PADI(m)];
                const double cc = hi * iv[m];
                double2 x = make_double2(d.x - cc * xn[q].x, d.y - cc * xn[q].y);
                if (CYCLIC) {
                    const double e = ev[m];
                    x.x -= e * X[q].x;
                    x.y -= e * X[q].y;
                }
                xn[q] = x;
            }
        } else if (half == 1) {   // the separator row itself
#pragma unroll
            for (int q = 0; q < 8; ++q) xn[q] = X[q];
        }
        if (gauge) {
            double acc = t == 0 ? 0.0 : st_acc[0];
            acc += xn[0].x * P.dzf[k];
            st_acc[0] = acc;
            if (t == NSTEP - 1) scal[half == 0 ? 2 : 6] = acc / P.lz;
        }
        if (G > 1 && t < NSTEP - 1) {
#pragma unroll
            for (int q = 0; q < 8; ++q) st_x[q * GT + tx] = xn[q];
            fz_bar_arrive(1 + (g + 1 == G ? 0 : g + 1), 2 * GT);
        }
        double2 v[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) v[q] = xn[q];
        const double2 *res = fft.regs_to_smem(jt, ln, scratch, v);
        double2 *out = spec + (long long)k * M + base;
        if (live) {
#pragma unroll
            for (int q = 0; q < 8; ++q) { const int m = jt + q * nt; out[m] = res[SPEC_PADI(m)]; }
        }
        cur = nxt;
        rcur ^= 1;
    }
    fz_cp_async_wait<0>();
}

// ---------------------------------------------------------------- host-side dispatch over log2(ny)
// which: 0 forward sweep, 1 backward sweep, < 0: shared-memory opt-in of both kernels (once, at fizzy_create)
template <bool CYCLIC, int LOG2N>
cudaError_t fz_spec_launch_one(int which, const FzP &P, const FzTri &Tt, double2 *spec, const double2 *tw,
                               double *scal, cudaStream_t st)
{
    constexpr int GF = spec_groups(LOG2N), GB = spec_groups(LOG2N), MPG = spec_mpg(LOG2N);
    const size_t sf = fz_spec_smem(LOG2N, true, CYCLIC), sb = fz_spec_smem(LOG2N, false, CYCLIC);
    if (which < 0) {
        cudaError_t e = cudaFuncSetAttribute(k_spec_fwd<CYCLIC, LOG2N, GF>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sf);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_spec_bwd<CYCLIC, LOG2N, GB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sb);
        return e;
    }
    if (which == 0) k_spec_fwd<CYCLIC, LOG2N, GF><<<dim3((P.nxh + MPG - 1) / MPG, 2), dim3(spec_gt(LOG2N), GF), sf, st>>>(P, Tt, spec, tw);
    else k_spec_bwd<CYCLIC, LOG2N, GB><<<dim3((P.nxh + MPG - 1) / MPG, 2), dim3(spec_gt(LOG2N), GB), sb, st>>>(P, Tt, spec, tw, scal);
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
