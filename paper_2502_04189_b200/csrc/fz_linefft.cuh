// fz_linefft.cuh -- complex FFT of ONE line of N = 2^LOG2N points by N/8 threads, for kernels that
// transform the same kind of line again and again (k_spec_fwd / k_spec_bwd march over z planes).
// Stockham autosort, radix-8 passes plus one radix-4 or radix-2 pass, out of place between two
// padded shared-memory buffers (element i at i + (i >> 3): conflict free for every pass), so a
// pass costs ONE barrier.  The twiddles of a thread are the same for every line it will ever
// transform, so they are computed once (init) and live in registers.  The first pass can take its
// inputs from registers and, when LOG2N is a multiple of 3, the last pass leaves its outputs in
// registers: thread jt then holds the elements m = jt + q*N/8, q = 0..7.
#pragma once
#include "fz_common.cuh"
#include "fz_fft.cuh"

#define FZL_PADI(i_) ((i_) + ((i_) >> 3))

// TWREG = false: a thread that transforms only one line reads its twiddles from the table when a pass
// needs them (L1 hits) instead of holding them in registers.
template <int LOG2N, int SGN, bool TWREG = true>
struct FzLineFFT {
    static constexpr int N = 1 << LOG2N, NP8 = LOG2N / 3, REM = LOG2N % 3, T8 = N / 8;
    static constexpr int R2 = 1 << REM, NB = 8 / R2;          // remainder pass: radix R2, NB butterflies per thread
    static constexpr bool OUT_IN_REGS = (REM == 0);
    double2 w8[(TWREG && NP8 > 1) ? NP8 - 1 : 1][7];
    double2 wr[(TWREG && REM) ? NB : 1][REM ? R2 - 1 : 1];
    const double2 *twp;
    // barrier between passes: the whole CTA (bar_id = 0) or only the bar_n threads (a multiple of 32) that share
    // named barrier bar_id -- several independent line transforms can then be in flight in one CTA
    int bar_id = 0, bar_n = 0;
    __device__ __forceinline__ void sync() const
    {
        if (bar_id == 0) __syncthreads();
        else asm volatile("bar.sync %0, %1;" ::"r"(bar_id), "r"(bar_n) : "memory");
    }

    __device__ __forceinline__ double2 twv(int q) const
    {
        double2 t = twp[q];
        if (SGN > 0) t.y = -t.y;
        return t;
    }

    // tw[q] = exp(-2 pi i q / N); jt = thread index within the line
    __device__ __forceinline__ void init(const double2 *__restrict__ tw, int jt)
    {
        twp = tw;
        if (!TWREG) return;
        int Ns = 8;
#pragma unroll
        for (int p = 1; p < NP8; ++p) {
            const int kk = jt & (Ns - 1), M = N / (Ns * 8);
#pragma unroll
            for (int r = 1; r < 8; ++r) {
                double2 t = tw[r * kk * M];
                if (SGN > 0) t.y = -t.y;
                w8[p - 1][r - 1] = t;
            }
            Ns <<= 3;
        }
        if (REM) {
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                const int j = jt + b * T8;   // Ns = N / R2 > j, so kk = j and M = 1
#pragma unroll
                for (int r = 1; r < R2; ++r) {
                    double2 t = tw[r * j];
                    if (SGN > 0) t.y = -t.y;
                    wr[b][r - 1] = t;
                }
            }
        }
    }

    // radix-8 pass number p (Ns = 8^p) of thread jt
    template <bool IN_REG, bool OUT_REG>
    __device__ __forceinline__ void pass8(int p, int jt, double2 (&v)[8], const double2 *src, double2 *dst) const
    {
        if (!IN_REG) {
#pragma unroll
            for (int r = 0; r < 8; ++r) v[r] = src[FZL_PADI(jt + r * T8)];
        }
        if (p > 0) {
            const int Nsp = 1 << (3 * p), kt = (jt & (Nsp - 1)) * (N / (Nsp * 8));
            if (TWREG) {
#pragma unroll
                for (int r = 1; r < 8; ++r) v[r] = fz_cmul(v[r], w8[p - 1][r - 1]);
            } else {
                // ONE table read per pass; w^2 .. w^7 by six complex products (depth 3, a few ulp): seven scattered
                // 16-byte reads per pass made the L1 data pipe the limiter of the x transforms (ncu r2a: 94 %)
                const double2 w1 = twv(kt), w2 = fz_cmul(w1, w1), w3 = fz_cmul(w2, w1), w4 = fz_cmul(w2, w2);
                v[1] = fz_cmul(v[1], w1); v[2] = fz_cmul(v[2], w2); v[3] = fz_cmul(v[3], w3); v[4] = fz_cmul(v[4], w4);
                v[5] = fz_cmul(v[5], fz_cmul(w4, w1)); v[6] = fz_cmul(v[6], fz_cmul(w4, w2)); v[7] = fz_cmul(v[7], fz_cmul(w4, w3));
            }
        }
        fz_dft8<SGN>(v);
        if (!OUT_REG) {
            const int Ns = 1 << (3 * p);
            const int kk = jt & (Ns - 1), base = (jt - kk) * 8 + kk;
#pragma unroll
            for (int r = 0; r < 8; ++r) dst[FZL_PADI(base + r * Ns)] = v[r];
        }
    }

    // remainder pass (radix 4 or 2), shared -> shared
    __device__ __forceinline__ void passr(int jt, const double2 *src, double2 *dst) const
    {
        constexpr int Ns = 1 << (3 * NP8), T = N / R2;
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            const int j = jt + b * T8;
            double2 u[R2];
#pragma unroll
            for (int r = 0; r < R2; ++r) u[r] = src[FZL_PADI(j + r * T)];
#pragma unroll
            for (int r = 1; r < R2; ++r) u[r] = fz_cmul(u[r], TWREG ? wr[b][r - 1] : twv(r * j));
            if constexpr (R2 == 4) fz_dft4<SGN>(u[0], u[1], u[2], u[3]);
            else fz_dft2<SGN>(u[0], u[1]);
            const int kk = j & (Ns - 1), base = (j - kk) * R2 + kk;
#pragma unroll
            for (int r = 0; r < R2; ++r) dst[FZL_PADI(base + r * Ns)] = u[r];
        }
    }

    // Input line in shared buffer A (visible to all threads), scratch buffer B.  On return thread jt
    // holds element m = jt + q*T8 in v[q].  Buffers A and B may both be overwritten.
    __device__ __forceinline__ void smem_to_regs(int jt, double2 *A, double2 *B, double2 (&v)[8]) const
    {
        double2 *cur = A, *oth = B;
#pragma unroll
        for (int p = 0; p < NP8; ++p) {
            if (OUT_IN_REGS && p == NP8 - 1) { pass8<false, true>(p, jt, v, cur, oth); return; }
            pass8<false, false>(p, jt, v, cur, oth);
            sync();
            double2 *t = cur; cur = oth; oth = t;
        }
        passr(jt, cur, oth);
        sync();
#pragma unroll
        for (int q = 0; q < 8; ++q) v[q] = oth[FZL_PADI(jt + q * T8)];
    }

    // Input element m = jt + q*T8 in v[q]; B must not be in use by any thread (A may still be read by
    // other threads until the first barrier inside).  Returns the shared buffer (A or B) that holds
    // the transformed line in natural (padded) order, visible to all threads.
    __device__ __forceinline__ double2 *regs_to_smem(int jt, double2 *A, double2 *B, double2 (&v)[8]) const
    {
        double2 *cur = A, *oth = B;   // pass p writes into `oth`
        pass8<true, false>(0, jt, v, cur, oth);
        sync();
        { double2 *t = cur; cur = oth; oth = t; }
#pragma unroll
        for (int p = 1; p < NP8; ++p) {
            pass8<false, false>(p, jt, v, cur, oth);
            sync();
            double2 *t = cur; cur = oth; oth = t;
        }
        if (REM) {
            passr(jt, cur, oth);
            sync();
            double2 *t = cur; cur = oth; oth = t;
        }
        return cur;
    }
    // Input element jt + r*T8 in v[r] (registers), output element jt + q*T8 in v[q].  Pass 0 writes X; Y is written
    // only after the barrier that follows pass 0, so the caller's inputs may live in memory that Y aliases.
    __device__ __forceinline__ void regs_to_regs(int jt, double2 *X, double2 *Y, double2 (&v)[8]) const
    {
        if (OUT_IN_REGS && NP8 == 1) { pass8<true, true>(0, jt, v, Y, X); return; }
        pass8<true, false>(0, jt, v, Y, X);
        sync();
        double2 *cur = X, *oth = Y;
#pragma unroll
        for (int p = 1; p < NP8; ++p) {
            if (OUT_IN_REGS && p == NP8 - 1) { pass8<false, true>(p, jt, v, cur, oth); return; }
            pass8<false, false>(p, jt, v, cur, oth);
            sync();
            double2 *t = cur; cur = oth; oth = t;
        }
        passr(jt, cur, oth);
        sync();
#pragma unroll
        for (int q = 0; q < 8; ++q) v[q] = oth[FZL_PADI(jt + q * T8)];
    }
};
