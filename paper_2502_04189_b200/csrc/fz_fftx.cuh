// fz_fftx.cuh -- S4a + S4b (x part) and S4d (x part): Poisson right-hand side and the real<->complex
// FFTs along x (kernel group (c) of BASELINE.json:5; "fast direct FFT solver").
//
// Two real lines (j, j+1) are transformed as one complex line z = a + i b by a group of nx/8
// threads (FzLineFFT: twiddles in registers, padded out-of-place passes); a CTA holds FX_PAIRS
// groups = 2*FX_PAIRS consecutive j lines of one plane k, so that the half-spectrum goes out in
// runs of 2*FX_PAIRS consecutive j:  spec[(k*nxh + l)*ny + j]  (y lines contiguous, fz_spectral.cuh).
//   A_l = (Z_l + conj Z_{n-l})/2,  B_l = (Z_l - conj Z_{n-l})/(2i)          (forward untangling)
//   Z_l = A_l + i B_l,  Z_{n-l} = conj(A_l) + i conj(B_l)                   (backward tangling)
// DIV = true: the real input is the Poisson right-hand side assembled on the fly,
//   b = coef * D(u**)  (BASELINE.json:5(iv) with the p_hat term folded into u**, D2);
// DIV = false: the real input is read from `src` (fizzy_poisson_solve).
#pragma once
#include "fz_common.cuh"
#include "fz_linefft.cuh"

// line pairs per CTA (2 buffers x pairs x padded line x 16 B of shared memory).  Forward: 2 pairs from
// nx = 512 up (64-byte runs in the spectrum, merged in L2 with the neighbouring CTA's; five 128-thread CTAs
// per SM at ~95 registers measured 20 % faster than three 256-thread CTAs).  Backward: 4 pairs (128-byte
// runs when READING the spectrum matter), 2 at nx = 1024 so that three CTAs still fit an SM.
__host__ __device__ constexpr int fx_pairs(int log2n, bool inverse)
{
    return inverse ? (log2n >= 10 ? 2 : 4) : (log2n >= 9 ? 2 : 4);
}
__host__ __device__ constexpr int fx_minb(int log2n, bool inverse) { return (!inverse && log2n == 9) ? 5 : 3; }
#define FX_LINE(n_) ((n_) + ((n_) >> 3))
// shared memory of one line pair: two padded lines + 2 elements of skew, so that the buffers of consecutive
// pairs start 8 banks apart and the (un)tangling accesses, which touch the same l in every pair, do not collide
#define FX_PAIR(n_) (2 * FX_LINE(n_) + 2)
// k_fftx_inv: L2 prefetch distance in CTAs = one residency (3 CTAs on each of 148 SMs): the CTA that takes this
// one's place finds its scattered 128-byte spectrum pieces in L2.  (The forward kernel reads whole contiguous lines
// and gained nothing from the same prefetch at nx = 512 and lost at nx = 1024; it does not prefetch.)
#define FX_AHEAD 444

__host__ __device__ inline size_t fz_fftx_smem(int log2n, bool inverse) { return (size_t)fx_pairs(log2n, inverse) * FX_PAIR(1 << log2n) * 16; }

template <bool DIV, int LOG2N>
__global__ void __launch_bounds__(fx_pairs(LOG2N, false) * ((1 << LOG2N) / 8), fx_minb(LOG2N, false))
k_fftx_fwd(FzP P, const double *__restrict__ src, const double *__restrict__ us,
           const double *__restrict__ vs, const double *__restrict__ ws, double coef,
           double2 *__restrict__ spec, const double2 *__restrict__ tw)
{
    extern __shared__ __align__(16) double2 smx[];
    constexpr int n = 1 << LOG2N, T8 = n / 8, LN = FX_LINE(n), PS = FX_PAIR(n), FX_PAIRS = fx_pairs(LOG2N, false);
    const int jt = threadIdx.x, g = threadIdx.y;
    double2 *A = smx + g * PS, *B = A + LN;
    FzLineFFT<LOG2N, -1, false> fft;
    fft.init(tw, jt);
    const long long L0 = (long long)blockIdx.x * (2 * FX_PAIRS);   // first line of the CTA; 2*FX_PAIRS | ny
    const int k = (int)(L0 / P.ny), j0 = (int)(L0 - (long long)k * P.ny);
    const int ja = j0 + 2 * g;                                      // lines ja (real part), ja+1 (imaginary part)
    const long long ra = ((long long)k * P.ny + ja) * n, rb = ra + n;
    double2 v[8];
    if (DIV) {
        const long long rm = ((long long)k * P.ny + fz_im(ja, P.ny)) * n;   // row ja-1 (periodic)
        const bool wall_lo = P.z_wall && k == 0;
        const long long dzl = (k == 0) ? (long long)(P.nz - 1) * P.sxy : -P.sxy;   // plane k-1 (periodic wrap)
        const double izf = P.idzf[k];
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const int i = jt + q * T8, im = fz_im(i, n);
            const double va = vs[ra + i];
            const double wla = wall_lo ? 0.0 : ws[ra + i + dzl], wlb = wall_lo ? 0.0 : ws[rb + i + dzl];
            v[q].x = coef * ((us[ra + i] - us[ra + im]) * P.idx + (va - vs[rm + i]) * P.idy + (ws[ra + i] - wla) * izf);
            v[q].y = coef * ((us[rb + i] - us[rb + im]) * P.idx + (vs[rb + i] - va) * P.idy + (ws[rb + i] - wlb) * izf);
        }
    } else {
#pragma unroll
        for (int q = 0; q < 8; ++q) { const int i = jt + q * T8; v[q] = make_double2(src[ra + i], src[rb + i]); }
    }
    const double2 *res = fft.regs_to_smem(jt, A, B, v);   // same buffer (A or B) in every group
    const int roff = (int)(res - A);
    // untangle and store: consecutive threads -> consecutive j (runs of 2*FX_PAIRS*16 bytes)
    const int nth = T8 * FX_PAIRS, t = g * T8 + jt;
    const int nxh = P.nxh;
    double2 *out = spec + (long long)k * nxh * P.ny + j0;
    for (int e = t; e < 2 * FX_PAIRS * nxh; e += nth) {
        const int l = e / (2 * FX_PAIRS), ln = e - l * (2 * FX_PAIRS);
        const double2 *buf = smx + (ln >> 1) * PS + roff;
        const double2 z1 = buf[FZL_PADI(l)];
        const int l2 = (n - l) & (n - 1);
        const double2 z2 = buf[FZL_PADI(l2)];
        double2 o;
        if (ln & 1) o = make_double2(0.5 * (z1.y + z2.y), -0.5 * (z1.x - z2.x));  // B_l
        else o = make_double2(0.5 * (z1.x + z2.x), 0.5 * (z1.y - z2.y));          // A_l
        out[(long long)l * P.ny + ln] = o;
    }
}

// ---------------------------------------------------------------- FFT along x, backward (c2r)
// out = Re / Im of the inverse transform * scale - gauge shift (N17: scal[2] + scal[6] = mean of mode (0,0),
// written by k_spec_bwd)
template <int LOG2N>
__global__ void __launch_bounds__(fx_pairs(LOG2N, true) * ((1 << LOG2N) / 8), fx_minb(LOG2N, true))
k_fftx_inv(FzP P, const double2 *__restrict__ spec, double *__restrict__ dst, double scale,
           const double2 *__restrict__ tw, const double *__restrict__ scal)
{
    extern __shared__ __align__(16) double2 smx[];
    constexpr int n = 1 << LOG2N, T8 = n / 8, LN = FX_LINE(n), PS = FX_PAIR(n), FX_PAIRS = fx_pairs(LOG2N, true);
    const int jt = threadIdx.x, g = threadIdx.y;
    double2 *A = smx + g * PS, *B = A + LN;
    FzLineFFT<LOG2N, +1, false> fft;
    fft.init(tw, jt);
    const long long L0 = (long long)blockIdx.x * (2 * FX_PAIRS);
    const int k = (int)(L0 / P.ny), j0 = (int)(L0 - (long long)k * P.ny);
    const double shift = (scal[2] + scal[6]) * scale;
    const int nth = T8 * FX_PAIRS, t = g * T8 + jt;
    const int nxh = P.nxh;
    const double2 *in = spec + (long long)k * nxh * P.ny + j0;
    {   // L2 prefetch of the spectrum rows of the CTA FX_AHEAD launches later (2*FX_PAIRS*16 bytes per l)
        const long long Lp = L0 + (long long)FX_AHEAD * (2 * FX_PAIRS);
        if (Lp < (long long)P.ny * P.nz) {
            const int kp = (int)(Lp / P.ny), jp = (int)(Lp - (long long)kp * P.ny);
            const double2 *inp = spec + (long long)kp * nxh * P.ny + jp;
            for (int l = t; l < nxh; l += nth) fz_prefetch_l2(inp + (long long)l * P.ny);
        }
    }
    // tangle: consecutive threads -> consecutive pairs (32-byte pieces, runs of 2*FX_PAIRS*16 bytes per l)
    for (int e = t; e < FX_PAIRS * nxh; e += nth) {
        const int l = e / FX_PAIRS, pr = e - l * FX_PAIRS;
        const double2 a = in[(long long)l * P.ny + 2 * pr], b = in[(long long)l * P.ny + 2 * pr + 1];
        double2 *buf = smx + pr * PS;
        if (l == 0 || l == n / 2) {
            buf[FZL_PADI(l)] = make_double2(a.x, b.x);
        } else {
            buf[FZL_PADI(l)] = make_double2(a.x - b.y, a.y + b.x);
            buf[FZL_PADI(n - l)] = make_double2(a.x + b.y, b.x - a.y);
        }
    }
    __syncthreads();
    double2 v[8];
    fft.smem_to_regs(jt, A, B, v);
    const int ja = j0 + 2 * g;
    const long long ra = ((long long)k * P.ny + ja) * n, rb = ra + n;
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const int i = jt + q * T8;
        dst[ra + i] = v[q].x * scale - shift;
        dst[rb + i] = v[q].y * scale - shift;
    }
}

// ---------------------------------------------------------------- host-side dispatch over log2(nx)
// which < 0: opt the three kernels of this length in to their dynamic shared memory (once, at fizzy_create)
template <int LOG2N>
cudaError_t fz_fftx_launch_one(int which /*0 fwd DIV, 1 fwd plain, 2 inv*/, const FzP &P, const double *src,
                               const double *us, const double *vs, const double *ws, double coef, double2 *spec,
                               double *dst, const double2 *tw, const double *scal, cudaStream_t st)
{
    if (which < 0) {
        const int sf = (int)fz_fftx_smem(LOG2N, false), si = (int)fz_fftx_smem(LOG2N, true);
        cudaError_t e = cudaFuncSetAttribute(k_fftx_fwd<true, LOG2N>, cudaFuncAttributeMaxDynamicSharedMemorySize, sf);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_fftx_fwd<false, LOG2N>, cudaFuncAttributeMaxDynamicSharedMemorySize, sf);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_fftx_inv<LOG2N>, cudaFuncAttributeMaxDynamicSharedMemorySize, si);
        return e;
    }
    const int n = 1 << LOG2N;
    const int np = fx_pairs(LOG2N, which == 2);
    const size_t smem = fz_fftx_smem(LOG2N, which == 2);
    const dim3 block(n / 8, np);
    const unsigned grid = (unsigned)(((long long)P.ny * P.nz) / (2 * np));
    if (which == 0) k_fftx_fwd<true, LOG2N><<<grid, block, smem, st>>>(P, nullptr, us, vs, ws, coef, spec, tw);
    else if (which == 1) k_fftx_fwd<false, LOG2N><<<grid, block, smem, st>>>(P, src, nullptr, nullptr, nullptr, 1.0, spec, tw);
    else k_fftx_inv<LOG2N><<<grid, block, smem, st>>>(P, spec, dst, coef, tw, scal);
    return cudaSuccess;
}

inline cudaError_t fz_fftx_launch(int which, int log2n, const FzP &P, const double *src, const double *us,
                                  const double *vs, const double *ws, double coef, double2 *spec, double *dst,
                                  const double2 *tw, const double *scal, cudaStream_t st)
{
    switch (log2n) {
#define FZ_CASE(L_) case L_: return fz_fftx_launch_one<L_>(which, P, src, us, vs, ws, coef, spec, dst, tw, scal, st);
        FZ_CASE(3) FZ_CASE(4) FZ_CASE(5) FZ_CASE(6) FZ_CASE(7) FZ_CASE(8) FZ_CASE(9) FZ_CASE(10)
#undef FZ_CASE
    }
    return cudaErrorInvalidValue;
}
