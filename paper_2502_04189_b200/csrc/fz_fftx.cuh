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
#include <cuda.h>
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
// written by k_spec_bwd).
// The CTA's input is, for every x-mode l, a run of 2*FX_PAIRS consecutive j of the spectrum: nxh pieces of 128 (64)
// bytes, 16*ny bytes apart.  Read by the threads themselves these scattered pieces kept the LSU data pipe 87 % busy
// with DRAM at 53 % (ncu r2a).  They are one BOX of a rank-3 tensor (2 ny doubles | nxh | nz), so ONE thread fetches
// them with TMA (cp.async.bulk.tensor, boxes of at most 256 rows, 128-byte swizzle, completion on an mbarrier) into
// a staging area [l][2*FX_PAIRS]; every thread then takes the eight inputs of its first radix-8 pass straight from
// there, tangling on the fly (rows l <= n/2 directly, the others from the mirror row n-l) -- no tangle pass through
// shared memory, no barrier before the transform.  The staging area aliases the second FFT buffer, which the transform
// writes only after the barrier that follows its first pass.
struct FzFxInvGeom {   // staging geometry, the same on the host (tensor map) and in the kernel
    int pairs, rowb, nbox, brows, swz;   // bytes per staged row, boxes, rows per box, swizzle mask (16-byte chunks)
};
__host__ __device__ constexpr FzFxInvGeom fx_inv_geom(int log2n)
{
    const int pairs = fx_pairs(log2n, true), nxh = (1 << log2n) / 2 + 1;
    const int rowb = pairs * 32, nbox = (nxh + 255) / 256;
    const int brows = ((nxh + nbox - 1) / nbox + 7) / 8 * 8;   // a multiple of 8 rows: every box starts on a swizzle period
    return FzFxInvGeom{pairs, rowb, nbox, brows, rowb / 16 - 1};
}
__host__ __device__ constexpr size_t fx_inv_smem(int log2n)
{
    const FzFxInvGeom G = fx_inv_geom(log2n);
    const size_t buf = (size_t)G.pairs * FX_LINE(1 << log2n) * 16, stage = (size_t)G.nbox * G.brows * G.rowb;
    return ((buf > stage ? buf : stage) + 127) / 128 * 128 + buf;   // [Y | staging][X]
}

template <int LOG2N>
__global__ void __launch_bounds__(fx_pairs(LOG2N, true) * ((1 << LOG2N) / 8), fx_minb(LOG2N, true))
k_fftx_inv(FzP P, const __grid_constant__ CUtensorMap tm_spec, double *__restrict__ dst, double scale,
           const double2 *__restrict__ tw, const double *__restrict__ scal)
{
    extern __shared__ __align__(1024) unsigned char smb[];
    __shared__ __align__(8) unsigned long long bar;
    constexpr int n = 1 << LOG2N, T8 = n / 8, LN = FX_LINE(n);
    constexpr FzFxInvGeom G = fx_inv_geom(LOG2N);
    constexpr size_t YB = fx_inv_smem(LOG2N) - (size_t)G.pairs * LN * 16;
    const int jt = threadIdx.x, g = threadIdx.y, t = g * T8 + jt;
    double2 *Y = reinterpret_cast<double2 *>(smb) + g * LN, *X = reinterpret_cast<double2 *>(smb + YB) + g * LN;
    const long long L0 = (long long)blockIdx.x * (2 * G.pairs);
    const int k = (int)(L0 / P.ny), j0 = (int)(L0 - (long long)k * P.ny);
    if (t == 0) fz_mbar_init(&bar, 1);
    __syncthreads();
    if (t == 0) {
        fz_mbar_expect_tx(&bar, (unsigned)(G.nbox * G.brows * G.rowb));
#pragma unroll
        for (int b = 0; b < G.nbox; ++b)   // rows past nxh are outside the tensor: filled with zeros, never read
            fz_tma_load_3d(smb + (size_t)b * G.brows * G.rowb, &tm_spec, 2 * j0, b * G.brows, k, &bar);
    }
    FzLineFFT<LOG2N, +1, false> fft;
    fft.init(tw, jt);
    const double shift = (scal[2] + scal[6]) * scale;
    fz_mbar_wait(&bar, 0);
    // inputs of the first pass: Z_l = A_l + i B_l (l <= n/2), Z_l = conj(A_{n-l}) + i conj(B_{n-l}) (l > n/2); the
    // pair's A_l, B_l are the 16-byte chunks 2g, 2g+1 of staged row l (chunk index XOR row: the TMA swizzle)
    double2 v[8];
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const int l = jt + r * T8;
        const bool mir = l > n / 2;
        const int row = mir ? n - l : l;
        unsigned off = (unsigned)row * G.rowb + 32u * g;
        off ^= ((off >> 7) & G.swz) << 4;
        const double2 a = *reinterpret_cast<const double2 *>(smb + off), b = *reinterpret_cast<const double2 *>(smb + (off ^ 16u));
        if (mir) v[r] = make_double2(a.x + b.y, b.x - a.y);
        else if (l == 0 || l == n / 2) v[r] = make_double2(a.x, b.x);
        else v[r] = make_double2(a.x - b.y, a.y + b.x);
    }
    fft.regs_to_regs(jt, X, Y, v);
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
                               double *dst, const double2 *tw, const double *scal, const CUtensorMap *tm_spec,
                               cudaStream_t st)
{
    if (which < 0) {
        const int sf = (int)fz_fftx_smem(LOG2N, false), si = (int)fx_inv_smem(LOG2N);
        cudaError_t e = cudaFuncSetAttribute(k_fftx_fwd<true, LOG2N>, cudaFuncAttributeMaxDynamicSharedMemorySize, sf);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_fftx_fwd<false, LOG2N>, cudaFuncAttributeMaxDynamicSharedMemorySize, sf);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_fftx_inv<LOG2N>, cudaFuncAttributeMaxDynamicSharedMemorySize, si);
        return e;
    }
    const int n = 1 << LOG2N;
    const int np = fx_pairs(LOG2N, which == 2);
    const size_t smem = which == 2 ? fx_inv_smem(LOG2N) : fz_fftx_smem(LOG2N, false);
    const dim3 block(n / 8, np);
    const unsigned grid = (unsigned)(((long long)P.ny * P.nz) / (2 * np));
    if (which == 0) k_fftx_fwd<true, LOG2N><<<grid, block, smem, st>>>(P, nullptr, us, vs, ws, coef, spec, tw);
    else if (which == 1) k_fftx_fwd<false, LOG2N><<<grid, block, smem, st>>>(P, src, nullptr, nullptr, nullptr, 1.0, spec, tw);
    else k_fftx_inv<LOG2N><<<grid, block, smem, st>>>(P, *tm_spec, dst, coef, tw, scal);
    return cudaSuccess;
}

inline cudaError_t fz_fftx_launch(int which, int log2n, const FzP &P, const double *src, const double *us,
                                  const double *vs, const double *ws, double coef, double2 *spec, double *dst,
                                  const double2 *tw, const double *scal, const CUtensorMap *tm_spec, cudaStream_t st)
{
    switch (log2n) {
#define FZ_CASE(L_) case L_: return fz_fftx_launch_one<L_>(which, P, src, us, vs, ws, coef, spec, dst, tw, scal, tm_spec, st);
        FZ_CASE(3) FZ_CASE(4) FZ_CASE(5) FZ_CASE(6) FZ_CASE(7) FZ_CASE(8) FZ_CASE(9) FZ_CASE(10)
#undef FZ_CASE
    }
    return cudaErrorInvalidValue;
}
