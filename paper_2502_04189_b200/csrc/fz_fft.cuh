// fz_fft.cuh -- S4: Poisson right-hand side, batched shared-memory FFTs along x (real<->complex)
// and y (complex), BASELINE.json:5(iv) / kernel group (c).  PAPER.md:36 ("fast direct FFT solver").
//
// A CTA transforms S lines at once.  The lines sit side by side in shared memory as
// sm[element * (S+1) + slot] (double2), so that the 8 lanes of a quarter-warp, which hold the 8
// slots of one element, always touch 128 contiguous bytes: every butterfly load/store is
// bank-conflict free without index swizzles, and the +1 pad makes the transposing loads/stores
// of the x-kernels conflict free as well.  Each FFT of length n is done by n/8 threads with the
// Stockham autosort scheme: radix-8 passes, then one radix-4 or radix-2 pass if log2(n) % 3 != 0.
// Twiddles W_n^q = exp(-2 pi i q/n) come from a table computed on the host in fp64.
#pragma once
#include "fz_common.cuh"

// in-register DFT of R points, SGN = -1 forward, +1 backward
template <int SGN>
__device__ __forceinline__ double2 fz_mul_i(double2 a)  // a * (SGN * i)
{
    return SGN > 0 ? make_double2(-a.y, a.x) : make_double2(a.y, -a.x);
}
__device__ __forceinline__ double2 operator+(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 operator-(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }

template <int SGN>
__device__ __forceinline__ void fz_dft2(double2 &a, double2 &b)
{
    const double2 t = a - b;
    a = a + b;
    b = t;
}
template <int SGN>
__device__ __forceinline__ void fz_dft4(double2 &v0, double2 &v1, double2 &v2, double2 &v3)
{
    const double2 t0 = v0 + v2, t1 = v0 - v2, t2 = v1 + v3, t3 = fz_mul_i<SGN>(v1 - v3);
    v0 = t0 + t2;
    v1 = t1 + t3;
    v2 = t0 - t2;
    v3 = t1 - t3;
}
template <int SGN>
__device__ __forceinline__ void fz_dft8(double2 (&v)[8])
{
    // even / odd halves, then combine with W8^k = exp(SGN 2 pi i k/8)
    fz_dft4<SGN>(v[0], v[2], v[4], v[6]);
    fz_dft4<SGN>(v[1], v[3], v[5], v[7]);
    const double h = 0.70710678118654752440;
    const double2 o0 = v[1];
    const double2 o1 = make_double2(h * (v[3].x - SGN * v[3].y), h * (v[3].y + SGN * v[3].x));   // *(1+SGN i)/sqrt2
    const double2 o2 = fz_mul_i<SGN>(v[5]);
    const double2 o3 = make_double2(h * (-v[7].x - SGN * v[7].y), h * (-v[7].y + SGN * v[7].x)); // *(-1+SGN i)/sqrt2
    const double2 e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6];
    v[0] = e0 + o0; v[4] = e0 - o0;
    v[1] = e1 + o1; v[5] = e1 - o1;
    v[2] = e2 + o2; v[6] = e2 - o2;
    v[3] = e3 + o3; v[7] = e3 - o3;
}

// One Stockham pass of radix R over the S side-by-side FFTs held in sm (in place: all loads,
// barrier, all stores, barrier).  jt in [0, n/8) is this thread's index within its FFT.
// PAD = true: a single line per CTA stored as sm[i + (i >> 3)] (one 16-byte pad per 8 elements),
// which makes every butterfly load/store of the radix-8 passes conflict free without side-by-side
// lines (slot and LP are ignored).
template <int R, int SGN, bool PAD = false>
__device__ __forceinline__ void fz_fft_pass(double2 *sm, const double2 *__restrict__ tw, int n, int Ns,
                                            int jt, int slot, int LP)
{
#define FZ_SMI(i_) (PAD ? ((i_) + ((i_) >> 3)) : ((i_) * LP + slot))
    constexpr int NB = 8 / R;  // butterflies per thread
    const int T = n / R;       // butterflies per FFT
    const int T8 = n >> 3;
    double2 v[NB][R];
#pragma unroll
    for (int b = 0; b < NB; ++b) {
        const int j = jt + b * T8;
#pragma unroll
        for (int r = 0; r < R; ++r) v[b][r] = sm[FZ_SMI(j + r * T)];
    }
    __syncthreads();
#pragma unroll
    for (int b = 0; b < NB; ++b) {
        const int j = jt + b * T8;
        const int kk = j & (Ns - 1);
        if (Ns > 1) {
            const int M = n / (Ns * R);
#pragma unroll
            for (int r = 1; r < R; ++r) {
                double2 t = tw[r * kk * M];
                if (SGN > 0) t.y = -t.y;
                v[b][r] = fz_cmul(v[b][r], t);
            }
        }
        if constexpr (R == 8) {
            fz_dft8<SGN>(v[b]);
        } else if constexpr (R == 4) {
            fz_dft4<SGN>(v[b][0], v[b][1], v[b][2], v[b][3]);
        } else {
            fz_dft2<SGN>(v[b][0], v[b][1]);
        }
        const int base = (j - kk) * R + kk;
#pragma unroll
        for (int r = 0; r < R; ++r) sm[FZ_SMI(base + r * Ns)] = v[b][r];
    }
    __syncthreads();
#undef FZ_SMI
}

// Full FFT of the S lines in sm.  Data must be in sm and visible (barrier done by the caller).
template <int SGN, bool PAD = false>
__device__ __forceinline__ void fz_fft_tile(double2 *sm, const double2 *__restrict__ tw, int n, int log2n,
                                            int jt, int slot, int LP)
{
    int Ns = 1;
    const int n8 = log2n / 3;
    for (int q = 0; q < n8; ++q) {
        fz_fft_pass<8, SGN, PAD>(sm, tw, n, Ns, jt, slot, LP);
        Ns <<= 3;
    }
    const int rem = log2n - 3 * n8;
    if (rem == 2) fz_fft_pass<4, SGN, PAD>(sm, tw, n, Ns, jt, slot, LP);
    else if (rem == 1) fz_fft_pass<2, SGN, PAD>(sm, tw, n, Ns, jt, slot, LP);
}

// ---------------------------------------------------------------- FFT along x, forward
// Lines are (j,k) pairs flattened as L = j + ny*k; a CTA takes 2S consecutive lines, two real
// lines per complex FFT (a + i b), and writes nxh = nx/2+1 modes per line:
//   spec[(k*nxh + l)*ny + j]   (y lines contiguous, see fz_spectral.cuh).
//   A_l = (Z_l + conj Z_{n-l})/2,  B_l = (Z_l - conj Z_{n-l})/(2i).
// DIV = true: the real input is the Poisson right-hand side assembled on the fly,
//   b = coef * D(u**)  (BASELINE.json:5(iv) with the p_hat term folded into u**, D2);
// DIV = false: the real input is read from `src` (fizzy_poisson_solve).
template <bool DIV>
__global__ void __launch_bounds__(512, 2) k_fftx_fwd(FzP P, const double *__restrict__ src, const double *__restrict__ us,
                           const double *__restrict__ vs, const double *__restrict__ ws, double coef,
                           double2 *__restrict__ spec, const double2 *__restrict__ tw, int log2n, int S)
{
    extern __shared__ double2 sm[];
    const int n = P.nx, LP = S + 1;
    const int nth = blockDim.x;  // = S * n / 8
    const long long nlines = (long long)P.ny * P.nz;
    const long long L0 = (long long)blockIdx.x * 2 * S;
    // load: thread -> x index, loop over lines
    for (int e = threadIdx.x; e < 2 * S * n; e += nth) {
        const int ln = e >> log2n, i = e & (n - 1);
        const long long L = L0 + ln;
        double val = 0.0;
        if (L < nlines) {
            const long long c = L * n + i;
            if (DIV) {
                const int k = (int)(L / P.ny), j = (int)(L - (long long)k * P.ny);
                const long long xm = L * n + fz_im(i, n);
                const long long ym = ((long long)k * P.ny + fz_im(j, P.ny)) * n + i;
                double wlo;
                if (P.z_wall) wlo = (k == 0) ? 0.0 : ws[c - P.sxy];
                else wlo = ws[(k == 0) ? c + (long long)(P.nz - 1) * P.sxy : c - P.sxy];
                val = coef * ((us[c] - us[xm]) * P.idx + (vs[c] - vs[ym]) * P.idy + (ws[c] - wlo) * P.idzf[k]);
            } else {
                val = src[c];
            }
        }
        double *d = reinterpret_cast<double *>(&sm[i * LP + (ln >> 1)]);
        d[ln & 1] = val;
    }
    __syncthreads();
    const int slot = threadIdx.x % S, jt = threadIdx.x / S;
    fz_fft_tile<-1>(sm, tw, n, log2n, jt, slot, LP);
    // untangle and store: spec[(k*nxh + l)*ny + j], j fastest -> 2S consecutive lines give 32*S-byte runs
    const int nxh = P.nxh, lgy = __ffs(P.ny) - 1;
    for (int e = threadIdx.x; e < 2 * S * nxh; e += nth) {
        const int l = e / (2 * S), ln = e - l * (2 * S);
        const long long L = L0 + ln;
        if (L >= nlines) continue;
        const int sl = ln >> 1;
        const double2 z1 = sm[l * LP + sl];
        const double2 z2 = sm[((n - l) & (n - 1)) * LP + sl];
        double2 o;
        if (ln & 1) o = make_double2(0.5 * (z1.y + z2.y), -0.5 * (z1.x - z2.x));  // B_l
        else o = make_double2(0.5 * (z1.x + z2.x), 0.5 * (z1.y - z2.y));          // A_l
        const long long k = L >> lgy, j = L & (P.ny - 1);
        spec[(k * nxh + l) * P.ny + j] = o;
    }
}

// ---------------------------------------------------------------- FFT along x, backward (c2r)
// Z_l = A_l + i B_l, Z_{n-l} = conj(A_l) + i conj(B_l); out = Re/Im of the inverse transform * scale - gauge shift
__global__ void __launch_bounds__(512, 2) k_fftx_inv(FzP P, const double2 *__restrict__ spec, double *__restrict__ dst, double scale,
                           const double2 *__restrict__ tw, int log2n, int S, const double *__restrict__ scal)
{
    extern __shared__ double2 sm[];
    const int n = P.nx, LP = S + 1, nxh = P.nxh;
    const int nth = blockDim.x;
    const long long nlines = (long long)P.ny * P.nz;
    const long long L0 = (long long)blockIdx.x * 2 * S;
    const int lgy = __ffs(P.ny) - 1;
    const double shift = scal[2] * scale;   // gauge (N17): mean of mode (0,0), from k_spec_bwd
    // pairs of lines: slot sl holds lines 2 sl (A) and 2 sl + 1 (B)
    for (int e = threadIdx.x; e < S * nxh; e += nth) {
        const int l = e / S, sl = e - l * S;
        const long long LA = L0 + 2 * sl, LB = LA + 1;
        double2 a = make_double2(0, 0), b = make_double2(0, 0);
        if (LA < nlines) { const long long k = LA >> lgy, j = LA & (P.ny - 1); a = spec[(k * nxh + l) * P.ny + j]; }
        if (LB < nlines) { const long long k = LB >> lgy, j = LB & (P.ny - 1); b = spec[(k * nxh + l) * P.ny + j]; }
        if (l == 0 || l == n / 2) {
            sm[l * LP + sl] = make_double2(a.x, b.x);
        } else {
            sm[l * LP + sl] = make_double2(a.x - b.y, a.y + b.x);
            sm[(n - l) * LP + sl] = make_double2(a.x + b.y, b.x - a.y);
        }
    }
    __syncthreads();
    const int slot = threadIdx.x % S, jt = threadIdx.x / S;
    fz_fft_tile<+1>(sm, tw, n, log2n, jt, slot, LP);
    for (int e = threadIdx.x; e < 2 * S * n; e += nth) {
        const int ln = e >> log2n, i = e & (n - 1);
        const long long L = L0 + ln;
        if (L >= nlines) continue;
        const double *d = reinterpret_cast<const double *>(&sm[i * LP + (ln >> 1)]);
        dst[L * n + i] = d[ln & 1] * scale - shift;
    }
}

