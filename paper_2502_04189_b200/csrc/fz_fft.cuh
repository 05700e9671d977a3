// fz_fft.cuh -- in-register butterflies shared by the FFT kernels (kernel group (c) of BASELINE.json:5).
// SGN = -1 forward (exp(-2 pi i jk/n)), +1 backward (unscaled).
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

