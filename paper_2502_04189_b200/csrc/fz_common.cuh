// fz_common.cuh -- kernel-side parameter block and small device helpers of libfizzy.
// Notation follows DESIGN.md "The method" (hc = centre spacing at a face, hf = cell height).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define FZ_H 2  // ghost entries on each side of the 1-D z metric tables

// Passed by value to every kernel (lives in constant bank 0).
struct FzP {
    int nx, ny, nz, nxh;       // nxh = nx/2 + 1 retained x-modes
    int z_wall, heat;
    int kzf;                   // z-faces that carry an unknown w: nz (periodic) or nz-1 (walls)
    long long N;               // nx*ny*nz
    long long sxy;             // nx*ny (plane stride)
    double dx, dy, idx, idy;   // spacings and reciprocals
    double lz;                 // channel height (Nusselt number)
    // 1-D z metric tables, device pointers already offset by FZ_H (index k = -2 .. nz+1)
    const double *dzf, *dzc, *idzf, *idzc, *igz;  // igz[k] = 1/(dzc[k] + dzc[k-1])
    double rho1, rho2, mu1, mu2, k1, k2, cp1, cp2;
    double sigma, eps, delta, gamma_rel, gamma_abs;
    double gx, gy, gz, rho_ref, beta, t_ref, fx, fy, fz, a_lin;
    double t_bot, t_top;
    double rho0, drho;         // min(rho1, rho2), rho1 - rho2
};

// clip(f, 0, 1) on the bit pattern: f < 0 (sign bit) -> 0, f >= 1 (high word >= that of 1.0) -> 1, else f.  Equal to
// fmin(fmax(f, 0), 1) for every non-NaN f, in two integer compares and three selects; fmin/fmax cost a DSETP, two
// selects, a NaN fix-up and several moves each (14 instructions per clip in k_iface_march, two of them on the fp64 pipe).
__device__ __forceinline__ double fz_clip01(double f)
{
    const int hi = __double2hiint(f), lo = __double2loint(f);
    const bool neg = hi < 0, big = hi >= 0x3ff00000;
    return __hiloint2double(neg ? 0 : (big ? 0x3ff00000 : hi), (neg || big) ? 0 : lo);
}
// 2 clip(f,0,1) - 1 = |f| - |f - 1| without a comparison (two DADD with operand modifiers instead of DSETP + selects
// + moves per fmin/fmax): exact outside [0,1], within one rounding of 1 (1.1e-16 ABSOLUTE) inside.  For the linear
// property maps q2 + (q1-q2) clip(phi) = (q2+q1)/2 + (q1-q2)/2 * fz_sclip(phi), where an absolute error of that size
// is the rounding error of the map itself; NOT for psi, which needs tiny phi to full relative accuracy.
__device__ __forceinline__ double fz_sclip(double f) { return fabs(f) - fabs(f - 1.0); }

// neighbour indices of a cell in the periodic directions
__device__ __forceinline__ int fz_ip(int i, int n) { return (i + 1 == n) ? 0 : i + 1; }
__device__ __forceinline__ int fz_im(int i, int n) { return (i == 0) ? n - 1 : i - 1; }

// z neighbours: plane index used for EVEN (mirrored) fields, and flags telling whether the
// neighbour is a wall ghost.  Periodic z wraps, never a ghost.
struct FzZ {
    int km, kp;        // plane indices to read for k-1 / k+1 (mirror at walls, wrap if periodic)
    bool gm, gp;       // true if k-1 / k+1 lies outside a wall
};
__device__ __forceinline__ FzZ fz_zn(const FzP &P, int k)
{
    FzZ z;
    if (P.z_wall) {
        z.gm = (k == 0);
        z.gp = (k == P.nz - 1);
        z.km = z.gm ? 0 : k - 1;
        z.kp = z.gp ? P.nz - 1 : k + 1;
    } else {
        z.gm = z.gp = false;
        z.km = (k == 0) ? P.nz - 1 : k - 1;
        z.kp = (k + 1 == P.nz) ? 0 : k + 1;
    }
    return z;
}

// order-preserving max of non-negative doubles through their bit pattern
__device__ __forceinline__ void fz_atomic_max_nonneg(double *addr, double v)
{
    atomicMax(reinterpret_cast<unsigned long long *>(addr),
              static_cast<unsigned long long>(__double_as_longlong(v)));
}

__device__ __forceinline__ double2 fz_cmul(double2 a, double2 b)
{
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

// Branch-free reciprocal and reciprocal square root for NORMAL, finite, positive arguments whose
// results are normal too (callers guarantee the range): hardware seed (MUFU.RCP64H / RSQ64H, relative
// error e0 ~ 2^-22) + ONE third-order step, x (1 + e + e^2) resp. y (1 + e/2 + 3 e^2/8), which leaves
// e0^3 ~ 2^-66 -> ~1 ulp in 3 (5) dependent fp64 operations instead of the 4 (7) of two Newton steps.
// The IEEE `/` and rsqrt() carry a slow-path branch per call that these stencils never need.
__device__ __forceinline__ double fz_rcp(double d)
{
    double x;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(x) : "d"(d));
    const double e = fma(-d, x, 1.0);
    return fma(x, fma(e, e, e), x);
}
__device__ __forceinline__ double fz_rsqrt(double a)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    const double e = fma(-a * y, y, 1.0);            // 1 - a y^2
    return fma(y, e * fma(0.375, e, 0.5), y);
}
// reciprocal of a normal, finite d of EITHER sign whose reciprocal is normal (tridiagonal pivots)
__device__ __forceinline__ double fz_rcp_signed(double d) { return fz_rcp(d); }   // the seed keeps the sign
// psi = eps ln q of a phase field value, q = (phic + delta)/(1 - phic + delta) (N2); 1 - phic + delta lies in
// [delta, 1 + delta], delta >= 1e-150: the branch-free reciprocal applies
__device__ __forceinline__ double fz_psi(const FzP &P, double f)
{
    const double ph = fz_clip01(f);
    return P.eps * log((ph + P.delta) * fz_rcp(1.0 - ph + P.delta));
}

// prefetch the 128-byte line at p into L2 (no register, no scoreboard)
__device__ __forceinline__ void fz_prefetch_l2(const void *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// 8- and 16-byte asynchronous global -> shared copies (LDGSTS) and their group fences
__device__ __forceinline__ void fz_cp_async16(void *smem_dst, const void *gsrc)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void fz_cp_async8(void *smem_dst, const void *gsrc)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void fz_cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void fz_cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// ---------------------------------------------------------------- TMA (cp.async.bulk.tensor) and mbarrier
// One elected thread initialises the barrier, announces the byte count and issues the tensor copies; every thread
// then waits for the phase to flip.  The tensor map is built on the host (fizzy_create, cuTensorMapEncodeTiled).
__device__ __forceinline__ unsigned fz_smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void fz_mbar_init(void *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(fz_smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void fz_mbar_expect_tx(void *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(fz_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void fz_mbar_wait(void *bar, unsigned phase)
{
    unsigned done;
    do {
        asm volatile("{\n\t.reg .pred P1;\n\tmbarrier.try_wait.parity.shared::cta.b64 P1, [%1], %2;\n\tselp.b32 %0, 1, 0, P1;\n\t}"
                     : "=r"(done) : "r"(fz_smem_u32(bar)), "r"(phase) : "memory");
    } while (!done);
}
// box of a rank-3 tensor map -> shared memory; coordinates innermost first
__device__ __forceinline__ void fz_tma_load_3d(void *smem_dst, const void *tmap, int c0, int c1, int c2, void *bar)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
                 ::"r"(fz_smem_u32(smem_dst)), "l"(tmap), "r"(fz_smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
