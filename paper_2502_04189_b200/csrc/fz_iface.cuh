// fz_iface.cuh -- kernel group (a): interface quantities of a phase field in ONE marching sweep.
// Inputs psi = eps ln q (written pointwise by the kernel that produced phi) and phi; outputs
// kappa = -D(nf), divRn = D(R/Gamma) and, when rho1 != rho2, Rn on the three "+" faces
// (BASELINE.json:5(i),(iii); readings N3-N5).  The cell-centred normal nhat = G/max(|G|,1e-30) and
// r = sqrt(q) are computed ONCE per cell on chip and shared through shared memory -- they never go
// to HBM (r is a pointwise function of phi: one reciprocal and one rsqrt per staged cell).
//
// A CTA owns an x-y tile of ITX x ITY cells and marches over a chunk of z planes.  Shared memory
// holds rings of IRING planes of psi and phi (tile + halo 2), of three planes of r (tile + halo 1)
// and of two planes of the HALF normals 0.5 nhat_x, 0.5 nhat_y (tile + halo 1); nhat_z of the
// thread's own column and the z face below it live in registers.  Planes arrive by 16-byte cp.async
// (LDGSTS) issued IDEPTH = IRING-3 planes ahead of their first use, so no register is tied up by a
// load in flight and HBM latency under load (several microseconds) hides behind IDEPTH planes of
// compute.  Step s (kk = k0-2+s): (1) wait for plane kk+1, (2) barrier, (3) issue the copies of
// plane kk+1+IDEPTH into the slot plane kk-2 just left, (4) r of plane kk+1, (5) half normals of
// plane kk for the tile and its halo-1 cross, (6) plane k = kk-1 is finished and written.  One
// barrier per plane.  The plane loop is unrolled by IRING (a multiple of 2 and 3) so that every ring
// slot is a COMPILE-TIME constant: all shared-memory accesses are [thread base + immediate].
//   psi, phi:     planes kk-1, kk, kk+1 in slots (s-1, s, s+1) mod IRING
//   r:            plane kk+1 is written into slot (s+1) mod 3; planes kk-1, kk are read from (s-1, s) mod 3
//   half normals: plane kk is written into slot s mod 2, plane k = kk-1 is read from slot (s-1) mod 2
#pragma once
#include <type_traits>
#include "fz_common.cuh"

#define ITX 32
#define ITY 16
#define IPW (ITX + 4)
#define IPH (ITY + 4)
#define IPS (IPW * IPH)
#define INW (ITX + 2)
#define INH (ITY + 2)
#define INS (INW * INH)
#ifndef IRING
#define IRING 6
#endif
#define IDEPTH (IRING - 3)
#define ICHUNKS (IPS / 2)   // 16-byte chunks of one staged plane
#define IFACE_SMEM ((2 * IRING * IPS + 7 * INS) * sizeof(double))   // psi, phi rings + 3 planes of r + 2 x (nhx, nhy)
static_assert(IRING % 6 == 0, "the plane loop is unrolled by IRING: ring slots of depth 2 and 3 must be compile-time too");

// 1/(1+s)^2 * s with one reciprocal: sharpening coefficient 1/4 (1 - tanh^2((psi_a+psi_b)/(4 eps)))
// = s/(1+s)^2, s = r_a r_b (D1)
__device__ __forceinline__ double fz_sharp2(double ra, double rb)
{
    const double s = ra * rb;
    const double t = fz_rcp(1.0 + s);   // 1 + s in [1, 1e100]
    return s * t * t;
}

// r = sqrt(q), q = a/b, a = phic + delta, b = 1 - phic + delta (N2), as a * rsqrt(a b): ONE rsqrt and no reciprocal.
// a b lies in [delta (1 + delta), (1/2 + delta)^2] with delta >= 1e-150 (fizzy_create): normal, so the branch-free
// helper applies
__device__ __forceinline__ double fz_sqrtq(double phi, double delta)
{
    const double ph = fz_clip01(phi);
    const double a = ph + delta, b = 1.0 - ph + delta;
    return a * fz_rsqrt(a * b);
}

template <bool STORE_R>
__global__ void __launch_bounds__(ITX * ITY, 2)
k_iface_march(FzP P, const double *__restrict__ psi, const double *__restrict__ phi,
               double *__restrict__ kappa, double *__restrict__ divrn,
               double *__restrict__ rnx, double *__restrict__ rny, double *__restrict__ rnz, int KC)
{
    extern __shared__ __align__(16) double smi[];
    const int tx = threadIdx.x, ty = threadIdx.y, t = ty * ITX + tx;
    const int i0 = blockIdx.x * ITX, j0 = blockIdx.y * ITY;
    const int k0 = blockIdx.z * KC, k1 = min(k0 + KC, P.nz);
    // per-thread base pointers: own cell in a psi / phi plane, own cell in an r / half-normal plane
    const double *PSIc = smi + (ty + 2) * IPW + tx + 2;
    const double *PHIc = PSIc + IRING * IPS;
    double *RRc = smi + 2 * IRING * IPS + (ty + 1) * INW + tx + 1;
    double *NHXc = RRc + 3 * INS, *NHYc = NHXc + INS;   // [slot 0: x, y][slot 1: x, y]
    // staging map (16-byte chunks of the tile + halo 2 rectangle)
    const bool loader = t < ICHUNKS;
    const int lrow = t / (IPW / 2), lcp = t - lrow * (IPW / 2);
    const unsigned ugoff = (unsigned)(((i0 - 2 + 2 * lcp + P.nx) & (P.nx - 1)) + P.nx * ((j0 - 2 + lrow + P.ny) & (P.ny - 1)));
    double *stg = smi + lrow * IPW + 2 * lcp;
    const int zlo = P.z_wall ? -1 : P.nz, zhi = P.z_wall ? 2 * P.nz - 1 : -P.nz, zsg = P.z_wall ? -1 : 1;
    const unsigned sxy = (unsigned)P.sxy;
    // plane kk of psi, phi -> ring slot `slot` (compile-time in the loop)
    auto issue = [&](int kk, int slot) {
        if (loader) {
            const int zs = kk < 0 ? zlo + zsg * kk : (kk >= P.nz ? zhi + zsg * kk : kk);
            const unsigned g = (unsigned)zs * sxy + ugoff;
            double *d = stg + slot * IPS;
            fz_cp_async16(d, psi + g);
            fz_cp_async16(d + IRING * IPS, phi + g);
        }
    };
    // halo-1 cross cell of the r / half-normal planes handled by this thread (threads 0 .. 95)
    int hr = 1, hc = 2;
    const bool has_h = t < 2 * (ITX + ITY);
    if (t < ITX) { hr = 1; hc = 2 + t; }
    else if (t < 2 * ITX) { hr = ITY + 2; hc = 2 + t - ITX; }
    else if (t < 2 * ITX + ITY) { hr = 2 + t - 2 * ITX; hc = 1; }
    else if (has_h) { hr = 2 + t - 2 * ITX - ITY; hc = ITX + 2; }
    const double *PSIh = smi + hr * IPW + hc, *PHIh = PSIh + IRING * IPS;
    double *RRh = smi + 2 * IRING * IPS + (hr - 1) * INW + hc - 1;
    double *NHXh = RRh + 3 * INS, *NHYh = NHXh + INS;
    const double hx = 0.5 * P.idx, hy = 0.5 * P.idy;
    const double ex = P.eps * P.idx, ey = P.eps * P.idy;
    const double delta = P.delta;
    // HALF normal 0.5 G / max(|G|, 1e-30) (N4) of the cell at q, psi planes at slots SM, S0, SP
    auto normal = [&](const double *q, int om, int o0, int op, double igz, double &nx_, double &ny_, double &nz_) {
        const double gx = (q[o0 + 1] - q[o0 - 1]) * hx;
        const double gy = (q[o0 + IPW] - q[o0 - IPW]) * hy;
        const double gz = (q[op] - q[om]) * igz;
        // max(|G|^2, 1e-60) for a non-negative, non-NaN |G|^2: ordered like its bit pattern (fmax costs ten instructions)
        double g2 = gx * gx + gy * gy + gz * gz;
        if (__double_as_longlong(g2) < __double_as_longlong(1e-60)) g2 = 1e-60;
        const double inv = 0.5 * fz_rsqrt(g2);
        nx_ = gx * inv; ny_ = gy * inv; nz_ = gz * inv;
    };

    // prologue: planes k0-2 .. k0-2+IDEPTH in IDEPTH groups (the first holds two planes)
    issue(k0 - 2, 0); issue(k0 - 1, 1);
    fz_cp_async_commit();
#pragma unroll
    for (int d = 2; d <= IDEPTH; ++d) { issue(k0 - 2 + d, d); fz_cp_async_commit(); }
    double nz0 = 0.0, nzp = 0.0, nfz_prev = 0.0, Rz_prev = 0.0;
    const unsigned gc = (unsigned)((i0 + tx) + P.nx * (j0 + ty));
    double igz_n = P.igz[k0 - 2], idzc_n = 0.0, idzf_n = 0.0;   // z metrics: loaded one step ahead (plane k0-3 is never used)
    // PH = 0, 1, 2: the first three steps of a chunk (r only | + half normals | + the z face below the first plane); PH = 3:
    // a full step.  A compile-time phase keeps the three prologue tests out of the steady-state steps.
    auto step = [&](auto Sc, auto Pc, int kk) {
        constexpr int S = decltype(Sc)::value, PH = decltype(Pc)::value;
        constexpr int om = ((S + IRING - 1) % IRING) * IPS, o0 = (S % IRING) * IPS, op = ((S + 1) % IRING) * IPS;
        constexpr int rm = ((S + 2) % 3) * INS, r0s = (S % 3) * INS, rp = ((S + 1) % 3) * INS;   // r planes kk-1, kk, kk+1
        constexpr int n0 = (S % 2) * 2 * INS, nm = ((S + 1) % 2) * 2 * INS;                       // half-normal planes kk, kk-1
        fz_cp_async_wait<IDEPTH - 1>();
        __syncthreads();
        if (kk + 1 + IDEPTH <= k1 + 1) issue(kk + 1 + IDEPTH, (S + IRING - 2) % IRING);
        fz_cp_async_commit();
        // r = sqrt(q) of plane kk+1: own cell and the halo cross
        RRc[rp] = fz_sqrtq(PHIc[op], delta);
        if (has_h) RRh[rp] = fz_sqrtq(PHIh[op], delta);
        const double igz = igz_n;
        igz_n = P.igz[kk + 1];
        const double idzc_k = idzc_n, idzf_k = idzf_n;   // metrics of plane k = kk-1, loaded one step ago
        idzc_n = P.idzc[kk]; idzf_n = P.idzf[kk];
        if (PH < 1) return;
        {   // half normals of plane kk: own cell, then the halo cross
            double ax, ay, az;
            normal(PSIc, om, o0, op, igz, ax, ay, az);
            NHXc[n0] = ax; NHYc[n0] = ay;
            nz0 = nzp; nzp = az;
            if (has_h) {
                normal(PSIh, om, o0, op, igz, ax, ay, az);
                NHXh[n0] = ax; NHYh[n0] = ay;
            }
        }
        const int k = kk - 1;
        if (PH < 2) return;
        const double f0 = PHIc[om], r0 = RRc[rm];
        // z face k+1/2; the face k-1/2 is carried in registers.  On a wall face both terms vanish by themselves, exactly:
        // the ghost planes hold the mirrored psi and phi (and igz is mirrored), so nhat_z of the ghost cell is bit for bit
        // minus that of the wall cell (nf_z = 0, N3/walls) and phi(ghost) - phi(wall cell) = 0 (R_z = 0)
        const double nfzp = nz0 + nzp;
        const double Rzp = P.eps * (PHIc[o0] - f0) * idzc_k - fz_sharp2(r0, RRc[r0s]) * nfzp;
        if (PH < 3) { nfz_prev = nfzp; Rz_prev = Rzp; return; }
        // half normals of plane k were written one step ago: visible after this step's barrier
        const double ax = NHXc[nm], ay = NHYc[nm];
        const double nfxp = ax + NHXc[nm + 1], nfxm = NHXc[nm - 1] + ax;
        const double nfyp = ay + NHYc[nm + INW], nfym = NHYc[nm - INW] + ay;
        const double Rxp = ex * (PHIc[om + 1] - f0) - fz_sharp2(r0, RRc[rm + 1]) * nfxp;
        const double Rxm = ex * (f0 - PHIc[om - 1]) - fz_sharp2(RRc[rm - 1], r0) * nfxm;
        const double Ryp = ey * (PHIc[om + IPW] - f0) - fz_sharp2(r0, RRc[rm + INW]) * nfyp;
        const double Rym = ey * (f0 - PHIc[om - IPW]) - fz_sharp2(RRc[rm - INW], r0) * nfym;
        const unsigned c = (unsigned)k * sxy + gc;
        kappa[c] = -((nfxp - nfxm) * P.idx + (nfyp - nfym) * P.idy + (nfzp - nfz_prev) * idzf_k);
        divrn[c] = (Rxp - Rxm) * P.idx + (Ryp - Rym) * P.idy + (Rzp - Rz_prev) * idzf_k;
        if (STORE_R) { rnx[c] = Rxp; rny[c] = Ryp; rnz[c] = Rzp; }
        nfz_prev = nfzp; Rz_prev = Rzp;
    };
    // steps kk = k0-2 .. k1 (plane k = kk-1 = k1-1 is the last one written); a chunk holds at least one plane, so the three
    // prologue steps always run
#define IC_(n_) std::integral_constant<int, n_>{}
    step(IC_(0), IC_(0), k0 - 2);
    step(IC_(1), IC_(1), k0 - 1);
    step(IC_(2), IC_(2), k0);
    for (int kk = k0 + 1; kk <= k1; kk += IRING) {
        step(IC_(3), IC_(3), kk);
        if (kk + 1 > k1) break;
        step(IC_(4), IC_(3), kk + 1);
        if (kk + 2 > k1) break;
        step(IC_(5), IC_(3), kk + 2);
        if (kk + 3 > k1) break;
        step(IC_(0), IC_(3), kk + 3);
        if (kk + 4 > k1) break;
        step(IC_(1), IC_(3), kk + 4);
        if (kk + 5 > k1) break;
        step(IC_(2), IC_(3), kk + 5);
    }
#undef IC_
    fz_cp_async_wait<0>();
}
