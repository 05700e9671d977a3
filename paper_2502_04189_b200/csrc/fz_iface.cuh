// fz_iface.cuh -- kernel group (a): interface quantities of a phase field in ONE marching sweep.
// Inputs psi = eps ln q, r = sqrt q (written pointwise by the kernel that produced phi) and phi;
// outputs kappa = -D(nf), divRn = D(R/Gamma) and, when rho1 != rho2, Rn on the three "+" faces
// (BASELINE.json:5(i),(iii); readings N3-N5).  The cell-centred normal nhat = G/max(|G|,1e-30)
// is computed ONCE per cell on chip and shared through shared memory -- it never goes to HBM.
//
// A CTA owns an x-y tile of ITX x ITY cells and marches over a chunk of z planes.  Shared memory
// holds rings of five planes of psi and four of r, phi (tile + halo 2) and a ring of three planes of
// nhat_x, nhat_y (tile + halo 1); nhat_z of the thread's own column lives in registers.
// Planes arrive by 16-byte cp.async (LDGSTS) two steps ahead of their use, so no register is
// tied up by a load in flight.  Step kk: (1) wait for psi(kk+1), r/phi(kk), (2) barrier, (3) issue
// the copies of psi(kk+3), r/phi(kk+2), (4) nhat(kk) for the tile and its halo-1 cross,
// (5) plane kk-1 is finished and written.  One barrier per plane.
#pragma once
#include "fz_common.cuh"

#define ITX 32
#define ITY 16
#define IPW (ITX + 4)
#define IPH (ITY + 4)
#define IPS (IPW * IPH)
#define INW (ITX + 2)
#define INH (ITY + 2)
#define INS (INW * INH)
#define IRING_PSI 5   // psi planes kk-1 .. kk+3
#define IRING_RF 4    // r, phi planes kk-1 .. kk+2
#define INRING 3
#define ICHUNKS (IPS / 2)   // 16-byte chunks of one staged plane
#define IFACE_SMEM (((IRING_PSI + 2 * IRING_RF) * IPS + 2 * INRING * INS) * sizeof(double))

// 1/(1+s)^2 * s with one reciprocal: sharpening coefficient 1/4 (1 - tanh^2((psi_a+psi_b)/(4 eps)))
// = s/(1+s)^2, s = r_a r_b (D1)
__device__ __forceinline__ double fz_sharp2(double ra, double rb)
{
    const double s = ra * rb;
    const double t = fz_rcp(1.0 + s);   // 1 + s in [1, 1e100]
    return s * t * t;
}

// source plane of z index kk in [-2, nz+1]: periodic wrap or wall mirror (even fields)
__device__ __forceinline__ int fz_zsrc(const FzP &P, int kk)
{
    if (P.z_wall) return kk < 0 ? -1 - kk : (kk >= P.nz ? 2 * P.nz - 1 - kk : kk);
    return kk < 0 ? kk + P.nz : (kk >= P.nz ? kk - P.nz : kk);
}

template <bool STORE_R>
__global__ void __launch_bounds__(ITX * ITY, 2)
k_iface_march(FzP P, const double *__restrict__ psi, const double *__restrict__ rr,
              const double *__restrict__ phi, double *__restrict__ kappa, double *__restrict__ divrn,
              double *__restrict__ rnx, double *__restrict__ rny, double *__restrict__ rnz, int KC)
{
    extern __shared__ __align__(16) double smi[];
    double *PSI = smi, *RR = smi + IRING_PSI * IPS, *PHI = RR + IRING_RF * IPS;
    double *NHX = PHI + IRING_RF * IPS, *NHY = NHX + INRING * INS;
    const int tx = threadIdx.x, ty = threadIdx.y, t = ty * ITX + tx;
    const int i0 = blockIdx.x * ITX, j0 = blockIdx.y * ITY;
    const int k0 = blockIdx.z * KC, k1 = min(k0 + KC, P.nz);
    // staging map: thread t < ICHUNKS copies the 16-byte chunk t of the (tile + halo 2) rectangle;
    // i0 - 2 and nx are even, so a chunk never straddles the periodic wrap
    const bool loader = t < ICHUNKS;
    const int lrow = t / (IPW / 2), lcp = t - lrow * (IPW / 2);
    const long long goff = ((i0 - 2 + 2 * lcp + P.nx) & (P.nx - 1)) +
                           (long long)P.nx * ((j0 - 2 + lrow + P.ny) & (P.ny - 1));
    const int soff = lrow * IPW + 2 * lcp;
    // planes are issued in increasing order, so the ring slots advance incrementally; offsets are
    // 32-bit (fizzy_create guarantees N < 2^31) and the ghost-plane map is branch-free
    const int zlo = P.z_wall ? -1 : P.nz, zhi = P.z_wall ? 2 * P.nz - 1 : -P.nz, zsg = P.z_wall ? -1 : 1;
    auto zsrc = [&](int kk) { return kk < 0 ? zlo + zsg * kk : (kk >= P.nz ? zhi + zsg * kk : kk); };
    const unsigned sxy = (unsigned)P.sxy, ugoff = (unsigned)goff;
    int sl_psi = (k0 - 2 + 2 * IRING_PSI) % IRING_PSI, sl_rf = (k0 - 2 + 2 * IRING_RF) & (IRING_RF - 1);
    auto issue_psi = [&](int kk) {   // plane kk of psi -> ring slot kk mod 5
        if (loader) fz_cp_async16(PSI + sl_psi * IPS + soff, psi + ((unsigned)zsrc(kk) * sxy + ugoff));
        sl_psi = (sl_psi + 1 == IRING_PSI) ? 0 : sl_psi + 1;
    };
    auto issue_rf = [&](int kk) {    // plane kk of r, phi -> ring slot kk mod 4
        if (loader) {
            const unsigned g = (unsigned)zsrc(kk) * sxy + ugoff;
            const int o = sl_rf * IPS + soff;
            fz_cp_async16(RR + o, rr + g);
            fz_cp_async16(PHI + o, phi + g);
        }
        sl_rf = (sl_rf + 1) & (IRING_RF - 1);
    };
    // halo-1 cross cell of the nhat plane handled by this thread (threads 0 .. 2(ITX+ITY)-1)
    int hr = 1, hc = 2;
    const bool has_h = t < 2 * (ITX + ITY);
    if (t < ITX) { hr = 1; hc = 2 + t; }
    else if (t < 2 * ITX) { hr = ITY + 2; hc = 2 + t - ITX; }
    else if (t < 2 * ITX + ITY) { hr = 2 + t - 2 * ITX; hc = 1; }
    else if (has_h) { hr = 2 + t - 2 * ITX - ITY; hc = ITX + 2; }
    const int pc = (ty + 2) * IPW + tx + 2;   // own cell in a psi/r/phi plane
    const int nc = (ty + 1) * INW + tx + 1;   // own cell in an nhat plane
    const int ph = hr * IPW + hc, nh = (hr - 1) * INW + hc - 1;
    const double hx = 0.5 * P.idx, hy = 0.5 * P.idy;
    // nhat of the cell at rectangle position q from psi planes at ring offsets om / o0 / op
    auto normal = [&](int q, int om, int o0, int op, double igz, double &nx_, double &ny_, double &nz_) {
        const double gx = (PSI[o0 + q + 1] - PSI[o0 + q - 1]) * hx;
        const double gy = (PSI[o0 + q + IPW] - PSI[o0 + q - IPW]) * hy;
        const double gz = (PSI[op + q] - PSI[om + q]) * igz;
        // HALF the normal: 0.5 G / max(|G|, 1e-30) (N4), so that a face normal is a plain sum
        const double inv = 0.5 * fz_rsqrt(fmax(gx * gx + gy * gy + gz * gz, 1e-60));
        nx_ = gx * inv; ny_ = gy * inv; nz_ = gz * inv;
    };

    // prologue: psi(k0-2 .. k0+1), r/phi(k0-2 .. k0) in three groups (the loop waits with "<= 1 pending")
    issue_psi(k0 - 2); issue_psi(k0 - 1); issue_rf(k0 - 2); fz_cp_async_commit();
    issue_psi(k0); issue_rf(k0 - 1); fz_cp_async_commit();
    issue_psi(k0 + 1); issue_rf(k0); fz_cp_async_commit();
    double nz0 = 0.0, nzp = 0.0, nfz_prev = 0.0, Rz_prev = 0.0;
    const long long gc = (i0 + tx) + (long long)P.nx * (j0 + ty);
    // ring offsets of psi planes kk-1, kk, kk+1 and of the nhat planes kk-1, kk, advanced incrementally
    int sp = (k0 - 3 + 2 * IRING_PSI) % IRING_PSI;   // slot of psi plane kk-2 before the first step
    int pm, p0 = ((sp + 1) % IRING_PSI) * IPS, pp = ((sp + 2) % IRING_PSI) * IPS;
    sp = (sp + 2) % IRING_PSI;                       // slot of plane kk (kk = k0-2 "before" the loop)
    int sn = (k0 - 2 + INRING) % INRING, n0 = sn * INS, nm;
    double igz_n = P.igz[k0 - 1], idzc_n = P.idzc[k0 - 2], idzf_n = P.idzf[k0 - 2];   // z metrics: one step ahead
    for (int kk = k0 - 1; kk <= k1; ++kk) {
        fz_cp_async_wait<1>();
        __syncthreads();
        if (kk + 3 <= k1 + 1) issue_psi(kk + 3);
        if (kk + 2 <= k1) issue_rf(kk + 2);
        fz_cp_async_commit();
        sp = (sp + 1 == IRING_PSI) ? 0 : sp + 1;
        pm = p0; p0 = pp; pp = sp * IPS;             // psi planes kk-1, kk, kk+1
        sn = (sn + 1 == INRING) ? 0 : sn + 1;
        nm = n0; n0 = sn * INS;                      // nhat planes kk-1, kk
        {   // nhat(kk): own cell, then the halo cross
            const double igz = igz_n;
            igz_n = P.igz[kk + 1];
            double ax, ay, az;
            normal(pc, pm, p0, pp, igz, ax, ay, az);
            NHX[n0 + nc] = ax; NHY[n0 + nc] = ay;
            nz0 = nzp; nzp = az;
            if (has_h) {
                normal(ph, pm, p0, pp, igz, ax, ay, az);
                NHX[n0 + nh] = ax; NHY[n0 + nh] = ay;
            }
        }
        const int k = kk - 1;
        const double idzc_k = idzc_n, idzf_k = idzf_n;   // metrics of plane k, loaded one step ago
        idzc_n = P.idzc[kk]; idzf_n = P.idzf[kk];
        if (k < k0 - 1) continue;
        const int rk = ((k + 2 * IRING_RF) & (IRING_RF - 1)) * IPS + pc;    // r, phi plane k, own cell
        const int rp = ((kk + 2 * IRING_RF) & (IRING_RF - 1)) * IPS + pc;   // plane k+1
        const double f0 = PHI[rk], r0 = RR[rk];
        // z face k+1/2 (between planes k and k+1): zero on a wall face; the face k-1/2 is carried in
        // registers from the previous step (hz = half the face normal = nf_z)
        const double zf = (P.z_wall && (k == -1 || k == P.nz - 1)) ? 0.0 : 1.0;
        const double nfzp = zf * (nz0 + nzp);
        const double Rzp = zf * (P.eps * (PHI[rp] - f0) * idzc_k - fz_sharp2(r0, RR[rp]) * nfzp);
        if (k < k0) { nfz_prev = nfzp; Rz_prev = Rzp; continue; }
        // half normals of plane k were written one step ago: visible after this step's barrier
        const double ax = NHX[nm + nc], ay = NHY[nm + nc];
        const double nfxp = ax + NHX[nm + nc + 1], nfxm = NHX[nm + nc - 1] + ax;
        const double nfyp = ay + NHY[nm + nc + INW], nfym = NHY[nm + nc - INW] + ay;
        const double ex = P.eps * P.idx, ey = P.eps * P.idy;
        const double Rxp = ex * (PHI[rk + 1] - f0) - fz_sharp2(r0, RR[rk + 1]) * nfxp;
        const double Rxm = ex * (f0 - PHI[rk - 1]) - fz_sharp2(RR[rk - 1], r0) * nfxm;
        const double Ryp = ey * (PHI[rk + IPW] - f0) - fz_sharp2(r0, RR[rk + IPW]) * nfyp;
        const double Rym = ey * (f0 - PHI[rk - IPW]) - fz_sharp2(RR[rk - IPW], r0) * nfym;
        const double izf = idzf_k;
        const long long c = (long long)k * P.sxy + gc;
        kappa[c] = -((nfxp - nfxm) * P.idx + (nfyp - nfym) * P.idy + (nfzp - nfz_prev) * izf);
        divrn[c] = (Rxp - Rxm) * P.idx + (Ryp - Rym) * P.idy + (Rzp - Rz_prev) * izf;
        if (STORE_R) { rnx[c] = Rxp; rny[c] = Ryp; rnz[c] = Rzp; }
        nfz_prev = nfzp; Rz_prev = Rzp;
    }
    fz_cp_async_wait<0>();
}
