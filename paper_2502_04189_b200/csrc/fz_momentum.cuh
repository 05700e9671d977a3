// fz_momentum.cuh -- S3, the momentum predictor (BASELINE.json:5(iii)).
// For component a at its face:
//   RHS_a = A_a + (V_a + S_a + M_a)/rho_f + B_a
//   A advection (divergence form, 2nd order), V variable-viscosity stress, S = sigma*kappabar*d_a phi
//   (CSF), M = (rho1-rho2)(R.grad)u_a (mass-consistent regularisation flux, N9), B gravity +
//   body force + linear forcing - Boussinesq buoyancy.
//   u** = u + dt (g RHS + z RHS_old) - a dt (1/rho_f - 1/rho0) d_a p_hat,  p_hat = 2p - p_prev (N7)
// (the p_hat part of the splitting of BASELINE.json:5(iv),(v) is folded in here; D2).
// VARRHO: rho1 != rho2 (M term, 1/rho_f, p_hat term);  VARMU: mu1 != mu2;  HEAT: buoyancy.
#pragma once
#include "fz_common.cuh"

struct FzMomArgs {
    const double *u, *v, *w, *phi, *kappa, *rnx, *rny, *rnz, *p, *pp, *phat, *T;   // phat = 2p - pp (N7), marching kernel
    double *us, *vs, *ws, *hu, *hv, *hw;
    const double *scal;  // scal[1] = Gamma
    double dt, gs, zs, adt;  // adt = (gs+zs)*dt
    int keep_h;              // 0 at stage 2: the next stage has zeta = 0 and never reads the history
};

template <bool VARRHO, bool VARMU, bool HEAT>
__global__ void __launch_bounds__(256)
k_momentum(FzP P, FzMomArgs A)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i >= P.nx || j >= P.ny) return;
    const FzZ z = fz_zn(P, k);
    const int ip = fz_ip(i, P.nx), im = fz_im(i, P.nx);
    const long long nx = P.nx;
    // row bases [plane][row]
    const long long r_m = nx * (fz_im(j, P.ny) + (long long)P.ny * k);
    const long long r_0 = nx * (j + (long long)P.ny * k);
    const long long r_p = nx * (fz_ip(j, P.ny) + (long long)P.ny * k);
    const long long dzm = (long long)(z.km - k) * P.sxy, dzp = (long long)(z.kp - k) * P.sxy;
    // ghost multipliers: no-slip (odd) for u, v; wall faces zero for w and R_z
    const double om = z.gm ? -1.0 : 1.0, op = z.gp ? -1.0 : 1.0;
    const double wm = z.gm ? 0.0 : 1.0;
    const double dx = P.idx, dy = P.idy;
    const double izf = P.idzf[k], izc = P.idzc[k], izcm = P.idzc[k - 1];
    const long long c = r_0 + i;

    const double *__restrict__ u = A.u, *__restrict__ v = A.v, *__restrict__ w = A.w;
    // velocities: name = field + x offset (m,0,p) + y offset + z offset
    const double u000 = u[c], up00 = u[r_0 + ip], um00 = u[r_0 + im];
    const double u0p0 = u[r_p + i], u0m0 = u[r_m + i], ump0 = u[r_p + im];
    const double u00p = op * u[c + dzp], u00m = om * u[c + dzm], um0p = op * u[r_0 + im + dzp];
    const double v000 = v[c], vp00 = v[r_0 + ip], vm00 = v[r_0 + im];
    const double v0p0 = v[r_p + i], v0m0 = v[r_m + i], vpm0 = v[r_m + ip];
    const double v00p = op * v[c + dzp], v00m = om * v[c + dzm], v0mp = op * v[r_m + i + dzp];
    const double w000 = w[c], wp00 = w[r_0 + ip], wm00 = w[r_0 + im];
    const double w0p0 = w[r_p + i], w0m0 = w[r_m + i];
    const double w00m = wm * w[c + dzm], wp0m = wm * w[r_0 + ip + dzm], w0pm = wm * w[r_p + i + dzm];

    const double *__restrict__ phi = A.phi;
    const double f000 = phi[c], fp00 = phi[r_0 + ip], f0p0 = phi[r_p + i], f00p = phi[c + dzp];
    const double dmu = P.mu1 - P.mu2;
    // viscosities (S2: mu = mu2 + (mu1-mu2) clip(phi)); even ghosts come from the mirrored plane index
    double m000, mp00, mm00, m0p0, m0m0, m00p, m00m, mpp0, mpm0, mmp0, mp0p, mp0m, mm0p, m0pp, m0pm, m0mp;
    if (VARMU) {
#define FZ_MU(x) (P.mu2 + dmu * fz_clip01(x))
        m000 = FZ_MU(f000); mp00 = FZ_MU(fp00); m0p0 = FZ_MU(f0p0); m00p = FZ_MU(f00p);
        mm00 = FZ_MU(phi[r_0 + im]); m0m0 = FZ_MU(phi[r_m + i]); m00m = FZ_MU(phi[c + dzm]);
        mpp0 = FZ_MU(phi[r_p + ip]); mpm0 = FZ_MU(phi[r_m + ip]); mmp0 = FZ_MU(phi[r_p + im]);
        mp0p = FZ_MU(phi[r_0 + ip + dzp]); mp0m = FZ_MU(phi[r_0 + ip + dzm]); mm0p = FZ_MU(phi[r_0 + im + dzp]);
        m0pp = FZ_MU(phi[r_p + i + dzp]); m0pm = FZ_MU(phi[r_p + i + dzm]); m0mp = FZ_MU(phi[r_m + i + dzp]);
#undef FZ_MU
    } else {
        m000 = mp00 = mm00 = m0p0 = m0m0 = m00p = m00m = mpp0 = mpm0 = mmp0 = mp0p = mp0m = mm0p = m0pp =
            m0pm = m0mp = P.mu2;
    }
    const double kap0 = A.kappa[c];
    const double Gam = A.scal[1];
    double irx = 1.0 / P.rho2, iry = irx, irz = irx;
    if (VARRHO) {
        const double r000 = P.rho2 + P.drho * fz_clip01(f000);
        irx = 1.0 / (0.5 * (r000 + P.rho2 + P.drho * fz_clip01(fp00)));
        iry = 1.0 / (0.5 * (r000 + P.rho2 + P.drho * fz_clip01(f0p0)));
        irz = 1.0 / (0.5 * (r000 + P.rho2 + P.drho * fz_clip01(f00p)));
    }
    double ph000 = 0, php00 = 0, ph0p0 = 0, ph00p = 0;
    if (VARRHO) {
        ph000 = 2.0 * A.p[c] - A.pp[c];
        php00 = 2.0 * A.p[r_0 + ip] - A.pp[r_0 + ip];
        ph0p0 = 2.0 * A.p[r_p + i] - A.pp[r_p + i];
        ph00p = 2.0 * A.p[c + dzp] - A.pp[c + dzp];
    }
    const double ir0 = 1.0 / P.rho0;
    double T000 = 0;
    if (HEAT) T000 = A.T[c];

    // ================= x component, face (i+1/2, j, k) =================
    {
        const double uc_p = 0.5 * (up00 + u000), uc_m = 0.5 * (u000 + um00);
        const double Exy_p = 0.5 * (v000 + vp00) * 0.5 * (u000 + u0p0);
        const double Exy_m = 0.5 * (v0m0 + vpm0) * 0.5 * (u0m0 + u000);
        const double Exz_p = 0.5 * (w000 + wp00) * 0.5 * (u000 + u00p);
        const double Exz_m = 0.5 * (w00m + wp0m) * 0.5 * (u00m + u000);
        const double Aa = -(uc_p * uc_p - uc_m * uc_m) * dx - (Exy_p - Exy_m) * dy - (Exz_p - Exz_m) * izf;
        const double nrm_p = 2.0 * mp00 * (up00 - u000) * dx, nrm_m = 2.0 * m000 * (u000 - um00) * dx;
        const double txy_p = 0.25 * (m000 + mp00 + m0p0 + mpp0) * ((u0p0 - u000) * dy + (vp00 - v000) * dx);
        const double txy_m = 0.25 * (m0m0 + mpm0 + m000 + mp00) * ((u000 - u0m0) * dy + (vpm0 - v0m0) * dx);
        const double txz_p = 0.25 * (m000 + mp00 + m00p + mp0p) * ((u00p - u000) * izc + (wp00 - w000) * dx);
        const double txz_m = 0.25 * (m00m + mp0m + m000 + mp00) * ((u000 - u00m) * izcm + (wp0m - w00m) * dx);
        const double V = (nrm_p - nrm_m) * dx + (txy_p - txy_m) * dy + (txz_p - txz_m) * izf;
        const double S = P.sigma * 0.5 * (kap0 + A.kappa[r_0 + ip]) * (fp00 - f000) * dx;
        double M = 0.0;
        if (VARRHO) {
            const double Rty = 0.25 * (A.rny[c] + A.rny[r_0 + ip] + A.rny[r_m + i] + A.rny[r_m + ip]);
            const double Rtz = 0.25 * (A.rnz[c] + A.rnz[r_0 + ip] + wm * A.rnz[c + dzm] + wm * A.rnz[r_0 + ip + dzm]);
            M = P.drho * Gam * (A.rnx[c] * (up00 - um00) * (0.5 * dx) + Rty * (u0p0 - u0m0) * (0.5 * dy) +
                                Rtz * (u00p - u00m) * P.igz[k]);
        }
        double B = P.gx * (1.0 - P.rho_ref * irx) + P.fx + P.a_lin * u000;
        if (HEAT) B -= P.gx * P.beta * (0.5 * (T000 + A.T[r_0 + ip]) - P.t_ref);
        const double rhs = Aa + (V + S + M) * irx + B;
        double un = u000 + A.dt * (A.gs * rhs + A.zs * A.hu[c]);
        if (VARRHO) un -= A.adt * (irx - ir0) * (php00 - ph000) * dx;
        A.us[c] = un;
        if (A.keep_h) A.hu[c] = rhs;
    }
    // ================= y component, face (i, j+1/2, k) =================
    {
        const double vc_p = 0.5 * (v0p0 + v000), vc_m = 0.5 * (v000 + v0m0);
        const double Eyx_p = 0.5 * (u000 + u0p0) * 0.5 * (v000 + vp00);
        const double Eyx_m = 0.5 * (um00 + ump0) * 0.5 * (vm00 + v000);
        const double Eyz_p = 0.5 * (w000 + w0p0) * 0.5 * (v000 + v00p);
        const double Eyz_m = 0.5 * (w00m + w0pm) * 0.5 * (v00m + v000);
        const double Aa = -(vc_p * vc_p - vc_m * vc_m) * dy - (Eyx_p - Eyx_m) * dx - (Eyz_p - Eyz_m) * izf;
        const double nrm_p = 2.0 * m0p0 * (v0p0 - v000) * dy, nrm_m = 2.0 * m000 * (v000 - v0m0) * dy;
        const double tyx_p = 0.25 * (m000 + m0p0 + mp00 + mpp0) * ((vp00 - v000) * dx + (u0p0 - u000) * dy);
        const double tyx_m = 0.25 * (mm00 + mmp0 + m000 + m0p0) * ((v000 - vm00) * dx + (ump0 - um00) * dy);
        const double tyz_p = 0.25 * (m000 + m0p0 + m00p + m0pp) * ((v00p - v000) * izc + (w0p0 - w000) * dy);
        const double tyz_m = 0.25 * (m00m + m0pm + m000 + m0p0) * ((v000 - v00m) * izcm + (w0pm - w00m) * dy);
        const double V = (nrm_p - nrm_m) * dy + (tyx_p - tyx_m) * dx + (tyz_p - tyz_m) * izf;
        const double S = P.sigma * 0.5 * (kap0 + A.kappa[r_p + i]) * (f0p0 - f000) * dy;
        double M = 0.0;
        if (VARRHO) {
            const double Rtx = 0.25 * (A.rnx[c] + A.rnx[r_p + i] + A.rnx[r_0 + im] + A.rnx[r_p + im]);
            const double Rtz = 0.25 * (A.rnz[c] + A.rnz[r_p + i] + wm * A.rnz[c + dzm] + wm * A.rnz[r_p + i + dzm]);
            M = P.drho * Gam * (A.rny[c] * (v0p0 - v0m0) * (0.5 * dy) + Rtx * (vp00 - vm00) * (0.5 * dx) +
                                Rtz * (v00p - v00m) * P.igz[k]);
        }
        double B = P.gy * (1.0 - P.rho_ref * iry) + P.fy + P.a_lin * v000;
        if (HEAT) B -= P.gy * P.beta * (0.5 * (T000 + A.T[r_p + i]) - P.t_ref);
        const double rhs = Aa + (V + S + M) * iry + B;
        double vn = v000 + A.dt * (A.gs * rhs + A.zs * A.hv[c]);
        if (VARRHO) vn -= A.adt * (iry - ir0) * (ph0p0 - ph000) * dy;
        A.vs[c] = vn;
        if (A.keep_h) A.hv[c] = rhs;
    }
    // ================= z component, face (i, j, k+1/2) =================
    if (k < P.kzf) {
        // here k+1 is never a wall ghost, so the "p" plane values are plain (op = 1)
        const double w00p = w[c + dzp];
        const double izfp = P.idzf[k + 1];
        const double wc_p = 0.5 * (w00p + w000), wc_m = 0.5 * (w000 + w00m);
        const double Ezx_p = 0.5 * (u000 + u00p) * 0.5 * (w000 + wp00);
        const double Ezx_m = 0.5 * (um00 + um0p) * 0.5 * (wm00 + w000);
        const double Ezy_p = 0.5 * (v000 + v00p) * 0.5 * (w000 + w0p0);
        const double Ezy_m = 0.5 * (v0m0 + v0mp) * 0.5 * (w0m0 + w000);
        const double Aa = -(wc_p * wc_p - wc_m * wc_m) * izc - (Ezx_p - Ezx_m) * dx - (Ezy_p - Ezy_m) * dy;
        const double nrm_p = 2.0 * m00p * (w00p - w000) * izfp, nrm_m = 2.0 * m000 * (w000 - w00m) * izf;
        const double tzx_p = 0.25 * (m000 + m00p + mp00 + mp0p) * ((wp00 - w000) * dx + (u00p - u000) * izc);
        const double tzx_m = 0.25 * (mm00 + mm0p + m000 + m00p) * ((w000 - wm00) * dx + (um0p - um00) * izc);
        const double tzy_p = 0.25 * (m000 + m00p + m0p0 + m0pp) * ((w0p0 - w000) * dy + (v00p - v000) * izc);
        const double tzy_m = 0.25 * (m0m0 + m0mp + m000 + m00p) * ((w000 - w0m0) * dy + (v0mp - v0m0) * izc);
        const double V = (nrm_p - nrm_m) * izc + (tzx_p - tzx_m) * dx + (tzy_p - tzy_m) * dy;
        const double S = P.sigma * 0.5 * (kap0 + A.kappa[c + dzp]) * (f00p - f000) * izc;
        double M = 0.0;
        if (VARRHO) {
            const double Rtx = 0.25 * (A.rnx[c] + A.rnx[c + dzp] + A.rnx[r_0 + im] + A.rnx[r_0 + im + dzp]);
            const double Rty = 0.25 * (A.rny[c] + A.rny[c + dzp] + A.rny[r_m + i] + A.rny[r_m + i + dzp]);
            M = P.drho * Gam * (A.rnz[c] * (w00p - w00m) / (P.dzf[k + 1] + P.dzf[k]) +
                                Rtx * (wp00 - wm00) * (0.5 * dx) + Rty * (w0p0 - w0m0) * (0.5 * dy));
        }
        double B = P.gz * (1.0 - P.rho_ref * irz) + P.fz + P.a_lin * w000;
        if (HEAT) B -= P.gz * P.beta * (0.5 * (T000 + A.T[c + dzp]) - P.t_ref);
        const double rhs = Aa + (V + S + M) * irz + B;
        double wn = w000 + A.dt * (A.gs * rhs + A.zs * A.hw[c]);
        if (VARRHO) wn -= A.adt * (irz - ir0) * (ph00p - ph000) * izc;
        A.ws[c] = wn;
        if (A.keep_h) A.hw[c] = rhs;
    } else {
        A.ws[c] = 0.0;
        if (A.keep_h) A.hw[c] = 0.0;
    }
}

// =====================================================================================
// 2.5-D marching variant (the one used when nx >= 32 and ny >= 8).  A CTA owns an x-y tile of
// MTX x MTY cells and marches over a chunk of z planes.  Every staged field keeps a ring of five
// planes (tile + halo 2 in x, 1 in y) in shared memory, filled by 16-byte cp.async copies (LDGSTS)
// issued two planes ahead of their use: each plane is read from HBM once per chunk, all 60-odd
// neighbour reads of the stencil are shared-memory reads, and no register is tied up by a load in
// flight -- DRAM latency is hidden by the pipeline rather than by occupancy.  One barrier per
// plane.  Wall ghosts (no-slip: -u, -v; impermeable: w = 0, R_z = 0; mirror: phi, kappa, p_hat)
// are applied when a ghost plane is READ: the ring holds the mirrored source plane unchanged.
#ifndef MOM_MINB
#define MOM_MINB 3
#endif
#define MTX 32
#define MTY 8
#define MPW (MTX + 4)
#define MPH (MTY + 2)
#define MPS (MPW * MPH)
#define MCHUNKS (MPS / 2)

// Staged fields and ring depth.  rho1 == rho2: u, v, w, phi, kappa (+T), rings of five planes (copies issued two
// planes ahead), three (two with heat) CTAs per SM.  rho1 != rho2: also Rn on the three faces and p_hat = 2p - p_prev
// (formed once by k_correct, N7): nine fields, rings of FOUR planes (one plane ahead: a plane of this variant takes
// several microseconds) = 104 KB (115 200 B with T: two CTAs of that size still fit the 228 KB of an SM), so that TWO
// CTAs share an SM -- the variant is bound by dependent fp64 chains and needs the warps.
template <bool VARRHO, bool HEAT>
struct FzMomFields {
    static constexpr int U = 0, V = 1, W = 2, PHI = 3, KAP = 4;
    static constexpr bool T_STAGED = HEAT;
    static constexpr int T = 5;                            // valid if T_STAGED
    static constexpr int RX = 5 + (T_STAGED ? 1 : 0);      // valid if VARRHO
    static constexpr int RY = RX + 1, RZ = RX + 2, PH = RX + 3;
    static constexpr int NF = 5 + (T_STAGED ? 1 : 0) + (VARRHO ? 4 : 0);
    static constexpr int RING = VARRHO ? 4 : 5;
    static constexpr int MINB = VARRHO ? 2 : (HEAT ? 2 : MOM_MINB);
};

template <bool VARRHO, bool VARMU, bool HEAT>
__global__ void __launch_bounds__(MTX * MTY, FzMomFields<VARRHO, HEAT>::MINB)
k_momentum_march(FzP P, FzMomArgs A, int KC)
{
    using F = FzMomFields<VARRHO, HEAT>;
    constexpr int NF = F::NF, MRING = F::RING;
    extern __shared__ __align__(16) double smm[];  // [NF][MRING][MPS]
    const int tx = threadIdx.x, ty = threadIdx.y, t = ty * MTX + tx;
    const int i0 = blockIdx.x * MTX, j0 = blockIdx.y * MTY;
    const int i = i0 + tx, j = j0 + ty;
    const int k0 = blockIdx.z * KC, k1 = min(k0 + KC, P.nz);
    const int cidx = (ty + 1) * MPW + (tx + 2);
    const unsigned ugc = (unsigned)(i + P.nx * j);   // 32-bit cell offsets: N < 2^31 (fizzy_create)
    // staging map: thread t < MCHUNKS copies 16-byte chunk t of the staged rectangle of every field
    const bool loader = t < MCHUNKS;
    const int lrow = t / (MPW / 2), lcp = t - lrow * (MPW / 2);
    const long long goff_l = ((i0 - 2 + 2 * lcp + P.nx) & (P.nx - 1)) +
                             (long long)P.nx * ((j0 - 1 + lrow + P.ny) & (P.ny - 1));
    const int soff = lrow * MPW + 2 * lcp;

    const double *src[NF];
    src[F::U] = A.u; src[F::V] = A.v; src[F::W] = A.w; src[F::PHI] = A.phi; src[F::KAP] = A.kappa;
    if (F::T_STAGED) src[F::T] = A.T;
    if (VARRHO) { src[F::RX] = A.rnx; src[F::RY] = A.rny; src[F::RZ] = A.rnz; src[F::PH] = A.phat; }

    // copy plane kk (k0-1 .. k1; ghosts: periodic wrap or wall mirror) of every field into ring slot
    // kk mod MRING.  Planes are issued in increasing order: the slot advances incrementally; offsets are
    // 32-bit (fizzy_create guarantees N < 2^31).
    const unsigned sxy = (unsigned)P.sxy, ugoff = (unsigned)goff_l;
    const int zlo = P.z_wall ? 0 : P.nz - 1, zhi = P.z_wall ? P.nz - 1 : 0;   // source of plane -1 / nz
    int sl_is = (k0 - 1 + MRING) % MRING;
    auto issue = [&](int kk) {
        if (loader && kk <= k1) {
            const int sp = kk < 0 ? zlo : (kk >= P.nz ? zhi : kk);
            const unsigned g = (unsigned)sp * sxy + ugoff;
            const int o = sl_is * MPS + soff;
#pragma unroll
            for (int f = 0; f < NF; ++f) fz_cp_async16(smm + f * (MRING * MPS) + o, src[f] + g);
        }
        sl_is = (sl_is + 1 == MRING) ? 0 : sl_is + 1;
    };
    issue(k0 - 1); issue(k0); fz_cp_async_commit();
#pragma unroll
    for (int d = 1; d <= MRING - 3; ++d) { issue(k0 + d); fz_cp_async_commit(); }

    const double dx = P.idx, dy = P.idy;
    const double hdmu = 0.5 * (P.mu1 - P.mu2), mumid = 0.5 * (P.mu1 + P.mu2);
    const double qdrho = 0.25 * P.drho, rhomid = 0.5 * (P.rho1 + P.rho2);
    const double ir0 = 1.0 / P.rho0;
    const double Gam = A.scal[1];

    int sl = (k0 - 1 + MRING) % MRING;   // ring slot of plane k-1, advanced incrementally
    int om, o0 = sl * MPS + cidx, op = ((sl + 1) % MRING) * MPS + cidx;
    sl = (sl + 1) % MRING;
    // stage 0 has zeta = 0: the RK histories are not read at all (-24 B/cell on that substep)
    const bool use_h = A.zs != 0.0;
    double hu_nx = 0.0, hv_nx = 0.0, hw_nx = 0.0;
    if (use_h) {
        hu_nx = A.hu[(unsigned)k0 * sxy + ugc]; hv_nx = A.hv[(unsigned)k0 * sxy + ugc];
        hw_nx = A.hw[(unsigned)k0 * sxy + ugc];
    }
    double izc_0 = P.idzc[k0 - 1], izc_n = P.idzc[k0], izf_p = P.idzf[k0], izf_n = P.idzf[k0 + 1];
    for (int k = k0; k < k1; ++k) {
        fz_cp_async_wait<MRING - 4>();
        __syncthreads();
        issue(k + MRING - 2);
        fz_cp_async_commit();
        sl = (sl + 1 == MRING) ? 0 : sl + 1;
        om = o0; o0 = op; op = sl * MPS + cidx;   // planes k-1, k, k+1
        const unsigned c = (unsigned)k * sxy + ugc;
        // RK histories: loaded one plane ahead (registers), so their latency hides behind a whole plane
        const double hu_old = hu_nx, hv_old = hv_nx, hw_old = hw_nx;
        if (use_h && k + 1 < k1) { hu_nx = A.hu[c + sxy]; hv_nx = A.hv[c + sxy]; hw_nx = A.hw[c + sxy]; }
        // ghost rules at the walls: the ring slot of plane -1 / nz arrives holding the mirrored interior plane.
        // rho1 == rho2 (GHOST_SMEM): the two plane steps that read it turn it into the ghost plane first (no-slip: -u, -v;
        // impermeable: w = 0; phi, kappa, T are even and stay), so that the other nz-2 steps -- and every step of a periodic
        // grid -- carry no sign factors (round 2: nine DMUL and a dozen select / predicate instructions per cell, in every
        // configuration).  rho1 != rho2: the factors are applied when a ghost plane is READ, as before -- with nine staged
        // fields at 128 registers the extra block costs that variant 3-4 % (measured on configs 3 and 5).
        constexpr bool GHOST_SMEM = !VARRHO;
        const bool gm = !GHOST_SMEM && P.z_wall && k == 0, gp = !GHOST_SMEM && P.z_wall && k == P.nz - 1;
        const double sgm = gm ? -1.0 : 1.0, sgp = gp ? -1.0 : 1.0, wm = gm ? 0.0 : 1.0;
        if (GHOST_SMEM && P.z_wall && (k == 0 || k == P.nz - 1)) {
            const int gb = (k == 0 ? om : op) - cidx;
            for (int e = t; e < MPS; e += MTX * MTY) {
                smm[F::U * (MRING * MPS) + gb + e] = -smm[F::U * (MRING * MPS) + gb + e];
                smm[F::V * (MRING * MPS) + gb + e] = -smm[F::V * (MRING * MPS) + gb + e];
                if (k == 0) smm[F::W * (MRING * MPS) + gb + e] = 0.0;
            }
            __syncthreads();
        }
        // S(f, di, dj, plane offset) -- shared-memory neighbour read
#define S_(f, di, dj, o) smm[(f) * (MRING * MPS) + (o) + (dj) * MPW + (di)]   // o includes cidx
        // z metrics come from global tables: carried / loaded one plane ahead so that no plane waits for them
        const double izf = izf_p, izc = izc_n, izcm = izc_0;
        izc_0 = izc_n; izf_p = izf_n;
        izc_n = P.idzc[k + 1]; izf_n = P.idzf[k + 2];
        const double izfp = izf_p;   // 1/dzf[k+1]
        const double u000 = S_(F::U, 0, 0, o0), up00 = S_(F::U, 1, 0, o0), um00 = S_(F::U, -1, 0, o0);
        const double u0p0 = S_(F::U, 0, 1, o0), u0m0 = S_(F::U, 0, -1, o0), ump0 = S_(F::U, -1, 1, o0);
        const double u00p = sgp * S_(F::U, 0, 0, op), u00m = sgm * S_(F::U, 0, 0, om), um0p = sgp * S_(F::U, -1, 0, op);
        const double v000 = S_(F::V, 0, 0, o0), vp00 = S_(F::V, 1, 0, o0), vm00 = S_(F::V, -1, 0, o0);
        const double v0p0 = S_(F::V, 0, 1, o0), v0m0 = S_(F::V, 0, -1, o0), vpm0 = S_(F::V, 1, -1, o0);
        const double v00p = sgp * S_(F::V, 0, 0, op), v00m = sgm * S_(F::V, 0, 0, om), v0mp = sgp * S_(F::V, 0, -1, op);
        const double w000 = S_(F::W, 0, 0, o0), wp00 = S_(F::W, 1, 0, o0), wm00 = S_(F::W, -1, 0, o0);
        const double w0p0 = S_(F::W, 0, 1, o0), w0m0 = S_(F::W, 0, -1, o0);
        const double w00m = wm * S_(F::W, 0, 0, om), wp0m = wm * S_(F::W, 1, 0, om), w0pm = wm * S_(F::W, 0, 1, om);
        const double f000 = S_(F::PHI, 0, 0, o0), fp00 = S_(F::PHI, 1, 0, o0), f0p0 = S_(F::PHI, 0, 1, o0),
                     f00p = S_(F::PHI, 0, 0, op);
        double m000, mp00, mm00, m0p0, m0m0, m00p, m00m, mpp0, mpm0, mmp0, mp0p, mp0m, mm0p, m0pp, m0pm, m0mp;
        if (VARMU) {
#define FZ_MU(x) fma(hdmu, fz_sclip(x), mumid)
            m000 = FZ_MU(f000); mp00 = FZ_MU(fp00); m0p0 = FZ_MU(f0p0); m00p = FZ_MU(f00p);
            mm00 = FZ_MU(S_(F::PHI, -1, 0, o0)); m0m0 = FZ_MU(S_(F::PHI, 0, -1, o0)); m00m = FZ_MU(S_(F::PHI, 0, 0, om));
            mpp0 = FZ_MU(S_(F::PHI, 1, 1, o0)); mpm0 = FZ_MU(S_(F::PHI, 1, -1, o0)); mmp0 = FZ_MU(S_(F::PHI, -1, 1, o0));
            mp0p = FZ_MU(S_(F::PHI, 1, 0, op)); mp0m = FZ_MU(S_(F::PHI, 1, 0, om)); mm0p = FZ_MU(S_(F::PHI, -1, 0, op));
            m0pp = FZ_MU(S_(F::PHI, 0, 1, op)); m0pm = FZ_MU(S_(F::PHI, 0, 1, om)); m0mp = FZ_MU(S_(F::PHI, 0, -1, op));
#undef FZ_MU
        } else {
            m000 = mp00 = mm00 = m0p0 = m0m0 = m00p = m00m = mpp0 = mpm0 = mmp0 = mp0p = mp0m = mm0p = m0pp =
                m0pm = m0mp = P.mu2;
        }
        const double kap0 = S_(F::KAP, 0, 0, o0);
        double irx = 1.0 / P.rho2, iry = irx, irz = irx;
        double ph000 = 0, php00 = 0, ph0p0 = 0, ph00p = 0;
        if (VARRHO) {
            // rho_f = 1/2 (rho + rho(+1_a)) = rhomid + 1/4 drho (sclip + sclip(+1_a))   (fz_sclip: 2 clip - 1)
            const double s000 = fz_sclip(f000);
            irx = fz_rcp(fma(qdrho, s000 + fz_sclip(fp00), rhomid));
            iry = fz_rcp(fma(qdrho, s000 + fz_sclip(f0p0), rhomid));
            irz = fz_rcp(fma(qdrho, s000 + fz_sclip(f00p), rhomid));
            // p_hat = 2 p - p_prev (N7), formed by k_correct of the previous substep
            ph000 = S_(F::PH, 0, 0, o0); php00 = S_(F::PH, 1, 0, o0); ph0p0 = S_(F::PH, 0, 1, o0);
            ph00p = S_(F::PH, 0, 0, op);
        }
        // temperature at the cell and its three "+" neighbours: staged, or straight from global memory (T_ mirrors S_)
        double T000 = 0, Tp00 = 0, T0p0 = 0, T00p = 0;
        if (HEAT) {
            if (F::T_STAGED) {
                T000 = S_(F::T, 0, 0, o0); Tp00 = S_(F::T, 1, 0, o0); T0p0 = S_(F::T, 0, 1, o0); T00p = S_(F::T, 0, 0, op);
            } else {
                const long long row = (long long)k * P.sxy + (long long)P.nx * j;
                T000 = A.T[c]; Tp00 = A.T[row + fz_ip(i, P.nx)];
                T0p0 = A.T[(long long)k * P.sxy + (long long)P.nx * fz_ip(j, P.ny) + i];
                T00p = k < P.kzf ? A.T[c + P.sxy - (k + 1 == P.nz ? P.N : 0)] : 0.0;
            }
        }
        // edge viscosity (N11): mean of the four cells around the edge; a constant if mu1 == mu2
#define MUE_(a_, b_, c_, d_) (VARMU ? 0.25 * ((a_) + (b_) + (c_) + (d_)) : P.mu2)
        // advective edge products and edge stresses on the three "+" edges of the cell, shared by
        // the two components that meet there.  The halves of the face averages are folded into the metric factors
        // (q* = 1/4 of the reciprocal spacing): E' = (sum of two)(sum of two), uc' = sum of two.
        const double qx = 0.25 * dx, qy = 0.25 * dy, qzf = 0.25 * izf, qzc = 0.25 * izc;
        const double Exy_p = (v000 + vp00) * (u000 + u0p0);
        const double Exz_p = (w000 + wp00) * (u000 + u00p);
        const double Eyz_p = (w000 + w0p0) * (v000 + v00p);
        const double txy_p = MUE_(m000, mp00, m0p0, mpp0) * ((u0p0 - u000) * dy + (vp00 - v000) * dx);
        const double txz_p = MUE_(m000, mp00, m00p, mp0p) * ((u00p - u000) * izc + (wp00 - w000) * dx);
        const double tyz_p = MUE_(m000, m0p0, m00p, m0pp) * ((v00p - v000) * izc + (w0p0 - w000) * dy);
        const double hs = 0.5 * P.sigma;
        // ================= x component =================
        {
            const double uc_p = up00 + u000, uc_m = u000 + um00;
            const double Exy_m = (v0m0 + vpm0) * (u0m0 + u000);
            const double Exz_m = (w00m + wp0m) * (u00m + u000);
            const double Aa = -((uc_p * uc_p - uc_m * uc_m) * qx + (Exy_p - Exy_m) * qy + (Exz_p - Exz_m) * qzf);
            const double nrm_p = mp00 * (up00 - u000), nrm_m = m000 * (u000 - um00);
            const double txy_m = MUE_(m0m0, mpm0, m000, mp00) * ((u000 - u0m0) * dy + (vpm0 - v0m0) * dx);
            const double txz_m = MUE_(m00m, mp0m, m000, mp00) * ((u000 - u00m) * izcm + (wp0m - w00m) * dx);
            const double V = (nrm_p - nrm_m) * (2.0 * dx * dx) + (txy_p - txy_m) * dy + (txz_p - txz_m) * izf;
            const double Sf = (hs * dx) * (kap0 + S_(F::KAP, 1, 0, o0)) * (fp00 - f000);
            double M = 0.0;
            if (VARRHO) {
                const double Rty = 0.25 * (S_(F::RY, 0, 0, o0) + S_(F::RY, 1, 0, o0) + S_(F::RY, 0, -1, o0) + S_(F::RY, 1, -1, o0));
                const double Rtz = 0.25 * (S_(F::RZ, 0, 0, o0) + S_(F::RZ, 1, 0, o0) + wm * (S_(F::RZ, 0, 0, om) + S_(F::RZ, 1, 0, om)));
                M = P.drho * Gam * (S_(F::RX, 0, 0, o0) * (up00 - um00) * (0.5 * dx) + Rty * (u0p0 - u0m0) * (0.5 * dy) +
                                    Rtz * (u00p - u00m) * P.igz[k]);
            }
            double B = P.gx * (1.0 - P.rho_ref * irx) + P.fx + P.a_lin * u000;
            if (HEAT) B -= P.gx * P.beta * (0.5 * (T000 + Tp00) - P.t_ref);
            const double rhs = Aa + (V + Sf + M) * irx + B;
            double un = u000 + A.dt * (A.gs * rhs + A.zs * hu_old);
            if (VARRHO) un -= A.adt * (irx - ir0) * (php00 - ph000) * dx;
            A.us[c] = un;
            if (A.keep_h) A.hu[c] = rhs;
        }
        // ================= y component =================
        {
            const double vc_p = v0p0 + v000, vc_m = v000 + v0m0;
            const double Eyx_p = Exy_p;
            const double Eyx_m = (um00 + ump0) * (vm00 + v000);
            const double Eyz_m = (w00m + w0pm) * (v00m + v000);
            const double Aa = -((vc_p * vc_p - vc_m * vc_m) * qy + (Eyx_p - Eyx_m) * qx + (Eyz_p - Eyz_m) * qzf);
            const double nrm_p = m0p0 * (v0p0 - v000), nrm_m = m000 * (v000 - v0m0);
            const double tyx_p = txy_p;
            const double tyx_m = MUE_(mm00, mmp0, m000, m0p0) * ((v000 - vm00) * dx + (ump0 - um00) * dy);
            const double tyz_m = MUE_(m00m, m0pm, m000, m0p0) * ((v000 - v00m) * izcm + (w0pm - w00m) * dy);
            const double V = (nrm_p - nrm_m) * (2.0 * dy * dy) + (tyx_p - tyx_m) * dx + (tyz_p - tyz_m) * izf;
            const double Sf = (hs * dy) * (kap0 + S_(F::KAP, 0, 1, o0)) * (f0p0 - f000);
            double M = 0.0;
            if (VARRHO) {
                const double Rtx = 0.25 * (S_(F::RX, 0, 0, o0) + S_(F::RX, 0, 1, o0) + S_(F::RX, -1, 0, o0) + S_(F::RX, -1, 1, o0));
                const double Rtz = 0.25 * (S_(F::RZ, 0, 0, o0) + S_(F::RZ, 0, 1, o0) + wm * (S_(F::RZ, 0, 0, om) + S_(F::RZ, 0, 1, om)));
                M = P.drho * Gam * (S_(F::RY, 0, 0, o0) * (v0p0 - v0m0) * (0.5 * dy) + Rtx * (vp00 - vm00) * (0.5 * dx) +
                                    Rtz * (v00p - v00m) * P.igz[k]);
            }
            double B = P.gy * (1.0 - P.rho_ref * iry) + P.fy + P.a_lin * v000;
            if (HEAT) B -= P.gy * P.beta * (0.5 * (T000 + T0p0) - P.t_ref);
            const double rhs = Aa + (V + Sf + M) * iry + B;
            double vn = v000 + A.dt * (A.gs * rhs + A.zs * hv_old);
            if (VARRHO) vn -= A.adt * (iry - ir0) * (ph0p0 - ph000) * dy;
            A.vs[c] = vn;
            if (A.keep_h) A.hv[c] = rhs;
        }
        // ================= z component =================
        if (k < P.kzf) {
            const double w00p = S_(F::W, 0, 0, op);
            const double wc_p = w00p + w000, wc_m = w000 + w00m;
            const double Ezx_p = Exz_p;
            const double Ezx_m = (um00 + um0p) * (wm00 + w000);
            const double Ezy_p = Eyz_p;
            const double Ezy_m = (v0m0 + v0mp) * (w0m0 + w000);
            const double Aa = -((wc_p * wc_p - wc_m * wc_m) * qzc + (Ezx_p - Ezx_m) * qx + (Ezy_p - Ezy_m) * qy);
            const double nrm_p = m00p * (w00p - w000) * izfp, nrm_m = m000 * (w000 - w00m) * izf;
            const double tzx_p = txz_p;
            const double tzx_m = MUE_(mm00, mm0p, m000, m00p) * ((w000 - wm00) * dx + (um0p - um00) * izc);
            const double tzy_p = tyz_p;
            const double tzy_m = MUE_(m0m0, m0mp, m000, m00p) * ((w000 - w0m0) * dy + (v0mp - v0m0) * izc);
            const double V = (nrm_p - nrm_m) * (2.0 * izc) + (tzx_p - tzx_m) * dx + (tzy_p - tzy_m) * dy;
            const double Sf = (hs * izc) * (kap0 + S_(F::KAP, 0, 0, op)) * (f00p - f000);
            double M = 0.0;
            if (VARRHO) {
                const double Rtx = 0.25 * (S_(F::RX, 0, 0, o0) + S_(F::RX, 0, 0, op) + S_(F::RX, -1, 0, o0) + S_(F::RX, -1, 0, op));
                const double Rty = 0.25 * (S_(F::RY, 0, 0, o0) + S_(F::RY, 0, 0, op) + S_(F::RY, 0, -1, o0) + S_(F::RY, 0, -1, op));
                M = P.drho * Gam * (S_(F::RZ, 0, 0, o0) * (w00p - w00m) * fz_rcp(P.dzf[k + 1] + P.dzf[k]) +
                                    Rtx * (wp00 - wm00) * (0.5 * dx) + Rty * (w0p0 - w0m0) * (0.5 * dy));
            }
            double B = P.gz * (1.0 - P.rho_ref * irz) + P.fz + P.a_lin * w000;
            if (HEAT) B -= P.gz * P.beta * (0.5 * (T000 + T00p) - P.t_ref);
            const double rhs = Aa + (V + Sf + M) * irz + B;
            double wn = w000 + A.dt * (A.gs * rhs + A.zs * hw_old);
            if (VARRHO) wn -= A.adt * (irz - ir0) * (ph00p - ph000) * izc;
            A.ws[c] = wn;
            if (A.keep_h) A.hw[c] = rhs;
        } else {
            A.ws[c] = 0.0;
            if (A.keep_h) A.hw[c] = 0.0;
        }
#undef S_
#undef MUE_
    }
}
