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
    const double *u, *v, *w, *phi, *kappa, *rnx, *rny, *rnz, *p, *pp, *T;
    double *us, *vs, *ws, *hu, *hv, *hw;
    const double *scal;  // scal[1] = Gamma
    double dt, gs, zs, adt;  // adt = (gs+zs)*dt
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
        A.hu[c] = rhs;
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
        A.hv[c] = rhs;
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
        A.hw[c] = rhs;
    } else {
        A.ws[c] = 0.0;
        A.hw[c] = 0.0;
    }
}
