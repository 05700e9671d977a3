// fz_stencil.cuh -- finite-difference kernels of the RK3 substep (DESIGN.md steps S0-S3, S5).
// One thread per cell, x fastest; 3-D launch: blockIdx.z = k.  Neighbour reuse comes from L1/L2.
// Passages: BASELINE.json:5 (i)-(iii),(v); readings N2-N15 in DESIGN.md.
#pragma once
#include "fz_common.cuh"

#define FZ_CELL_IJK                                          \
    const int i = blockIdx.x * blockDim.x + threadIdx.x;     \
    const int j = blockIdx.y * blockDim.y + threadIdx.y;     \
    const int k = blockIdx.z;                                \
    if (i >= P.nx || j >= P.ny) return;

// ---------------------------------------------------------------- S0: max |u|, Gamma latch
__global__ void k_absmax3(FzP P, const double *__restrict__ u, const double *__restrict__ v,
                          const double *__restrict__ w, double *umax)
{
    double m = 0.0;
    for (long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x; c < P.N;
         c += (long long)gridDim.x * blockDim.x)
        m = fmax(m, fmax(fabs(u[c]), fmax(fabs(v[c]), fabs(w[c]))));
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) fz_atomic_max_nonneg(umax, m);
}

// fizzy_set_fields: running max|u| = 0 (k_absmax3 follows), Gamma = gamma_abs until the first stage-0 latch
__global__ void k_init_scalars(FzP P, double *scal)
{
    scal[0] = 0.0;
    scal[1] = P.gamma_abs;
}

// scal[0] = running max|u| (reset here), scal[1] = Gamma (latched here; N15)
__global__ void k_latch_gamma(FzP P, double *scal)
{
    scal[1] = P.gamma_rel * scal[0] + P.gamma_abs;
    scal[0] = 0.0;
}

// ---------------------------------------------------------------- interface quantities (N2-N5)
// (a) psi = eps ln q, r = sqrt(q), q = (phic+delta)/(1-phic+delta)
__global__ void k_iface_psi(FzP P, const double *__restrict__ phi, double *__restrict__ psi,
                            double *__restrict__ rr)
{
    FZ_CELL_IJK
    const long long c = i + (long long)P.nx * (j + (long long)P.ny * k);
    const double ph = fz_clip01(phi[c]);
    psi[c] = fz_psi(P, phi[c]);
    rr[c] = sqrt((ph + P.delta) / (1.0 - ph + P.delta));
}

// (b) nhat = G / max(|G|, 1e-30), G = central difference of psi (mirror at walls)
__global__ void k_iface_nhat(FzP P, const double *__restrict__ psi, double *__restrict__ nhx,
                             double *__restrict__ nhy, double *__restrict__ nhz)
{
    FZ_CELL_IJK
    const FzZ z = fz_zn(P, k);
    const long long row = (long long)P.nx * (j + (long long)P.ny * k);
    const long long c = row + i;
    const double gx = (psi[row + fz_ip(i, P.nx)] - psi[row + fz_im(i, P.nx)]) * (0.5 * P.idx);
    const double gy = (psi[i + (long long)P.nx * (fz_ip(j, P.ny) + (long long)P.ny * k)] -
                       psi[i + (long long)P.nx * (fz_im(j, P.ny) + (long long)P.ny * k)]) * (0.5 * P.idy);
    const double gz = (psi[c + (long long)(z.kp - k) * P.sxy] - psi[c + (long long)(z.km - k) * P.sxy]) * P.igz[k];
    const double mag = sqrt(gx * gx + gy * gy + gz * gz);
    const double inv = 1.0 / fmax(mag, 1e-30);
    nhx[c] = gx * inv;
    nhy[c] = gy * inv;
    nhz[c] = gz * inv;
}

// sharpening coefficient 1/4 (1 - tanh^2((psi_a+psi_b)/(4 eps))) = s/(1+s)^2, s = r_a r_b (N3)
__device__ __forceinline__ double fz_sharp(double ra, double rb)
{
    const double s = ra * rb;
    const double d = 1.0 + s;
    return s / (d * d);
}

// (c) Rn = R/Gamma on the three "+" faces, kappa = -D(nf), divRn = D(Rn)
template <bool STORE_R>
__global__ void k_iface_flux(FzP P, const double *__restrict__ phi, const double *__restrict__ rr,
                             const double *__restrict__ nhx, const double *__restrict__ nhy,
                             const double *__restrict__ nhz, double *__restrict__ kappa,
                             double *__restrict__ divrn, double *__restrict__ rnx,
                             double *__restrict__ rny, double *__restrict__ rnz)
{
    FZ_CELL_IJK
    const FzZ z = fz_zn(P, k);
    const long long pl = (long long)P.ny * k;
    const long long c = i + P.nx * (j + pl);
    const long long xp = fz_ip(i, P.nx) + P.nx * (j + pl), xm = fz_im(i, P.nx) + P.nx * (j + pl);
    const long long yp = i + P.nx * (fz_ip(j, P.ny) + pl), ym = i + P.nx * (fz_im(j, P.ny) + pl);
    const long long zp = c + (long long)(z.kp - k) * P.sxy, zm = c + (long long)(z.km - k) * P.sxy;
    const double f0 = phi[c], r0 = rr[c];
    const double ax = nhx[c], ay = nhy[c], az = nhz[c];
    // x faces
    const double nfxp = 0.5 * (ax + nhx[xp]), nfxm = 0.5 * (nhx[xm] + ax);
    const double Rxp = P.eps * (phi[xp] - f0) * P.idx - fz_sharp(r0, rr[xp]) * nfxp;
    const double Rxm = P.eps * (f0 - phi[xm]) * P.idx - fz_sharp(rr[xm], r0) * nfxm;
    // y faces
    const double nfyp = 0.5 * (ay + nhy[yp]), nfym = 0.5 * (nhy[ym] + ay);
    const double Ryp = P.eps * (phi[yp] - f0) * P.idy - fz_sharp(r0, rr[yp]) * nfyp;
    const double Rym = P.eps * (f0 - phi[ym]) * P.idy - fz_sharp(rr[ym], r0) * nfym;
    // z faces (zero on wall faces)
    double nfzp = 0.0, nfzm = 0.0, Rzp = 0.0, Rzm = 0.0;
    if (!z.gp) {
        nfzp = 0.5 * (az + nhz[zp]);
        Rzp = P.eps * (phi[zp] - f0) * P.idzc[k] - fz_sharp(r0, rr[zp]) * nfzp;
    }
    if (!z.gm) {
        nfzm = 0.5 * (nhz[zm] + az);
        Rzm = P.eps * (f0 - phi[zm]) * P.idzc[k - 1] - fz_sharp(rr[zm], r0) * nfzm;
    }
    kappa[c] = -((nfxp - nfxm) * P.idx + (nfyp - nfym) * P.idy + (nfzp - nfzm) * P.idzf[k]);
    divrn[c] = (Rxp - Rxm) * P.idx + (Ryp - Rym) * P.idy + (Rzp - Rzm) * P.idzf[k];
    if (STORE_R) {
        rnx[c] = Rxp;
        rny[c] = Ryp;
        rnz[c] = Rzp;
    }
}

// ---------------------------------------------------------------- S1: ACDI phi transport
// RHSphi = D(-u_a phibar_a) + Gamma D(Rn);  phi <- phi + dt (g RHS + z RHS_old)   (BASELINE.json:5(i))
// also writes psi = eps ln q of phi_new (N2), the input of k_iface_march (r = sqrt q is recomputed there)
__global__ void __launch_bounds__(256, 5)
k_phi_update(FzP P, const double *__restrict__ phi, const double *__restrict__ u,
                             const double *__restrict__ v, const double *__restrict__ w,
                             const double *__restrict__ divrn, double *__restrict__ hphi,
                             double *__restrict__ phin, double *__restrict__ psi,
                             const double *__restrict__ scal, double dt, double gs, double zs, int keep_h)
{
    FZ_CELL_IJK
    const FzZ z = fz_zn(P, k);
    const unsigned nx = P.nx, sxy = (unsigned)P.sxy;   // 32-bit offsets: N < 2^31 (fizzy_create)
    const unsigned pl = (unsigned)k * sxy, row = pl + nx * j, c = row + i;
    const unsigned xp = row + fz_ip(i, P.nx), xm = row + fz_im(i, P.nx);
    const unsigned yp = pl + nx * fz_ip(j, P.ny) + i, ym = pl + nx * fz_im(j, P.ny) + i;
    const unsigned zp = (unsigned)z.kp * sxy + nx * j + i, zm = (unsigned)z.km * sxy + nx * j + i;
    const double f0 = phi[c];
    const double Fxp = -u[c] * 0.5 * (f0 + phi[xp]), Fxm = -u[xm] * 0.5 * (phi[xm] + f0);
    const double Fyp = -v[c] * 0.5 * (f0 + phi[yp]), Fym = -v[ym] * 0.5 * (phi[ym] + f0);
    const double Fzp = z.gp ? 0.0 : -w[c] * 0.5 * (f0 + phi[zp]);
    const double Fzm = z.gm ? 0.0 : -w[zm] * 0.5 * (phi[zm] + f0);
    const double rhs = (Fxp - Fxm) * P.idx + (Fyp - Fym) * P.idy + (Fzp - Fzm) * P.idzf[k] + scal[1] * divrn[c];
    // stage 0 has zeta = 0: the history is not read (it may hold anything finite; 0 * h == 0)
    const double fn = f0 + dt * (gs * rhs + (zs != 0.0 ? zs * hphi[c] : 0.0));
    phin[c] = fn;
    if (keep_h) hphi[c] = rhs;   // not at stage 2: the next stage has zeta = 0 and never reads it
    psi[c] = fz_psi(P, fn);
}

// ---------------------------------------------------------------- S5 of the previous substep fused with S1
// corrected face velocity  u = u** - (a dt / rho0) d_a p_new  (one spelling for k_correct and k_corr_phi: the value a
// thread forms for a NEIGHBOUR's face is bit for bit the one the neighbour stores)
__device__ __forceinline__ double fz_corr(double us, double coef, double p_hi, double p_lo, double ih)
{
    return us - coef * (p_hi - p_lo) * ih;
}

// After stages 0 and 1 the velocity correction is not launched on its own: the next substep starts with this kernel,
// which forms u, v, w = u** - coef d(p_new) (stores them for S2b, S3) and uses them at once for the phi transport --
// the corrected velocity is written but never read back by S1: -24 B/cell against k_correct + k_phi_update.
// (After stage 2 k_correct runs on its own: Gamma of the next step needs max|u| before its S1, N15.)
// phat != NULL (rho1 != rho2): also p_hat = 2 p_new - p_old (N7).
__global__ void __launch_bounds__(256, 5)
k_corr_phi(FzP P, const double *__restrict__ us, const double *__restrict__ vs,
                           const double *__restrict__ ws, const double *__restrict__ pn,
                           const double *__restrict__ pold, double *__restrict__ phat,
                           double *__restrict__ u, double *__restrict__ v, double *__restrict__ w,
                           const double *__restrict__ phi, const double *__restrict__ divrn,
                           double *__restrict__ hphi, double *__restrict__ phin, double *__restrict__ psi,
                           const double *__restrict__ scal, double coef, double dt, double gs, double zs, int keep_h)
{
    FZ_CELL_IJK
    const FzZ z = fz_zn(P, k);
    const unsigned nx = P.nx, sxy = (unsigned)P.sxy;
    const unsigned pl = (unsigned)k * sxy, row = pl + nx * j, c = row + i;
    const unsigned xp = row + fz_ip(i, P.nx), xm = row + fz_im(i, P.nx);
    const unsigned yp = pl + nx * fz_ip(j, P.ny) + i, ym = pl + nx * fz_im(j, P.ny) + i;
    const unsigned zp = (unsigned)z.kp * sxy + nx * j + i, zm = (unsigned)z.km * sxy + nx * j + i;
    const double p0 = pn[c];
    if (phat) phat[c] = 2.0 * p0 - pold[c];
    // S5 at the cell's own three faces ...
    const double un = fz_corr(us[c], coef, pn[xp], p0, P.idx);
    const double vn = fz_corr(vs[c], coef, pn[yp], p0, P.idy);
    const double wn = k < P.kzf ? fz_corr(ws[c], coef, pn[zp], p0, P.idzc[k]) : 0.0;
    u[c] = un;
    v[c] = vn;
    w[c] = wn;
    // ... and at the three faces below it (stored by the neighbours)
    const double uxm = fz_corr(us[xm], coef, p0, pn[xm], P.idx);
    const double vym = fz_corr(vs[ym], coef, p0, pn[ym], P.idy);
    const double wzm = z.gm ? 0.0 : fz_corr(ws[zm], coef, p0, pn[zm], P.idzc[z.km]);
    // S1 (as k_phi_update)
    const double f0 = phi[c];
    const double Fxp = -un * 0.5 * (f0 + phi[xp]), Fxm = -uxm * 0.5 * (phi[xm] + f0);
    const double Fyp = -vn * 0.5 * (f0 + phi[yp]), Fym = -vym * 0.5 * (phi[ym] + f0);
    const double Fzp = z.gp ? 0.0 : -wn * 0.5 * (f0 + phi[zp]);
    const double Fzm = z.gm ? 0.0 : -wzm * 0.5 * (phi[zm] + f0);
    const double rhs = (Fxp - Fxm) * P.idx + (Fyp - Fym) * P.idy + (Fzp - Fzm) * P.idzf[k] + scal[1] * divrn[c];
    const double fn = f0 + dt * (gs * rhs + (zs != 0.0 ? zs * hphi[c] : 0.0));
    phin[c] = fn;
    if (keep_h) hphi[c] = rhs;
    psi[c] = fz_psi(P, fn);
}

// ---------------------------------------------------------------- S2b: temperature transport (N14)
// RHS_T = D(-u_a Tbar_a) + D(kbar_a d_a T)/(rho cp), properties from phi_new;  k is linear in clip(phi),
// so kbar_a = k2 + (k1-k2) * 0.5 (phic + phic(+1_a)).  32-bit offsets (N < 2^31).  64 registers, four CTAs per SM: all 21
// loads of a thread in flight at once (at 40 registers / six CTAs the kernel waited on serialised loads: 0.52 -> 0.44 ms at
// 512x256x256).
__global__ void __launch_bounds__(256, 4)
k_temp_update(FzP P, const double *__restrict__ T, const double *__restrict__ phi,
              const double *__restrict__ u, const double *__restrict__ v,
              const double *__restrict__ w, double *__restrict__ hT,
              double *__restrict__ Tn, double dt, double gs, double zs, int keep_h)
{
    FZ_CELL_IJK
    const FzZ z = fz_zn(P, k);
    const unsigned nx = P.nx, sxy = (unsigned)P.sxy;
    const unsigned pl = (unsigned)k * sxy, row = pl + nx * j, c = row + i;
    const unsigned xp = row + fz_ip(i, P.nx), xm = row + fz_im(i, P.nx);
    const unsigned yp = pl + nx * fz_ip(j, P.ny) + i, ym = pl + nx * fz_im(j, P.ny) + i;
    const unsigned zp = (unsigned)z.kp * sxy + nx * j + i, zm = (unsigned)z.km * sxy + nx * j + i;
    // face conductivity kbar_a = kmid + 1/4 (k1-k2) (sclip + sclip(+1_a)), fz_sclip = 2 clip - 1 (no comparisons)
    const double qdk = 0.25 * (P.k1 - P.k2), kmid = 0.5 * (P.k1 + P.k2);
    const double t0 = T[c], s0 = fz_sclip(phi[c]);
    const double izf = P.idzf[k], idx = P.idx, idy = P.idy;
    double adv, dif;
    {   // x
        const double tp = T[xp], tm = T[xm];
        const double kp = fma(qdk, s0 + fz_sclip(phi[xp]), kmid), km = fma(qdk, fz_sclip(phi[xm]) + s0, kmid);
        adv = (u[xm] * (tm + t0) - u[c] * (t0 + tp)) * (0.5 * idx);
        dif = (kp * (tp - t0) - km * (t0 - tm)) * (idx * idx);
    }
    {   // y
        const double tp = T[yp], tm = T[ym];
        const double kp = fma(qdk, s0 + fz_sclip(phi[yp]), kmid), km = fma(qdk, fz_sclip(phi[ym]) + s0, kmid);
        adv += (v[ym] * (tm + t0) - v[c] * (t0 + tp)) * (0.5 * idy);
        dif += (kp * (tp - t0) - km * (t0 - tm)) * (idy * idy);
    }
    {   // z: Dirichlet ghosts 2 T_wall - T, no advective flux through a wall face
        const double tp = z.gp ? 2.0 * P.t_top - t0 : T[zp], tm = z.gm ? 2.0 * P.t_bot - t0 : T[zm];
        const double kp = fma(qdk, s0 + fz_sclip(phi[zp]), kmid), km = fma(qdk, fz_sclip(phi[zm]) + s0, kmid);
        const double fp = z.gp ? 0.0 : w[c] * (t0 + tp), fm = z.gm ? 0.0 : w[zm] * (tm + t0);
        adv += (fm - fp) * (0.5 * izf);
        dif += (kp * (tp - t0) * P.idzc[k] - km * (t0 - tm) * P.idzc[k - 1]) * izf;
    }
    const double phc = 0.5 * s0 + 0.5;
    const double rcp = (P.rho2 + P.drho * phc) * (P.cp2 + (P.cp1 - P.cp2) * phc);
    const double rhs = adv + dif * fz_rcp(rcp);
    Tn[c] = t0 + dt * (gs * rhs + (zs != 0.0 ? zs * hT[c] : 0.0));
    if (keep_h) hT[c] = rhs;
}

// ---------------------------------------------------------------- S5: velocity correction
// u = u** - (a dt / rho0) d_a p_new  (the p_hat part of BASELINE.json:5(v) is already in u**)
// phat != NULL (rho1 != rho2): also p_hat = 2 p_new - p_old, the extrapolated pressure of the NEXT substep (N7)
template <bool WITH_MAX>
__global__ void k_correct(FzP P, const double *__restrict__ us, const double *__restrict__ vs,
                          const double *__restrict__ ws, const double *__restrict__ pn,
                          double *__restrict__ u, double *__restrict__ v, double *__restrict__ w,
                          double coef /* a dt / rho0 */, double *umax, const double *__restrict__ pold,
                          double *__restrict__ phat)
{
    FZ_CELL_IJK
    const FzZ z = fz_zn(P, k);
    const unsigned nx = P.nx, sxy = (unsigned)P.sxy;   // 32-bit offsets: N < 2^31 (fizzy_create)
    const unsigned pl = (unsigned)k * sxy, c = pl + nx * j + i;
    const double p0 = pn[c];
    if (phat) phat[c] = 2.0 * p0 - pold[c];
    const double un = fz_corr(us[c], coef, pn[pl + nx * j + fz_ip(i, P.nx)], p0, P.idx);
    const double vn = fz_corr(vs[c], coef, pn[pl + nx * fz_ip(j, P.ny) + i], p0, P.idy);
    double wn = 0.0;
    if (k < P.kzf) wn = fz_corr(ws[c], coef, pn[(unsigned)z.kp * sxy + nx * j + i], p0, P.idzc[k]);
    u[c] = un;
    v[c] = vn;
    w[c] = wn;
    if (WITH_MAX) {
        // block max, then at most one atomic per CTA (and none if the running max is already larger)
        __shared__ double wmax[8];
        double m = fmax(fabs(un), fmax(fabs(vn), fabs(wn)));
        for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
        const int t = threadIdx.x + blockDim.x * threadIdx.y;
        if ((t & 31) == 0) wmax[t >> 5] = m;
        __syncthreads();
        if (t == 0) {
            const int nw = (blockDim.x * blockDim.y + 31) >> 5;
            for (int q = 1; q < nw; ++q) m = fmax(m, wmax[q]);
            if (m > *reinterpret_cast<volatile double *>(umax)) fz_atomic_max_nonneg(umax, m);
        }
    }
}

// ---------------------------------------------------------------- S4', S5': the variable-coefficient path
// rhs = coef D(u*)   (coef = 1/(a dt); the velocity below the first cell of a wall-bounded grid is the wall: 0)
__global__ void k_div_rhs(FzP P, const double *__restrict__ us, const double *__restrict__ vs,
                          const double *__restrict__ ws, double coef, double *__restrict__ rhs)
{
    FZ_CELL_IJK
    const FzZ z = fz_zn(P, k);
    const unsigned nx = P.nx, sxy = (unsigned)P.sxy;
    const unsigned pl = (unsigned)k * sxy, row = pl + nx * j, c = row + i;
    const unsigned xm = row + fz_im(i, P.nx), ym = pl + nx * fz_im(j, P.ny) + i, zm = (unsigned)z.km * sxy + nx * j + i;
    const double wl = z.gm ? 0.0 : ws[zm];
    rhs[c] = coef * ((us[c] - us[xm]) * P.idx + (vs[c] - vs[ym]) * P.idy + (ws[c] - wl) * P.idzf[k]);
}

// u = u* - a dt (1/rho_f) d_a p_new,  rho_f = 1/2 (rho + rho(+1_a)) of phi_new (N11); max|u| at stage 2
template <bool WITH_MAX>
__global__ void k_correct_var(FzP P, const double *__restrict__ us, const double *__restrict__ vs,
                              const double *__restrict__ ws, const double *__restrict__ pn,
                              const double *__restrict__ phi, double *__restrict__ u, double *__restrict__ v,
                              double *__restrict__ w, double adt, double *umax)
{
    FZ_CELL_IJK
    const FzZ z = fz_zn(P, k);
    const unsigned nx = P.nx, sxy = (unsigned)P.sxy;
    const unsigned pl = (unsigned)k * sxy, row = pl + nx * j, c = row + i;
    const unsigned xp = row + fz_ip(i, P.nx), yp = pl + nx * fz_ip(j, P.ny) + i, zp = (unsigned)z.kp * sxy + nx * j + i;
    const double p0 = pn[c], r0 = P.rho2 + P.drho * fz_clip01(phi[c]);
    const double un = us[c] - adt * (pn[xp] - p0) * P.idx / (0.5 * (r0 + P.rho2 + P.drho * fz_clip01(phi[xp])));
    const double vn = vs[c] - adt * (pn[yp] - p0) * P.idy / (0.5 * (r0 + P.rho2 + P.drho * fz_clip01(phi[yp])));
    double wn = 0.0;
    if (k < P.kzf) wn = ws[c] - adt * (pn[zp] - p0) * P.idzc[k] / (0.5 * (r0 + P.rho2 + P.drho * fz_clip01(phi[zp])));
    u[c] = un;
    v[c] = vn;
    w[c] = wn;
    if (WITH_MAX) {
        double m = fmax(fabs(un), fmax(fabs(vn), fabs(wn)));
        for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
        if (((threadIdx.x + blockDim.x * threadIdx.y) & 31) == 0 && m > *reinterpret_cast<volatile double *>(umax))
            fz_atomic_max_nonneg(umax, m);
    }
}

// p_hat = 2p - p_prev (N7) of freshly loaded pressures
__global__ void k_phat(FzP P, const double *__restrict__ p, const double *__restrict__ pp, double *__restrict__ phat)
{
    FZ_CELL_IJK
    const long long c = i + P.nx * (j + (long long)P.ny * k);
    phat[c] = 2.0 * p[c] - pp[c];
}

// zero the top-wall w plane (w[:,:,nz-1] == 0 with walls)
__global__ void k_zero_plane(FzP P, double *w)
{
    const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t < P.sxy) w[(long long)(P.nz - 1) * P.sxy + t] = 0.0;
}
