/* fizzy_oracle.c -- CPU ORACLE (TEST INFRASTRUCTURE, NOT THE PRODUCT).  See fizzy_oracle.h.
 *
 * Style: every field lives in a ghost-padded array (halo H=2 in x, y and z).  After a
 * field is computed on the interior its ghosts are filled by the boundary rule of that
 * field (periodic in x,y; periodic or wall rule in z, SURVEY.md 8(c) "Walls").  All
 * stencils are then plain loops over the interior with +-1 index offsets, written in the
 * order and notation of SURVEY.md 8(c) / DESIGN.md "The method".  No blocking, no fusion.
 * OpenMP is used on the outermost (k) loop only.
 *
 * Discrete operators (a = axis):
 *   face average   fbar_a  = 0.5*(f + f(+1_a))
 *   face gradient  d_a f   = (f(+1_a) - f)/hc_a      hc = dx, dy, dzc[k]
 *   divergence     D(F)    = sum_a (F_a - F_a(-1_a))/hf_a   hf = dx, dy, dzf[k]
 */
#include "fizzy_oracle.h"
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define H 2

/* ghost rules in z when z_wall == 1 */
enum { BC_EVEN = 0,   /* cell-centred, mirror:            f(-1-m) =  f(m)            */
       BC_ODD = 1,    /* cell-centred, antisymmetric:     f(-1-m) = -f(m)  (no-slip) */
       BC_TWALL = 2,  /* cell-centred, Dirichlet:         f(-1-m) = 2 Twall - f(m)   */
       BC_WFACE = 3   /* on z-faces: wall faces k=-1 and k=nz-1 are 0, odd beyond    */ };

struct orc_state {
    orc_params P;
    int nx, ny, nz;
    size_t N, NP;          /* interior / padded sizes */
    size_t PX, PY, PZ;
    double dx, dy;
    double *dzf_, *dzc_;   /* with ghost entries; use DZF(k), DZC(k) */
    double gamma;
    int fields_set;
    int solver;            /* 0: constant-coefficient splitting (S4, S5 of BASELINE.json:5); 1: variable-coefficient problem */
    /* prognostic fields (padded) */
    double *u, *v, *w, *p, *pp, *phi, *T;
    /* RK history (padded, interior used) */
    double *hphi, *hT, *hu, *hv, *hw;
    /* intermediates (padded) */
    double *psi, *nhx, *nhy, *nhz, *Rx, *Ry, *Rz, *kappa, *rho, *mu, *kth, *cp;
    double *Fx, *Fy, *Fz;              /* face-flux scratch */
    double *rphi, *rT, *ru, *rv, *rw;  /* RHS of the last substep */
    double *us, *vs, *ws;              /* u*, v*, w* */
    double *prhs, *phat, *pnew;
    double complex *cw;                /* N complex, Poisson work array (unpadded) */
};

#define IDX(i, j, k) ((size_t)((i) + H) + st->PX * ((size_t)((j) + H) + st->PY * (size_t)((k) + H)))
#define DZF(k) (st->dzf_[(k) + H])   /* cell height, k = -H .. nz+H-1              */
#define DZC(k) (st->dzc_[(k) + H])   /* centre spacing at face k, k = -H .. nz+H-2 */

static double *palloc(const orc_state *st) { return (double *)calloc(st->NP, sizeof(double)); }

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------ ghosts */
static void fill_ghosts(const orc_state *st, double *f, int bc, double tb, double tt)
{
    const int nx = st->nx, ny = st->ny, nz = st->nz;
    /* z first (interior i,j), then y (all k), then x (all j,k): corners get filled */
    if (!st->P.z_wall) {
        for (int g = 1; g <= H; ++g)
            for (int j = 0; j < ny; ++j)
                for (int i = 0; i < nx; ++i) {
                    f[IDX(i, j, -g)] = f[IDX(i, j, nz - g)];
                    f[IDX(i, j, nz - 1 + g)] = f[IDX(i, j, g - 1)];
                }
    } else if (bc == BC_WFACE) {
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                f[IDX(i, j, -1)] = 0.0;        /* bottom wall face */
                f[IDX(i, j, nz - 1)] = 0.0;    /* top wall face    */
                f[IDX(i, j, -2)] = -f[IDX(i, j, 0)];
                f[IDX(i, j, nz)] = -f[IDX(i, j, nz - 2)];
                f[IDX(i, j, nz + 1)] = -f[IDX(i, j, nz - 3)];
            }
    } else {
        for (int g = 1; g <= H; ++g)
            for (int j = 0; j < ny; ++j)
                for (int i = 0; i < nx; ++i) {
                    double lo = f[IDX(i, j, g - 1)], hi = f[IDX(i, j, nz - g)];
                    if (bc == BC_EVEN) { /* mirror */
                    } else if (bc == BC_ODD) {
                        lo = -lo; hi = -hi;
                    } else { /* BC_TWALL */
                        lo = 2.0 * tb - lo; hi = 2.0 * tt - hi;
                    }
                    f[IDX(i, j, -g)] = lo;
                    f[IDX(i, j, nz - 1 + g)] = hi;
                }
    }
    for (int k = -H; k < nz + H; ++k)
        for (int g = 1; g <= H; ++g)
            for (int i = 0; i < nx; ++i) {
                f[IDX(i, -g, k)] = f[IDX(i, ny - g, k)];
                f[IDX(i, ny - 1 + g, k)] = f[IDX(i, g - 1, k)];
            }
    for (int k = -H; k < nz + H; ++k)
        for (int j = -H; j < ny + H; ++j)
            for (int g = 1; g <= H; ++g) {
                f[IDX(-g, j, k)] = f[IDX(nx - g, j, k)];
                f[IDX(nx - 1 + g, j, k)] = f[IDX(g - 1, j, k)];
            }
}

static void put_interior(const orc_state *st, double *dst_padded, const double *src)
{
    for (int k = 0; k < st->nz; ++k)
        for (int j = 0; j < st->ny; ++j)
            for (int i = 0; i < st->nx; ++i)
                dst_padded[IDX(i, j, k)] = src[(size_t)i + (size_t)st->nx * ((size_t)j + (size_t)st->ny * k)];
}

static void get_interior(const orc_state *st, const double *src_padded, double *dst)
{
    for (int k = 0; k < st->nz; ++k)
        for (int j = 0; j < st->ny; ++j)
            for (int i = 0; i < st->nx; ++i)
                dst[(size_t)i + (size_t)st->nx * ((size_t)j + (size_t)st->ny * k)] = src_padded[IDX(i, j, k)];
}

/* number of z-faces that carry an unknown w: all nz if periodic, nz-1 with walls */
static int nzw(const orc_state *st) { return st->P.z_wall ? st->nz - 1 : st->nz; }

/* ------------------------------------------------------------------ create */
orc_state *orc_create(const orc_params *prm, const double *zf)
{
    orc_state *st = (orc_state *)calloc(1, sizeof(orc_state));
    st->P = *prm;
    const int nx = st->nx = prm->nx, ny = st->ny = prm->ny, nz = st->nz = prm->nz;
    st->N = (size_t)nx * ny * nz;
    st->PX = nx + 2 * H; st->PY = ny + 2 * H; st->PZ = nz + 2 * H;
    st->NP = st->PX * st->PY * st->PZ;
    st->dx = prm->lx / nx;
    st->dy = prm->ly / ny;
    st->dzf_ = (double *)calloc(nz + 2 * H, sizeof(double));
    st->dzc_ = (double *)calloc(nz + 2 * H, sizeof(double));
    /* cell heights */
    for (int k = 0; k < nz; ++k)
        DZF(k) = (prm->has_zf && zf) ? zf[k + 1] - zf[k] : prm->lz / nz;
    for (int g = 1; g <= H; ++g) {
        if (prm->z_wall) { /* ghost cells mirror the interior cells */
            DZF(-g) = DZF(g - 1);
            DZF(nz - 1 + g) = DZF(nz - g);
        } else {
            DZF(-g) = DZF(nz - g);
            DZF(nz - 1 + g) = DZF(g - 1);
        }
    }
    /* centre-to-centre spacing at face k (centres are face midpoints, N10) */
    for (int k = -H; k < nz + H - 1; ++k) DZC(k) = 0.5 * (DZF(k) + DZF(k + 1));

    double **all[] = {&st->u, &st->v, &st->w, &st->p, &st->pp, &st->phi, &st->hphi, &st->hu, &st->hv,
                      &st->hw, &st->psi, &st->nhx, &st->nhy, &st->nhz, &st->Rx, &st->Ry, &st->Rz,
                      &st->kappa, &st->rho, &st->mu, &st->Fx, &st->Fy, &st->Fz, &st->rphi, &st->ru,
                      &st->rv, &st->rw, &st->us, &st->vs, &st->ws, &st->prhs, &st->phat, &st->pnew};
    for (size_t a = 0; a < sizeof(all) / sizeof(all[0]); ++a) *all[a] = palloc(st);
    if (prm->heat) {
        st->T = palloc(st); st->hT = palloc(st); st->rT = palloc(st);
        st->kth = palloc(st); st->cp = palloc(st);
    }
    st->cw = (double complex *)calloc(st->N, sizeof(double complex));
    return st;
}

void orc_destroy(orc_state *st)
{
    if (!st) return;
    double *all[] = {st->u, st->v, st->w, st->p, st->pp, st->phi, st->T, st->hphi, st->hT, st->hu,
                     st->hv, st->hw, st->psi, st->nhx, st->nhy, st->nhz, st->Rx, st->Ry, st->Rz,
                     st->kappa, st->rho, st->mu, st->kth, st->cp, st->Fx, st->Fy, st->Fz, st->rphi,
                     st->rT, st->ru, st->rv, st->rw, st->us, st->vs, st->ws, st->prhs, st->phat,
                     st->pnew, st->dzf_, st->dzc_};
    for (size_t a = 0; a < sizeof(all) / sizeof(all[0]); ++a) free(all[a]);
    free(st->cw);
    free(st);
}

static void fill_velocity_ghosts(const orc_state *st, double *u, double *v, double *w)
{
    fill_ghosts(st, u, BC_ODD, 0, 0);   /* no-slip: tangential velocity antisymmetric */
    fill_ghosts(st, v, BC_ODD, 0, 0);
    fill_ghosts(st, w, BC_WFACE, 0, 0); /* impermeable: wall faces are zero           */
}

void orc_set_fields(orc_state *st, const double *u, const double *v, const double *w, const double *p,
                    const double *phi, const double *T, const double *p_prev)
{
    put_interior(st, st->u, u); put_interior(st, st->v, v); put_interior(st, st->w, w);
    put_interior(st, st->p, p); put_interior(st, st->phi, phi);
    put_interior(st, st->pp, p_prev ? p_prev : p);
    if (st->P.heat && T) put_interior(st, st->T, T);
    fill_velocity_ghosts(st, st->u, st->v, st->w);
    fill_ghosts(st, st->p, BC_EVEN, 0, 0);
    fill_ghosts(st, st->pp, BC_EVEN, 0, 0);
    fill_ghosts(st, st->phi, BC_EVEN, 0, 0);
    if (st->P.heat) fill_ghosts(st, st->T, BC_TWALL, st->P.t_bot, st->P.t_top);
    memset(st->hphi, 0, st->NP * sizeof(double));
    memset(st->hu, 0, st->NP * sizeof(double));
    memset(st->hv, 0, st->NP * sizeof(double));
    memset(st->hw, 0, st->NP * sizeof(double));
    if (st->P.heat) memset(st->hT, 0, st->NP * sizeof(double));
    st->gamma = st->P.gamma_abs;
    st->fields_set = 1;
}

void orc_get_fields(const orc_state *st, double *u, double *v, double *w, double *p, double *phi,
                    double *T, double *p_prev)
{
    if (u) get_interior(st, st->u, u);
    if (v) get_interior(st, st->v, v);
    if (w) get_interior(st, st->w, w);
    if (p) get_interior(st, st->p, p);
    if (phi) get_interior(st, st->phi, phi);
    if (T && st->P.heat) get_interior(st, st->T, T);
    if (p_prev) get_interior(st, st->pp, p_prev);
}

double orc_gamma(const orc_state *st) { return st->gamma; }

/* ------------------------------------------------------------------ S0: Gamma (N15)
 * Gamma = gamma_rel * max over all faces of max(|u|,|v|,|w|) + gamma_abs, at stage 0. */
static void update_gamma(orc_state *st)
{
    double m = 0.0;
    for (int k = 0; k < st->nz; ++k)
        for (int j = 0; j < st->ny; ++j)
            for (int i = 0; i < st->nx; ++i) {
                size_t c = IDX(i, j, k);
                m = fmax(m, fabs(st->u[c]));
                m = fmax(m, fabs(st->v[c]));
                m = fmax(m, fabs(st->w[c]));
            }
    st->gamma = st->P.gamma_rel * m + st->P.gamma_abs;
}

/* ------------------------------------------------------------------ interface quantities
 * From a phase field phi (ghosts filled) compute, in this order (BASELINE.json:5(i), N2-N5):
 *   psi  = eps * ln((phic + delta)/(1 - phic + delta)),  phic = clip(phi, 0, 1)
 *   G_a  = (psi(+1_a) - psi(-1_a)) / (hc_a + hc_a(-1_a));  nhat = G / max(|G|, 1e-30)
 *   nf_a = 0.5*(nhat_a + nhat_a(+1_a))
 *   R_a  = Gamma * [ eps * d_a phi - 0.25*(1 - tanh^2((psi + psi(+1_a))/(4 eps))) * nf_a ]
 *   kappa = -D(nf)
 * With walls: psi mirror, nhat_x, nhat_y mirror, nhat_z antisymmetric (so nf_z = 0 on
 * wall faces), R_z = 0 on wall faces. */
static void interface_quantities(orc_state *st, const double *phi, double gamma)
{
    const int nx = st->nx, ny = st->ny, nz = st->nz;
    const double eps = st->P.eps, delta = st->P.delta, dx = st->dx, dy = st->dy;
    double *psi = st->psi, *nhx = st->nhx, *nhy = st->nhy, *nhz = st->nhz;

#pragma omp parallel for
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                double phic = fmin(fmax(phi[IDX(i, j, k)], 0.0), 1.0);
                psi[IDX(i, j, k)] = eps * log((phic + delta) / (1.0 - phic + delta));
            }
    fill_ghosts(st, psi, BC_EVEN, 0, 0);

#pragma omp parallel for
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                double Gx = (psi[IDX(i + 1, j, k)] - psi[IDX(i - 1, j, k)]) / (dx + dx);
                double Gy = (psi[IDX(i, j + 1, k)] - psi[IDX(i, j - 1, k)]) / (dy + dy);
                double Gz = (psi[IDX(i, j, k + 1)] - psi[IDX(i, j, k - 1)]) / (DZC(k) + DZC(k - 1));
                double mag = sqrt(Gx * Gx + Gy * Gy + Gz * Gz);
                double den = fmax(mag, 1e-30);
                nhx[IDX(i, j, k)] = Gx / den;
                nhy[IDX(i, j, k)] = Gy / den;
                nhz[IDX(i, j, k)] = Gz / den;
            }
    fill_ghosts(st, nhx, BC_EVEN, 0, 0);
    fill_ghosts(st, nhy, BC_EVEN, 0, 0);
    fill_ghosts(st, nhz, BC_ODD, 0, 0);

    const int kzf = nzw(st);
#pragma omp parallel for
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t c = IDX(i, j, k), xp = IDX(i + 1, j, k), yp = IDX(i, j + 1, k), zp = IDX(i, j, k + 1);
                double t, sharp;
                t = tanh((psi[c] + psi[xp]) / (4.0 * eps));
                sharp = 0.25 * (1.0 - t * t) * 0.5 * (nhx[c] + nhx[xp]);
                st->Rx[c] = gamma * (eps * (phi[xp] - phi[c]) / dx - sharp);
                t = tanh((psi[c] + psi[yp]) / (4.0 * eps));
                sharp = 0.25 * (1.0 - t * t) * 0.5 * (nhy[c] + nhy[yp]);
                st->Ry[c] = gamma * (eps * (phi[yp] - phi[c]) / dy - sharp);
                if (k < kzf) {
                    t = tanh((psi[c] + psi[zp]) / (4.0 * eps));
                    sharp = 0.25 * (1.0 - t * t) * 0.5 * (nhz[c] + nhz[zp]);
                    st->Rz[c] = gamma * (eps * (phi[zp] - phi[c]) / DZC(k) - sharp);
                } else {
                    st->Rz[c] = 0.0; /* top wall face */
                }
            }
    fill_ghosts(st, st->Rx, BC_EVEN, 0, 0);
    fill_ghosts(st, st->Ry, BC_EVEN, 0, 0);
    fill_ghosts(st, st->Rz, BC_WFACE, 0, 0);

    /* curvature kappa = -D(nf), nf_z = 0 on wall faces through the odd ghost of nhz */
#pragma omp parallel for
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                double nfx_p = 0.5 * (nhx[IDX(i, j, k)] + nhx[IDX(i + 1, j, k)]);
                double nfx_m = 0.5 * (nhx[IDX(i - 1, j, k)] + nhx[IDX(i, j, k)]);
                double nfy_p = 0.5 * (nhy[IDX(i, j, k)] + nhy[IDX(i, j + 1, k)]);
                double nfy_m = 0.5 * (nhy[IDX(i, j - 1, k)] + nhy[IDX(i, j, k)]);
                double nfz_p = 0.5 * (nhz[IDX(i, j, k)] + nhz[IDX(i, j, k + 1)]);
                double nfz_m = 0.5 * (nhz[IDX(i, j, k - 1)] + nhz[IDX(i, j, k)]);
                st->kappa[IDX(i, j, k)] =
                    -((nfx_p - nfx_m) / dx + (nfy_p - nfy_m) / dy + (nfz_p - nfz_m) / DZF(k));
            }
    fill_ghosts(st, st->kappa, BC_EVEN, 0, 0);
}

/* ------------------------------------------------------------------ S1: phase-field RHS
 * RHSphi = D(F),  F_a = -u_a * phibar_a + R_a      (BASELINE.json:5(i)) */
static void phi_rhs(orc_state *st, const double *phi, double gamma, double *rhs)
{
    const int nx = st->nx, ny = st->ny, nz = st->nz;
    const double dx = st->dx, dy = st->dy;
    interface_quantities(st, phi, gamma);
#pragma omp parallel for
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t c = IDX(i, j, k);
                st->Fx[c] = -st->u[c] * 0.5 * (phi[c] + phi[IDX(i + 1, j, k)]) + st->Rx[c];
                st->Fy[c] = -st->v[c] * 0.5 * (phi[c] + phi[IDX(i, j + 1, k)]) + st->Ry[c];
                st->Fz[c] = -st->w[c] * 0.5 * (phi[c] + phi[IDX(i, j, k + 1)]) + st->Rz[c];
            }
    fill_ghosts(st, st->Fx, BC_EVEN, 0, 0);
    fill_ghosts(st, st->Fy, BC_EVEN, 0, 0);
    fill_ghosts(st, st->Fz, BC_WFACE, 0, 0); /* no flux through walls */
#pragma omp parallel for
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t c = IDX(i, j, k);
                rhs[c] = (st->Fx[c] - st->Fx[IDX(i - 1, j, k)]) / dx +
                         (st->Fy[c] - st->Fy[IDX(i, j - 1, k)]) / dy +
                         (st->Fz[c] - st->Fz[IDX(i, j, k - 1)]) / DZF(k);
            }
}

void orc_phi_rhs(orc_state *st, double gamma, double *rhs_phi)
{
    phi_rhs(st, st->phi, gamma, st->rphi);
    get_interior(st, st->rphi, rhs_phi);
}

/* ------------------------------------------------------------------ S2: property map
 * q(phi) = q2 + (q1 - q2) * clip(phi,0,1)   ("linearly mapped"; N2) */
static void property_map(orc_state *st, const double *phi)
{
    const orc_params *P = &st->P;
#pragma omp parallel for
    for (int k = 0; k < st->nz; ++k)
        for (int j = 0; j < st->ny; ++j)
            for (int i = 0; i < st->nx; ++i) {
                size_t c = IDX(i, j, k);
                double phic = fmin(fmax(phi[c], 0.0), 1.0);
                st->rho[c] = P->rho2 + (P->rho1 - P->rho2) * phic;
                st->mu[c] = P->mu2 + (P->mu1 - P->mu2) * phic;
                if (P->heat) {
                    st->kth[c] = P->k2 + (P->k1 - P->k2) * phic;
                    st->cp[c] = P->cp2 + (P->cp1 - P->cp2) * phic;
                }
            }
    fill_ghosts(st, st->rho, BC_EVEN, 0, 0);
    fill_ghosts(st, st->mu, BC_EVEN, 0, 0);
    if (P->heat) {
        fill_ghosts(st, st->kth, BC_EVEN, 0, 0);
        fill_ghosts(st, st->cp, BC_EVEN, 0, 0);
    }
}

/* ------------------------------------------------------------------ S2b: temperature RHS
 * RHS_T = D(-u_a Tbar_a) + D(kbar_a d_a T)/(rho cp)   (N14), wall ghost T = 2 Twall - T */
static void temperature_rhs(orc_state *st, double *rhs)
{
    const int nx = st->nx, ny = st->ny, nz = st->nz;
    const double dx = st->dx, dy = st->dy;
    const double *T = st->T, *kth = st->kth;
    double *Ax = st->Fx, *Ay = st->Fy, *Az = st->Fz; /* advective face fluxes */
#pragma omp parallel for
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t c = IDX(i, j, k);
                Ax[c] = -st->u[c] * 0.5 * (T[c] + T[IDX(i + 1, j, k)]);
                Ay[c] = -st->v[c] * 0.5 * (T[c] + T[IDX(i, j + 1, k)]);
                Az[c] = -st->w[c] * 0.5 * (T[c] + T[IDX(i, j, k + 1)]);
            }
    fill_ghosts(st, Ax, BC_EVEN, 0, 0);
    fill_ghosts(st, Ay, BC_EVEN, 0, 0);
    fill_ghosts(st, Az, BC_WFACE, 0, 0);
#pragma omp parallel for
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t c = IDX(i, j, k);
                size_t xm = IDX(i - 1, j, k), xp = IDX(i + 1, j, k);
                size_t ym = IDX(i, j - 1, k), yp = IDX(i, j + 1, k);
                size_t zm = IDX(i, j, k - 1), zp = IDX(i, j, k + 1);
                double adv = (Ax[c] - Ax[xm]) / dx + (Ay[c] - Ay[ym]) / dy + (Az[c] - Az[zm]) / DZF(k);
                /* conductive face fluxes q_a = kbar_a * d_a T (wall faces use the ghost T) */
                double qxp = 0.5 * (kth[c] + kth[xp]) * (T[xp] - T[c]) / dx;
                double qxm = 0.5 * (kth[xm] + kth[c]) * (T[c] - T[xm]) / dx;
                double qyp = 0.5 * (kth[c] + kth[yp]) * (T[yp] - T[c]) / dy;
                double qym = 0.5 * (kth[ym] + kth[c]) * (T[c] - T[ym]) / dy;
                double qzp = 0.5 * (kth[c] + kth[zp]) * (T[zp] - T[c]) / DZC(k);
                double qzm = 0.5 * (kth[zm] + kth[c]) * (T[c] - T[zm]) / DZC(k - 1);
                double dif = (qxp - qxm) / dx + (qyp - qym) / dy + (qzp - qzm) / DZF(k);
                rhs[c] = adv + dif / (st->rho[c] * st->cp[c]);
            }
}

/* ------------------------------------------------------------------ S3: momentum RHS
 * For component a at its face:
 *   RHS_a = A_a + (V_a + S_a + M_a)/rho_f + B_a
 * Needs: u,v,w (ghosts), phi_new (ghosts), rho, mu, kappa, R (from phi_new), T_new. */
static void momentum_rhs(orc_state *st, const double *phi, double *ru, double *rv, double *rw)
{
    const int nx = st->nx, ny = st->ny, nz = st->nz;
    const double dx = st->dx, dy = st->dy;
    const orc_params *P = &st->P;
    const double *u = st->u, *v = st->v, *w = st->w, *mu = st->mu, *rho = st->rho;
    const double *kap = st->kappa, *Rx = st->Rx, *Ry = st->Ry, *Rz = st->Rz, *T = st->T;
    const double drho = P->rho1 - P->rho2;
    const int kzf = nzw(st);

#pragma omp parallel for
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                const size_t c = IDX(i, j, k);
#define AT(di, dj, dk) IDX(i + (di), j + (dj), k + (dk))
                /* ================= x component, face (i+1/2, j, k) ================= */
                {
                    /* advection: -d_x(uc uc) - d_y(E_xy) - d_z(E_xz) */
                    double uc_p = 0.5 * (u[AT(1, 0, 0)] + u[c]);   /* centre of cell i+1 */
                    double uc_m = 0.5 * (u[c] + u[AT(-1, 0, 0)]);  /* centre of cell i   */
                    double Exy_p = 0.5 * (v[c] + v[AT(1, 0, 0)]) * 0.5 * (u[c] + u[AT(0, 1, 0)]);
                    double Exy_m = 0.5 * (v[AT(0, -1, 0)] + v[AT(1, -1, 0)]) * 0.5 * (u[AT(0, -1, 0)] + u[c]);
                    double Exz_p = 0.5 * (w[c] + w[AT(1, 0, 0)]) * 0.5 * (u[c] + u[AT(0, 0, 1)]);
                    double Exz_m = 0.5 * (w[AT(0, 0, -1)] + w[AT(1, 0, -1)]) * 0.5 * (u[AT(0, 0, -1)] + u[c]);
                    double A = -(uc_p * uc_p - uc_m * uc_m) / dx - (Exy_p - Exy_m) / dy - (Exz_p - Exz_m) / DZF(k);
                    /* viscous: d_x(2 mu d_x u) + d_y(tau_xy) + d_z(tau_xz) */
                    double nrm_p = 2.0 * mu[AT(1, 0, 0)] * (u[AT(1, 0, 0)] - u[c]) / dx;
                    double nrm_m = 2.0 * mu[c] * (u[c] - u[AT(-1, 0, 0)]) / dx;
                    double mue;
                    mue = 0.25 * (mu[c] + mu[AT(1, 0, 0)] + mu[AT(0, 1, 0)] + mu[AT(1, 1, 0)]);
                    double txy_p = mue * ((u[AT(0, 1, 0)] - u[c]) / dy + (v[AT(1, 0, 0)] - v[c]) / dx);
                    mue = 0.25 * (mu[AT(0, -1, 0)] + mu[AT(1, -1, 0)] + mu[c] + mu[AT(1, 0, 0)]);
                    double txy_m = mue * ((u[c] - u[AT(0, -1, 0)]) / dy + (v[AT(1, -1, 0)] - v[AT(0, -1, 0)]) / dx);
                    mue = 0.25 * (mu[c] + mu[AT(1, 0, 0)] + mu[AT(0, 0, 1)] + mu[AT(1, 0, 1)]);
                    double txz_p = mue * ((u[AT(0, 0, 1)] - u[c]) / DZC(k) + (w[AT(1, 0, 0)] - w[c]) / dx);
                    mue = 0.25 * (mu[AT(0, 0, -1)] + mu[AT(1, 0, -1)] + mu[c] + mu[AT(1, 0, 0)]);
                    double txz_m = mue * ((u[c] - u[AT(0, 0, -1)]) / DZC(k - 1) + (w[AT(1, 0, -1)] - w[AT(0, 0, -1)]) / dx);
                    double V = (nrm_p - nrm_m) / dx + (txy_p - txy_m) / dy + (txz_p - txz_m) / DZF(k);
                    /* surface tension (CSF): sigma * kappabar * d_x phi */
                    double S = P->sigma * 0.5 * (kap[c] + kap[AT(1, 0, 0)]) * (phi[AT(1, 0, 0)] - phi[c]) / dx;
                    /* mass-consistent regularisation-flux term (N9): (rho1-rho2)(R.grad)u */
                    double Rty = 0.25 * (Ry[c] + Ry[AT(1, 0, 0)] + Ry[AT(0, -1, 0)] + Ry[AT(1, -1, 0)]);
                    double Rtz = 0.25 * (Rz[c] + Rz[AT(1, 0, 0)] + Rz[AT(0, 0, -1)] + Rz[AT(1, 0, -1)]);
                    double M = drho * (Rx[c] * (u[AT(1, 0, 0)] - u[AT(-1, 0, 0)]) / (dx + dx) +
                                       Rty * (u[AT(0, 1, 0)] - u[AT(0, -1, 0)]) / (dy + dy) +
                                       Rtz * (u[AT(0, 0, 1)] - u[AT(0, 0, -1)]) / (DZC(k) + DZC(k - 1)));
                    double rhof = 0.5 * (rho[c] + rho[AT(1, 0, 0)]);
                    double B = P->gx * (1.0 - P->rho_ref / rhof) + P->fx + P->a_lin * u[c];
                    if (P->heat) B -= P->gx * P->beta * (0.5 * (T[c] + T[AT(1, 0, 0)]) - P->t_ref);
                    ru[c] = A + (V + S + M) / rhof + B;
                }
                /* ================= y component, face (i, j+1/2, k) ================= */
                {
                    double vc_p = 0.5 * (v[AT(0, 1, 0)] + v[c]);
                    double vc_m = 0.5 * (v[c] + v[AT(0, -1, 0)]);
                    double Eyx_p = 0.5 * (u[c] + u[AT(0, 1, 0)]) * 0.5 * (v[c] + v[AT(1, 0, 0)]);
                    double Eyx_m = 0.5 * (u[AT(-1, 0, 0)] + u[AT(-1, 1, 0)]) * 0.5 * (v[AT(-1, 0, 0)] + v[c]);
                    double Eyz_p = 0.5 * (w[c] + w[AT(0, 1, 0)]) * 0.5 * (v[c] + v[AT(0, 0, 1)]);
                    double Eyz_m = 0.5 * (w[AT(0, 0, -1)] + w[AT(0, 1, -1)]) * 0.5 * (v[AT(0, 0, -1)] + v[c]);
                    double A = -(vc_p * vc_p - vc_m * vc_m) / dy - (Eyx_p - Eyx_m) / dx - (Eyz_p - Eyz_m) / DZF(k);
                    double nrm_p = 2.0 * mu[AT(0, 1, 0)] * (v[AT(0, 1, 0)] - v[c]) / dy;
                    double nrm_m = 2.0 * mu[c] * (v[c] - v[AT(0, -1, 0)]) / dy;
                    double mue;
                    mue = 0.25 * (mu[c] + mu[AT(0, 1, 0)] + mu[AT(1, 0, 0)] + mu[AT(1, 1, 0)]);
                    double tyx_p = mue * ((v[AT(1, 0, 0)] - v[c]) / dx + (u[AT(0, 1, 0)] - u[c]) / dy);
                    mue = 0.25 * (mu[AT(-1, 0, 0)] + mu[AT(-1, 1, 0)] + mu[c] + mu[AT(0, 1, 0)]);
                    double tyx_m = mue * ((v[c] - v[AT(-1, 0, 0)]) / dx + (u[AT(-1, 1, 0)] - u[AT(-1, 0, 0)]) / dy);
                    mue = 0.25 * (mu[c] + mu[AT(0, 1, 0)] + mu[AT(0, 0, 1)] + mu[AT(0, 1, 1)]);
                    double tyz_p = mue * ((v[AT(0, 0, 1)] - v[c]) / DZC(k) + (w[AT(0, 1, 0)] - w[c]) / dy);
                    mue = 0.25 * (mu[AT(0, 0, -1)] + mu[AT(0, 1, -1)] + mu[c] + mu[AT(0, 1, 0)]);
                    double tyz_m = mue * ((v[c] - v[AT(0, 0, -1)]) / DZC(k - 1) + (w[AT(0, 1, -1)] - w[AT(0, 0, -1)]) / dy);
                    double V = (nrm_p - nrm_m) / dy + (tyx_p - tyx_m) / dx + (tyz_p - tyz_m) / DZF(k);
                    double S = P->sigma * 0.5 * (kap[c] + kap[AT(0, 1, 0)]) * (phi[AT(0, 1, 0)] - phi[c]) / dy;
                    double Rtx = 0.25 * (Rx[c] + Rx[AT(0, 1, 0)] + Rx[AT(-1, 0, 0)] + Rx[AT(-1, 1, 0)]);
                    double Rtz = 0.25 * (Rz[c] + Rz[AT(0, 1, 0)] + Rz[AT(0, 0, -1)] + Rz[AT(0, 1, -1)]);
                    double M = drho * (Ry[c] * (v[AT(0, 1, 0)] - v[AT(0, -1, 0)]) / (dy + dy) +
                                       Rtx * (v[AT(1, 0, 0)] - v[AT(-1, 0, 0)]) / (dx + dx) +
                                       Rtz * (v[AT(0, 0, 1)] - v[AT(0, 0, -1)]) / (DZC(k) + DZC(k - 1)));
                    double rhof = 0.5 * (rho[c] + rho[AT(0, 1, 0)]);
                    double B = P->gy * (1.0 - P->rho_ref / rhof) + P->fy + P->a_lin * v[c];
                    if (P->heat) B -= P->gy * P->beta * (0.5 * (T[c] + T[AT(0, 1, 0)]) - P->t_ref);
                    rv[c] = A + (V + S + M) / rhof + B;
                }
                /* ================= z component, face (i, j, k+1/2) ================= */
                if (k < kzf) {
                    double wc_p = 0.5 * (w[AT(0, 0, 1)] + w[c]);   /* centre of cell k+1 */
                    double wc_m = 0.5 * (w[c] + w[AT(0, 0, -1)]);  /* centre of cell k   */
                    double Ezx_p = 0.5 * (u[c] + u[AT(0, 0, 1)]) * 0.5 * (w[c] + w[AT(1, 0, 0)]);
                    double Ezx_m = 0.5 * (u[AT(-1, 0, 0)] + u[AT(-1, 0, 1)]) * 0.5 * (w[AT(-1, 0, 0)] + w[c]);
                    double Ezy_p = 0.5 * (v[c] + v[AT(0, 0, 1)]) * 0.5 * (w[c] + w[AT(0, 1, 0)]);
                    double Ezy_m = 0.5 * (v[AT(0, -1, 0)] + v[AT(0, -1, 1)]) * 0.5 * (w[AT(0, -1, 0)] + w[c]);
                    double A = -(wc_p * wc_p - wc_m * wc_m) / DZC(k) - (Ezx_p - Ezx_m) / dx - (Ezy_p - Ezy_m) / dy;
                    double nrm_p = 2.0 * mu[AT(0, 0, 1)] * (w[AT(0, 0, 1)] - w[c]) / DZF(k + 1);
                    double nrm_m = 2.0 * mu[c] * (w[c] - w[AT(0, 0, -1)]) / DZF(k);
                    double mue;
                    mue = 0.25 * (mu[c] + mu[AT(0, 0, 1)] + mu[AT(1, 0, 0)] + mu[AT(1, 0, 1)]);
                    double tzx_p = mue * ((w[AT(1, 0, 0)] - w[c]) / dx + (u[AT(0, 0, 1)] - u[c]) / DZC(k));
                    mue = 0.25 * (mu[AT(-1, 0, 0)] + mu[AT(-1, 0, 1)] + mu[c] + mu[AT(0, 0, 1)]);
                    double tzx_m = mue * ((w[c] - w[AT(-1, 0, 0)]) / dx + (u[AT(-1, 0, 1)] - u[AT(-1, 0, 0)]) / DZC(k));
                    mue = 0.25 * (mu[c] + mu[AT(0, 0, 1)] + mu[AT(0, 1, 0)] + mu[AT(0, 1, 1)]);
                    double tzy_p = mue * ((w[AT(0, 1, 0)] - w[c]) / dy + (v[AT(0, 0, 1)] - v[c]) / DZC(k));
                    mue = 0.25 * (mu[AT(0, -1, 0)] + mu[AT(0, -1, 1)] + mu[c] + mu[AT(0, 0, 1)]);
                    double tzy_m = mue * ((w[c] - w[AT(0, -1, 0)]) / dy + (v[AT(0, -1, 1)] - v[AT(0, -1, 0)]) / DZC(k));
                    double V = (nrm_p - nrm_m) / DZC(k) + (tzx_p - tzx_m) / dx + (tzy_p - tzy_m) / dy;
                    double S = P->sigma * 0.5 * (kap[c] + kap[AT(0, 0, 1)]) * (phi[AT(0, 0, 1)] - phi[c]) / DZC(k);
                    double Rtx = 0.25 * (Rx[c] + Rx[AT(0, 0, 1)] + Rx[AT(-1, 0, 0)] + Rx[AT(-1, 0, 1)]);
                    double Rty = 0.25 * (Ry[c] + Ry[AT(0, 0, 1)] + Ry[AT(0, -1, 0)] + Ry[AT(0, -1, 1)]);
                    double M = drho * (Rz[c] * (w[AT(0, 0, 1)] - w[AT(0, 0, -1)]) / (DZF(k + 1) + DZF(k)) +
                                       Rtx * (w[AT(1, 0, 0)] - w[AT(-1, 0, 0)]) / (dx + dx) +
                                       Rty * (w[AT(0, 1, 0)] - w[AT(0, -1, 0)]) / (dy + dy));
                    double rhof = 0.5 * (rho[c] + rho[AT(0, 0, 1)]);
                    double B = P->gz * (1.0 - P->rho_ref / rhof) + P->fz + P->a_lin * w[c];
                    if (P->heat) B -= P->gz * P->beta * (0.5 * (T[c] + T[AT(0, 0, 1)]) - P->t_ref);
                    rw[c] = A + (V + S + M) / rhof + B;
                } else {
                    rw[c] = 0.0; /* top wall face: w stays zero */
                }
#undef AT
            }
}

void orc_momentum_rhs(orc_state *st, double *rhs_u, double *rhs_v, double *rhs_w)
{
    interface_quantities(st, st->phi, st->gamma);
    property_map(st, st->phi);
    momentum_rhs(st, st->phi, st->ru, st->rv, st->rw);
    get_interior(st, st->ru, rhs_u);
    get_interior(st, st->rv, rhs_v);
    get_interior(st, st->rw, rhs_w);
}

void orc_temperature_rhs(orc_state *st, double *rhs_T)
{
    if (!st->P.heat) return;
    property_map(st, st->phi);
    temperature_rhs(st, st->rT);
    get_interior(st, st->rT, rhs_T);
}

/* ------------------------------------------------------------------ FFT (own radix-2)
 * Iterative decimation-in-time Cooley-Tukey with bit reversal; twiddles from cos/sin of
 * the exact angle for each butterfly (no recurrences), so accuracy is ~log2(n) ulp. */
static void fft_c(int n, double complex *x, int sign)
{
    for (int i = 1, j = 0; i < n; ++i) { /* bit reversal permutation */
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) { double complex t = x[i]; x[i] = x[j]; x[j] = t; }
    }
    for (int len = 2; len <= n; len <<= 1) {
        const double ang = sign * 2.0 * M_PI / len;
        for (int s = 0; s < n; s += len)
            for (int q = 0; q < len / 2; ++q) {
                double complex wq = cos(ang * q) + I * sin(ang * q);
                double complex a = x[s + q], b = x[s + q + len / 2] * wq;
                x[s + q] = a + b;
                x[s + q + len / 2] = a - b;
            }
    }
}

void orc_fft(int n, double *re, double *im, int sign)
{
    double complex *x = (double complex *)malloc(sizeof(double complex) * n);
    for (int i = 0; i < n; ++i) x[i] = re[i] + I * im[i];
    fft_c(n, x, sign);
    for (int i = 0; i < n; ++i) { re[i] = creal(x[i]); im[i] = cimag(x[i]); }
    free(x);
}

/* ------------------------------------------------------------------ tridiagonal solvers
 * Thomas algorithm, real matrix (a,b,c), complex right-hand side d (overwritten by x). */
static void thomas(int n, const double *a, const double *b, const double *c, double complex *d,
                   double *cprime)
{
    double den = b[0];
    cprime[0] = c[0] / den;
    d[0] = d[0] / den;
    for (int k = 1; k < n; ++k) {
        den = b[k] - a[k] * cprime[k - 1];
        cprime[k] = c[k] / den;
        d[k] = (d[k] - a[k] * d[k - 1]) / den;
    }
    for (int k = n - 2; k >= 0; --k) d[k] -= cprime[k] * d[k + 1];
}

/* periodic (cyclic) tridiagonal: row 0 couples to x[n-1] through a[0], row n-1 couples to
 * x[0] through c[n-1].  Sherman-Morrison on top of Thomas (textbook). */
static void cyclic_thomas(int n, const double *a, const double *b, const double *c, double complex *d,
                          double *bb, double complex *q, double *cprime)
{
    const double gam = -b[0];
    for (int k = 0; k < n; ++k) { bb[k] = b[k]; q[k] = 0.0; }
    bb[0] = b[0] - gam;
    bb[n - 1] = b[n - 1] - a[0] * c[n - 1] / gam;
    q[0] = gam;
    q[n - 1] = c[n - 1];
    thomas(n, a, bb, c, d, cprime);
    thomas(n, a, bb, c, q, cprime);
    double complex fact = (d[0] + a[0] * d[n - 1] / gam) / (1.0 + q[0] + a[0] * q[n - 1] / gam);
    for (int k = 0; k < n; ++k) d[k] -= fact * q[k];
}

/* ------------------------------------------------------------------ S4: Poisson solve
 * L p = b with L = D(d .) (7-point).  DFT in x and y diagonalises the periodic directions:
 *   lam_x(l) = -4 sin^2(pi l/nx)/dx^2,  lam_y(m) = -4 sin^2(pi m/ny)/dy^2
 * and for each (l,m) a tridiagonal system in z remains:
 *   a_k x_{k-1} + (b_k + lam_x + lam_y) x_k + c_k x_{k+1} = bhat_k,
 *   a_k = 1/(dzf[k] dzc[k-1]),  c_k = 1/(dzf[k] dzc[k]),  b_k = -(a_k + c_k);
 * walls (Neumann): a_0 = 0, c_{nz-1} = 0 (the wall-face gradient is zero);
 * periodic z: cyclic.  Mode (0,0) is singular: its last row is replaced by x_{nz-1} = 0 and
 * afterwards the dzf-weighted mean of p is removed (N17). */
static void poisson_solve_unpadded(orc_state *st, const double *rhs, double *pout)
{
    const int nx = st->nx, ny = st->ny, nz = st->nz;
    double complex *cw = st->cw;
    const size_t N = st->N;
    for (size_t c = 0; c < N; ++c) cw[c] = rhs[c];

    /* forward DFT along x, then along y */
#pragma omp parallel
    {
        double complex *line = (double complex *)malloc(sizeof(double complex) * (nx > ny ? nx : ny));
#pragma omp for
        for (int k = 0; k < nz; ++k) {
            for (int j = 0; j < ny; ++j) fft_c(nx, cw + (size_t)nx * (j + (size_t)ny * k), -1);
            for (int i = 0; i < nx; ++i) {
                for (int j = 0; j < ny; ++j) line[j] = cw[i + (size_t)nx * (j + (size_t)ny * k)];
                fft_c(ny, line, -1);
                for (int j = 0; j < ny; ++j) cw[i + (size_t)nx * (j + (size_t)ny * k)] = line[j];
            }
        }
        free(line);
    }

    /* tridiagonal coefficients in z */
    double *a = (double *)malloc(sizeof(double) * nz), *b = (double *)malloc(sizeof(double) * nz),
           *c = (double *)malloc(sizeof(double) * nz);
    for (int k = 0; k < nz; ++k) {
        a[k] = 1.0 / (DZF(k) * DZC(k - 1));
        c[k] = 1.0 / (DZF(k) * DZC(k));
        if (st->P.z_wall && k == 0) a[k] = 0.0;
        if (st->P.z_wall && k == nz - 1) c[k] = 0.0;
        b[k] = -(a[k] + c[k]);
    }
#pragma omp parallel
    {
        double complex *d = (double complex *)malloc(sizeof(double complex) * nz);
        double complex *q = (double complex *)malloc(sizeof(double complex) * nz);
        double *bl = (double *)malloc(sizeof(double) * nz), *bb = (double *)malloc(sizeof(double) * nz),
               *cpr = (double *)malloc(sizeof(double) * nz);
#pragma omp for
        for (int m = 0; m < ny; ++m)
            for (int l = 0; l < nx; ++l) {
                double sx = sin(M_PI * l / nx), sy = sin(M_PI * m / ny);
                double lam = -4.0 * sx * sx / (st->dx * st->dx) - 4.0 * sy * sy / (st->dy * st->dy);
                for (int k = 0; k < nz; ++k) {
                    d[k] = cw[l + (size_t)nx * (m + (size_t)ny * k)];
                    bl[k] = b[k] + lam;
                }
                if (l == 0 && m == 0) {
                    /* singular mode: x_{nz-1} = 0, rows 0..nz-2 lose their coupling to it */
                    d[nz - 1] = 0.0;
                    thomas(nz - 1, a, bl, c, d, cpr); /* a[0] x_{nz-1} = 0, c[nz-2] x_{nz-1} = 0 */
                } else if (st->P.z_wall) {
                    thomas(nz, a, bl, c, d, cpr);
                } else {
                    cyclic_thomas(nz, a, bl, c, d, bb, q, cpr);
                }
                for (int k = 0; k < nz; ++k) cw[l + (size_t)nx * (m + (size_t)ny * k)] = d[k];
            }
        free(d); free(q); free(bl); free(bb); free(cpr);
    }
    free(a); free(b); free(c);

    /* inverse DFT along y, then x, scale 1/(nx ny) */
#pragma omp parallel
    {
        double complex *line = (double complex *)malloc(sizeof(double complex) * (nx > ny ? nx : ny));
#pragma omp for
        for (int k = 0; k < nz; ++k) {
            for (int i = 0; i < nx; ++i) {
                for (int j = 0; j < ny; ++j) line[j] = cw[i + (size_t)nx * (j + (size_t)ny * k)];
                fft_c(ny, line, +1);
                for (int j = 0; j < ny; ++j) cw[i + (size_t)nx * (j + (size_t)ny * k)] = line[j];
            }
            for (int j = 0; j < ny; ++j) fft_c(nx, cw + (size_t)nx * (j + (size_t)ny * k), +1);
        }
        free(line);
    }
    const double scale = 1.0 / ((double)nx * (double)ny);
    /* gauge: remove the dzf-weighted mean */
    double wsum = 0.0, vol = 0.0;
    for (int k = 0; k < nz; ++k) {
        double s = 0.0;
        for (size_t c2 = 0; c2 < (size_t)nx * ny; ++c2) s += creal(cw[(size_t)nx * ny * k + c2]) * scale;
        wsum += s * DZF(k);
        vol += (double)nx * ny * DZF(k);
    }
    const double mean = wsum / vol;
    for (int k = 0; k < nz; ++k)
        for (size_t c2 = 0; c2 < (size_t)nx * ny; ++c2)
            pout[(size_t)nx * ny * k + c2] = creal(cw[(size_t)nx * ny * k + c2]) * scale - mean;
}

void orc_poisson_solve(orc_state *st, const double *rhs, double *p) { poisson_solve_unpadded(st, rhs, p); }

/* ------------------------------------------------------------------ the substep
 * Low-storage RK3 (N1, Wray): f <- f + dt*(gamma_s RHS + zeta_s RHS_old), alpha = gamma+zeta */
/* ------------------------------------------------------------------------------------------------
 * SURVEY.md 8(f)-4, PAPER.md:36 ("the conventional variable-coefficients problem"): instead of the splitting,
 *     D( (1/rho_f) d_a p ) = rhs,   rho_f = 1/2 (rho + rho(+1_a))  (N11),
 * solved here by plain conjugate gradients (no preconditioner) in the dzf-weighted inner product, in which the
 * operator is self-adjoint; the dzf-weighted mean of rhs is removed first (the operator is singular) and the
 * solution returned with zero dzf-weighted mean (the gauge of N17).  An iteration, so the oracle follows it step by
 * step; what it converges to is pinned against the sparse direct solve of oracle/varcoef.py. */
static void varcoef_apply(orc_state *st, double *x, double *out)
{
    const int nx = st->nx, ny = st->ny, nz = st->nz, kzf = nzw(st);
    const double dx = st->dx, dy = st->dy;
    const double *rho = st->rho;
    fill_ghosts(st, x, BC_EVEN, 0, 0);
#pragma omp parallel for
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t c = IDX(i, j, k);
                st->Fx[c] = (x[IDX(i + 1, j, k)] - x[c]) / dx / (0.5 * (rho[c] + rho[IDX(i + 1, j, k)]));
                st->Fy[c] = (x[IDX(i, j + 1, k)] - x[c]) / dy / (0.5 * (rho[c] + rho[IDX(i, j + 1, k)]));
                st->Fz[c] = (k < kzf) ? (x[IDX(i, j, k + 1)] - x[c]) / DZC(k) / (0.5 * (rho[c] + rho[IDX(i, j, k + 1)])) : 0.0;
            }
    fill_ghosts(st, st->Fx, BC_EVEN, 0, 0);
    fill_ghosts(st, st->Fy, BC_EVEN, 0, 0);
    fill_ghosts(st, st->Fz, BC_WFACE, 0, 0);
#pragma omp parallel for
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t c = IDX(i, j, k);
                out[c] = (st->Fx[c] - st->Fx[IDX(i - 1, j, k)]) / dx + (st->Fy[c] - st->Fy[IDX(i, j - 1, k)]) / dy +
                         (st->Fz[c] - st->Fz[IDX(i, j, k - 1)]) / DZF(k);
            }
}

static double wdot(const orc_state *st, const double *a, const double *b)
{
    double s = 0.0;
    for (int k = 0; k < st->nz; ++k) {
        double sk = 0.0;
        for (int j = 0; j < st->ny; ++j)
            for (int i = 0; i < st->nx; ++i) sk += a[IDX(i, j, k)] * (b ? b[IDX(i, j, k)] : 1.0);
        s += DZF(k) * sk;
    }
    return s;
}

/* b (padded, interior used; overwritten by the final residual), x (padded): x = solution with zero weighted mean */
static int varcoef_solve(orc_state *st, double *b, double *x)
{
    const int nx = st->nx, ny = st->ny, nz = st->nz;
    double *d = palloc(st), *q = palloc(st);
    double V = 0.0;
    for (int k = 0; k < nz; ++k) V += DZF(k) * nx * ny;
    /* remove the weighted mean of the right-hand side; x = 0; r = b; d = r */
    double mb = 0.0;
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) mb += DZF(k) * b[IDX(i, j, k)];
    mb /= V;
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t c = IDX(i, j, k);
                b[c] -= mb; x[c] = 0.0; d[c] = b[c];
            }
    const double bb = wdot(st, b, b);
    double rr = bb;
    int it = 0;
    const int itmax = 200000;
    while (bb > 0.0 && rr > 1e-28 * bb && it < itmax) {
        varcoef_apply(st, d, q);
        const double alpha = rr / wdot(st, d, q);
#pragma omp parallel for
        for (int k = 0; k < nz; ++k)
            for (int j = 0; j < ny; ++j)
                for (int i = 0; i < nx; ++i) {
                    size_t c = IDX(i, j, k);
                    x[c] += alpha * d[c];
                    b[c] -= alpha * q[c];
                }
        const double rn = wdot(st, b, b);
        const double beta = rn / rr;
#pragma omp parallel for
        for (int k = 0; k < nz; ++k)
            for (int j = 0; j < ny; ++j)
                for (int i = 0; i < nx; ++i) {
                    size_t c = IDX(i, j, k);
                    d[c] = b[c] + beta * d[c];
                }
        rr = rn;
        ++it;
    }
    double mx = 0.0;
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) mx += DZF(k) * x[IDX(i, j, k)];
    mx /= V;
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) x[IDX(i, j, k)] -= mx;
    free(d); free(q);
    return it;
}

void orc_set_solver(orc_state *st, int solver) { st->solver = solver ? 1 : 0; }

/* rhs, p: N interior doubles; density from the CURRENT phase field */
int orc_varcoef_solve(orc_state *st, const double *rhs, double *p)
{
    double *b = palloc(st), *x = palloc(st);
    property_map(st, st->phi);
    put_interior(st, b, rhs);
    const int it = varcoef_solve(st, b, x);
    get_interior(st, x, p);
    free(b); free(x);
    return it;
}

static const double RK_GAMMA[3] = {8.0 / 15.0, 5.0 / 12.0, 3.0 / 4.0};
static const double RK_ZETA[3] = {0.0, -17.0 / 60.0, -5.0 / 12.0};

int orc_substep(orc_state *st, int stage, double dt)
{
    if (!st->fields_set || stage < 0 || stage > 2 || !(dt > 0.0)) return -1;
    const int nx = st->nx, ny = st->ny, nz = st->nz;
    const double dx = st->dx, dy = st->dy;
    const double gs = RK_GAMMA[stage], zs = RK_ZETA[stage], as = gs + zs;
    const orc_params *P = &st->P;
    const int kzf = nzw(st);

    /* S0 */
    if (stage == 0) update_gamma(st);

    /* S1: phi <- phi + dt*(gs RHSphi + zs RHSphi_old); RHSphi_old <- RHSphi */
    phi_rhs(st, st->phi, st->gamma, st->rphi);
#pragma omp parallel for
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t c = IDX(i, j, k);
                st->phi[c] = st->phi[c] + dt * (gs * st->rphi[c] + zs * st->hphi[c]);
                st->hphi[c] = st->rphi[c];
            }
    fill_ghosts(st, st->phi, BC_EVEN, 0, 0);

    /* S2: properties from phi_new; and (N6) interface quantities of phi_new for S3 */
    property_map(st, st->phi);
    interface_quantities(st, st->phi, st->gamma);

    /* S2b: temperature with the stage-start velocity and the new properties */
    if (P->heat) {
        temperature_rhs(st, st->rT);
#pragma omp parallel for
        for (int k = 0; k < nz; ++k)
            for (int j = 0; j < ny; ++j)
                for (int i = 0; i < nx; ++i) {
                    size_t c = IDX(i, j, k);
                    st->T[c] = st->T[c] + dt * (gs * st->rT[c] + zs * st->hT[c]);
                    st->hT[c] = st->rT[c];
                }
        fill_ghosts(st, st->T, BC_TWALL, P->t_bot, P->t_top);
    }

    /* S3: predictor, no pressure term (N8) */
    momentum_rhs(st, st->phi, st->ru, st->rv, st->rw);
#pragma omp parallel for
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t c = IDX(i, j, k);
                st->us[c] = st->u[c] + dt * (gs * st->ru[c] + zs * st->hu[c]);
                st->vs[c] = st->v[c] + dt * (gs * st->rv[c] + zs * st->hv[c]);
                st->ws[c] = (k < kzf) ? st->w[c] + dt * (gs * st->rw[c] + zs * st->hw[c]) : 0.0;
                st->hu[c] = st->ru[c];
                st->hv[c] = st->rv[c];
                st->hw[c] = st->rw[c];
            }
    fill_velocity_ghosts(st, st->us, st->vs, st->ws);

    if (st->solver == 1) {
        /* S4', S5': D((1/rho_f) d p_new) = D(u*)/(as dt);  u = u* - as dt (1/rho_f) d p_new */
        const double *rho = st->rho;
#pragma omp parallel for
        for (int k = 0; k < nz; ++k)
            for (int j = 0; j < ny; ++j)
                for (int i = 0; i < nx; ++i) {
                    size_t c = IDX(i, j, k);
                    st->prhs[c] = ((st->us[c] - st->us[IDX(i - 1, j, k)]) / dx + (st->vs[c] - st->vs[IDX(i, j - 1, k)]) / dy +
                                   (st->ws[c] - st->ws[IDX(i, j, k - 1)]) / DZF(k)) / (as * dt);
                }
        varcoef_solve(st, st->prhs, st->pnew);
        fill_ghosts(st, st->pnew, BC_EVEN, 0, 0);
        const double *pn = st->pnew;
#pragma omp parallel for
        for (int k = 0; k < nz; ++k)
            for (int j = 0; j < ny; ++j)
                for (int i = 0; i < nx; ++i) {
                    size_t c = IDX(i, j, k), xp = IDX(i + 1, j, k), yp = IDX(i, j + 1, k), zp = IDX(i, j, k + 1);
                    st->u[c] = st->us[c] - as * dt * (pn[xp] - pn[c]) / dx / (0.5 * (rho[c] + rho[xp]));
                    st->v[c] = st->vs[c] - as * dt * (pn[yp] - pn[c]) / dy / (0.5 * (rho[c] + rho[yp]));
                    st->w[c] = (k < kzf) ? st->ws[c] - as * dt * (pn[zp] - pn[c]) / DZC(k) / (0.5 * (rho[c] + rho[zp])) : 0.0;
                }
        fill_velocity_ghosts(st, st->u, st->v, st->w);
        memcpy(st->pp, st->p, st->NP * sizeof(double));
        memcpy(st->p, st->pnew, st->NP * sizeof(double));
        return 0;
    }

    /* S4: p_hat = 2p - p_prev (N7);  b = D((1 - rho0/rho_f) d p_hat) + rho0/(as dt) D(u*) */
    const double rho0 = fmin(P->rho1, P->rho2);
#pragma omp parallel for
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t c = IDX(i, j, k);
                st->phat[c] = 2.0 * st->p[c] - st->pp[c];
            }
    fill_ghosts(st, st->phat, BC_EVEN, 0, 0);
    {
        const double *rho = st->rho, *ph = st->phat;
#pragma omp parallel for
        for (int k = 0; k < nz; ++k)
            for (int j = 0; j < ny; ++j)
                for (int i = 0; i < nx; ++i) {
                    size_t c = IDX(i, j, k);
                    double rf;
                    rf = 0.5 * (rho[c] + rho[IDX(i + 1, j, k)]);
                    st->Fx[c] = (1.0 - rho0 / rf) * (ph[IDX(i + 1, j, k)] - ph[c]) / dx;
                    rf = 0.5 * (rho[c] + rho[IDX(i, j + 1, k)]);
                    st->Fy[c] = (1.0 - rho0 / rf) * (ph[IDX(i, j + 1, k)] - ph[c]) / dy;
                    rf = 0.5 * (rho[c] + rho[IDX(i, j, k + 1)]);
                    st->Fz[c] = (k < kzf) ? (1.0 - rho0 / rf) * (ph[IDX(i, j, k + 1)] - ph[c]) / DZC(k) : 0.0;
                }
        fill_ghosts(st, st->Fx, BC_EVEN, 0, 0);
        fill_ghosts(st, st->Fy, BC_EVEN, 0, 0);
        fill_ghosts(st, st->Fz, BC_WFACE, 0, 0);
#pragma omp parallel for
        for (int k = 0; k < nz; ++k)
            for (int j = 0; j < ny; ++j)
                for (int i = 0; i < nx; ++i) {
                    size_t c = IDX(i, j, k), xm = IDX(i - 1, j, k), ym = IDX(i, j - 1, k), zm = IDX(i, j, k - 1);
                    double div_split = (st->Fx[c] - st->Fx[xm]) / dx + (st->Fy[c] - st->Fy[ym]) / dy +
                                       (st->Fz[c] - st->Fz[zm]) / DZF(k);
                    double div_us = (st->us[c] - st->us[xm]) / dx + (st->vs[c] - st->vs[ym]) / dy +
                                    (st->ws[c] - st->ws[zm]) / DZF(k);
                    st->prhs[c] = div_split + rho0 / (as * dt) * div_us;
                }
    }
    {
        double *b = (double *)malloc(sizeof(double) * st->N), *x = (double *)malloc(sizeof(double) * st->N);
        get_interior(st, st->prhs, b);
        poisson_solve_unpadded(st, b, x);
        put_interior(st, st->pnew, x);
        free(b); free(x);
    }
    fill_ghosts(st, st->pnew, BC_EVEN, 0, 0);

    /* S5: u = u* - as dt [ (1/rho0) d p_new + (1/rho_f - 1/rho0) d p_hat ];  rotate pressures */
    {
        const double *rho = st->rho, *ph = st->phat, *pn = st->pnew;
#pragma omp parallel for
        for (int k = 0; k < nz; ++k)
            for (int j = 0; j < ny; ++j)
                for (int i = 0; i < nx; ++i) {
                    size_t c = IDX(i, j, k), xp = IDX(i + 1, j, k), yp = IDX(i, j + 1, k), zp = IDX(i, j, k + 1);
                    double rf;
                    rf = 0.5 * (rho[c] + rho[xp]);
                    st->u[c] = st->us[c] - as * dt * ((1.0 / rho0) * (pn[xp] - pn[c]) / dx +
                                                       (1.0 / rf - 1.0 / rho0) * (ph[xp] - ph[c]) / dx);
                    rf = 0.5 * (rho[c] + rho[yp]);
                    st->v[c] = st->vs[c] - as * dt * ((1.0 / rho0) * (pn[yp] - pn[c]) / dy +
                                                       (1.0 / rf - 1.0 / rho0) * (ph[yp] - ph[c]) / dy);
                    if (k < kzf) {
                        rf = 0.5 * (rho[c] + rho[zp]);
                        st->w[c] = st->ws[c] - as * dt * ((1.0 / rho0) * (pn[zp] - pn[c]) / DZC(k) +
                                                           (1.0 / rf - 1.0 / rho0) * (ph[zp] - ph[c]) / DZC(k));
                    } else {
                        st->w[c] = 0.0;
                    }
                }
    }
    fill_velocity_ghosts(st, st->u, st->v, st->w);
    memcpy(st->pp, st->p, st->NP * sizeof(double));
    memcpy(st->p, st->pnew, st->NP * sizeof(double));
    return 0;
}

int orc_get_intermediate(const orc_state *st, const char *name, double *out)
{
    struct { const char *n; const double *p; } tab[] = {
        {"psi", st->psi}, {"nhx", st->nhx}, {"nhy", st->nhy}, {"nhz", st->nhz}, {"Rx", st->Rx},
        {"Ry", st->Ry}, {"Rz", st->Rz}, {"kappa", st->kappa}, {"rho", st->rho}, {"mu", st->mu},
        {"rhs_phi", st->rphi}, {"rhs_T", st->rT}, {"rhs_u", st->ru}, {"rhs_v", st->rv},
        {"rhs_w", st->rw}, {"ustar", st->us}, {"vstar", st->vs}, {"wstar", st->ws},
        {"poisson_rhs", st->prhs}, {"p_hat", st->phat}};
    for (size_t a = 0; a < sizeof(tab) / sizeof(tab[0]); ++a)
        if (strcmp(tab[a].n, name) == 0 && tab[a].p) {
            get_interior(st, tab[a].p, out);
            return 0;
        }
    return -1;
}

/* ------------------------------------------------------------------ run-time diagnostics
 * (definitions in DESIGN.md section 10).  dV = dx dy dzf[k].
 *   out[0] = sum phi dV                                  (volume of fluid 1)
 *   out[1] = 1/2 sum rho(phi) (uc^2 + vc^2 + wc^2) dV,   uc = (u + u(-1_x))/2 etc. (cell-centred)
 *   out[2] = max over faces of max(|u|, |v|, |w|)
 *   out[3] = max |D(u)|
 *   out[4] = sum |grad phi| dV, central differences (phi(+1_a) - phi(-1_a))/(hc_a + hc_a(-1_a))
 *            (interfacial area of a diffuse interface)
 *   out[5] = sum T dV / sum dV   (0 if heat is off)
 *   out[6], out[7] = Nusselt number at the bottom / top wall (heat on, walls, t_bot != t_top; else 0):
 *            Nu = <-dT/dz>_wall * lz / (t_bot - t_top), the wall gradient taken through the Dirichlet
 *            ghost T(-1) = 2 T_wall - T(0) at distance dzf[0]  (SURVEY.md 8(c) "Walls")
 * Ghosts of u, v, w, phi, T are up to date after orc_set_fields / orc_substep. */
void orc_diagnostics(const orc_state *st, double *out)
{
    const int nx = st->nx, ny = st->ny, nz = st->nz;
    const double dx = st->dx, dy = st->dy;
    double vol1 = 0.0, ke = 0.0, umax = 0.0, dmax = 0.0, area = 0.0, tsum = 0.0, vsum = 0.0;
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                const size_t c = IDX(i, j, k);
                const double dV = dx * dy * DZF(k);
                const double phc = fmin(fmax(st->phi[c], 0.0), 1.0);
                const double rho = st->P.rho2 + (st->P.rho1 - st->P.rho2) * phc;
                const double uc = 0.5 * (st->u[c] + st->u[IDX(i - 1, j, k)]);
                const double vc = 0.5 * (st->v[c] + st->v[IDX(i, j - 1, k)]);
                const double wc = 0.5 * (st->w[c] + st->w[IDX(i, j, k - 1)]);
                const double div = (st->u[c] - st->u[IDX(i - 1, j, k)]) / dx + (st->v[c] - st->v[IDX(i, j - 1, k)]) / dy +
                                   (st->w[c] - st->w[IDX(i, j, k - 1)]) / DZF(k);
                const double gx = (st->phi[IDX(i + 1, j, k)] - st->phi[IDX(i - 1, j, k)]) / (2.0 * dx);
                const double gy = (st->phi[IDX(i, j + 1, k)] - st->phi[IDX(i, j - 1, k)]) / (2.0 * dy);
                const double gz = (st->phi[IDX(i, j, k + 1)] - st->phi[IDX(i, j, k - 1)]) / (DZC(k) + DZC(k - 1));
                vol1 += st->phi[c] * dV;
                ke += 0.5 * rho * (uc * uc + vc * vc + wc * wc) * dV;
                umax = fmax(umax, fmax(fabs(st->u[c]), fmax(fabs(st->v[c]), fabs(st->w[c]))));
                dmax = fmax(dmax, fabs(div));
                area += sqrt(gx * gx + gy * gy + gz * gz) * dV;
                vsum += dV;
                if (st->P.heat) tsum += st->T[c] * dV;
            }
    out[0] = vol1; out[1] = ke; out[2] = umax; out[3] = dmax; out[4] = area;
    out[5] = st->P.heat ? tsum / vsum : 0.0;
    out[6] = out[7] = 0.0;
    if (st->P.heat && st->P.z_wall && st->P.t_bot != st->P.t_top) {
        double gb = 0.0, gt = 0.0;   /* sum over the wall of -dT/dz */
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                gb += -(st->T[IDX(i, j, 0)] - st->T[IDX(i, j, -1)]) / DZC(-1);
                gt += -(st->T[IDX(i, j, nz)] - st->T[IDX(i, j, nz - 1)]) / DZC(nz - 1);
            }
        const double scale = st->P.lz / (st->P.t_bot - st->P.t_top) / ((double)nx * ny);
        out[6] = gb * scale;
        out[7] = gt * scale;
    }
}

/* ------------------------------------------------------------------ stable time step (N16)
 * dt = cfl * min(dt_adv, dt_visc, dt_sigma, dt_acdi, dt_heat) of the CURRENT fields:
 *   dt_adv   = 1 / max over cells of (|u|/dx + |v|/dy + |w|/dzf[k])   (face values of the same index)
 *   dt_visc  = 1 / (2 nu_max S),   nu_max = max(mu1/rho1, mu2/rho2),  S = 1/dx^2 + 1/dy^2 + 1/dzmin^2
 *   dt_sigma = sqrt((rho1 + rho2) dmin^3 / (4 pi sigma)),             dmin = min(dx, dy, dzmin)
 *   dt_acdi  = 1 / (2 Gamma eps S),  Gamma = gamma_rel * max(|u|,|v|,|w|) + gamma_abs   (N15)
 *   dt_heat  = 1 / (2 a_max S),    a_max = max(k1/(rho1 cp1), k2/(rho2 cp2))            (heat on)
 * a limit whose denominator vanishes is left out; returns 0 if every limit is left out. */
double orc_stable_dt(const orc_state *st, double cfl)
{
    const int nx = st->nx, ny = st->ny, nz = st->nz;
    const orc_params *P = &st->P;
    double adv = 0.0, umax = 0.0, dzmin = DZF(0);
    for (int k = 0; k < nz; ++k) {
        dzmin = fmin(dzmin, DZF(k));
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                const size_t c = IDX(i, j, k);
                adv = fmax(adv, fabs(st->u[c]) / st->dx + fabs(st->v[c]) / st->dy + fabs(st->w[c]) / DZF(k));
                umax = fmax(umax, fmax(fabs(st->u[c]), fmax(fabs(st->v[c]), fabs(st->w[c]))));
            }
    }
    const double S = 1.0 / (st->dx * st->dx) + 1.0 / (st->dy * st->dy) + 1.0 / (dzmin * dzmin);
    const double dmin = fmin(st->dx, fmin(st->dy, dzmin));
    const double gam = P->gamma_rel * umax + P->gamma_abs;
    const double nu = fmax(P->mu1 / P->rho1, P->mu2 / P->rho2);
    double lim = INFINITY;
    if (adv > 0.0) lim = fmin(lim, 1.0 / adv);
    if (nu > 0.0) lim = fmin(lim, 1.0 / (2.0 * nu * S));
    if (P->sigma > 0.0) lim = fmin(lim, sqrt((P->rho1 + P->rho2) * dmin * dmin * dmin / (4.0 * M_PI * P->sigma)));
    if (gam > 0.0) lim = fmin(lim, 1.0 / (2.0 * gam * P->eps * S));
    if (P->heat) lim = fmin(lim, 1.0 / (2.0 * fmax(P->k1 / (P->rho1 * P->cp1), P->k2 / (P->rho2 * P->cp2)) * S));
    return isinf(lim) ? 0.0 : cfl * lim;
}
