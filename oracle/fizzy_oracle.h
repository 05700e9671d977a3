/* fizzy_oracle.h -- CPU ORACLE (TEST INFRASTRUCTURE, NOT THE PRODUCT).
 *
 * Plain, slow, fp64 restatement of one low-storage RK3 substep of the one-fluid
 * two-phase solver described in PAPER.md:32 (model) and PAPER.md:36 (discretisation:
 * 2nd-order finite differences, staggered velocity, cell-centred scalars, low-storage
 * three-step Runge-Kutta, pressure-correction with the constant-coefficient splitting
 * and the FFT direct solver), with the formulas (i)-(v) of BASELINE.json:5 and the
 * readings N1..N22 of SURVEY.md section 8(c), which DESIGN.md restates.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * leg may build, load or call this.  It shares no code with the CUDA path.
 *
 * Parity unpinned (any consistent choice passes every check we have; fixed by DESIGN.md):
 *   N6  (which phi feeds S3),
 *   N9  (non-conservative form of the mass-consistent regularisation-flux term;
 *        pinned only by: vanishes for rho1 == rho2, exact for linear velocity),
 *   N14 (non-conservative temperature equation).
 * N7 (pressure extrapolation p_hat = 2p - p_prev and the rotation of p, p_prev) is pinned since round 3 by the
 * closed-form hydrostatic recurrence of tests/test_oracle_step.py.
 *
 * Layout: all field arrays are nx*ny*nz doubles, x fastest: idx = i + nx*(j + ny*k).
 * u[i,j,k] sits on the x-face between cells i and i+1, v on the y-face between j and
 * j+1, w on the z-face between k and k+1 (face zf[k+1]).  With walls w[:,:,nz-1] == 0.
 */
#ifndef FIZZY_ORACLE_H
#define FIZZY_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
    int nx, ny, nz;
    double lx, ly, lz;
    int z_wall;              /* 0: periodic in z, 1: no-slip walls at z=0 and z=lz */
    int has_zf;              /* 0: uniform z, 1: zf[] below is used (walls only)     */
    double rho1, rho2;       /* fluid 1 <-> phi = 1, fluid 2 <-> phi = 0             */
    double mu1, mu2;
    double k1, k2;           /* thermal conductivity */
    double cp1, cp2;         /* specific heat */
    double sigma, eps, delta;
    double gamma_rel, gamma_abs;   /* Gamma = gamma_rel * max|u| + gamma_abs (N15)   */
    double gx, gy, gz;
    double rho_ref, beta, t_ref;
    double fx, fy, fz;       /* uniform body acceleration */
    double a_lin;            /* linear (Lundgren) forcing coefficient (N22) */
    int heat;
    double t_bot, t_top;     /* wall temperatures */
} orc_params;

typedef struct orc_state orc_state;

orc_state *orc_create(const orc_params *prm, const double *zf /* nz+1 or NULL */);
void orc_destroy(orc_state *st);

/* NULL T allowed when heat==0; NULL p_prev => p_prev := p.  Zeroes the RK history. */
void orc_set_fields(orc_state *st, const double *u, const double *v, const double *w,
                    const double *p, const double *phi, const double *T, const double *p_prev);
/* any pointer may be NULL */
void orc_get_fields(const orc_state *st, double *u, double *v, double *w, double *p,
                    double *phi, double *T, double *p_prev);

/* one RK3 substep, stage in {0,1,2}; returns 0 on success */
int orc_substep(orc_state *st, int stage, double dt);

/* solves Lap p = rhs with the state's grid and z boundary condition; gauge: N17 */
void orc_poisson_solve(orc_state *st, const double *rhs, double *p);

/* SURVEY.md 8(f)-4 (the variable-coefficient alternative to the splitting): solver = 1 makes orc_substep solve
 * D((1/rho_f) d p_new) = D(u*)/(a dt) and correct with u = u* - a dt (1/rho_f) d p_new (no p_hat anywhere); plain CG in the
 * dzf-weighted inner product to a relative residual of 1e-14.  orc_varcoef_solve: that solve alone, density from the current
 * phase field; returns the iterations.  Pinned against oracle/varcoef.py (sparse direct) and, for rho1 = rho2, against the
 * splitting itself. */
void orc_set_solver(orc_state *st, int solver);
int orc_varcoef_solve(orc_state *st, const double *rhs, double *p);

double orc_gamma(const orc_state *st);

/* intermediates of the LAST substep (unpadded nx*ny*nz copies). names:
 *  "psi" "nhx" "nhy" "nhz" "Rx" "Ry" "Rz" (R includes Gamma; from phi_new, as used by S3)
 *  "kappa" "rho" "mu" "rhs_phi" "rhs_T" "rhs_u" "rhs_v" "rhs_w"
 *  "ustar" "vstar" "wstar" "poisson_rhs" "p_hat"
 * returns 0 if known, -1 otherwise */
int orc_get_intermediate(const orc_state *st, const char *name, double *out);

/* momentum RHS (S3) of the current state, without touching it: props from current phi */
void orc_momentum_rhs(orc_state *st, double *rhs_u, double *rhs_v, double *rhs_w);
/* phase-field RHS (S1) of the current state with given Gamma */
void orc_phi_rhs(orc_state *st, double gamma, double *rhs_phi);

/* temperature RHS (S2b) of the current state: props from current phi (heat==1 only) */
void orc_temperature_rhs(orc_state *st, double *rhs_T);

/* the oracle's own radix-2 FFT, exposed so a test can pin it against a naive DFT.
 * in-place, n a power of two, sign=-1 forward (e^{-2 pi i jk/n}), +1 backward (no scaling) */
void orc_fft(int n, double *re, double *im, int sign);

/* run-time diagnostics of the current state: out[8] = volume of fluid 1,
 * kinetic energy, max|u|, max|D(u)|, interfacial area, mean temperature, Nusselt number at the
 * bottom and at the top wall (see fizzy_oracle.c) */
void orc_diagnostics(const orc_state *st, double *out);

/* stable time step of the current fields, reading N16: cfl * min of the advective,
 * viscous, capillary, ACDI and thermal limits (see fizzy_oracle.c) */
double orc_stable_dt(const orc_state *st, double cfl);

int orc_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
