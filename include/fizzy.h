/* fizzy.h -- C ABI of libfizzy.so: one low-storage RK3 substep of the CaNS-Fizzy one-fluid
 * two-phase solver (arXiv 2502.04189) on one NVIDIA B200 (sm_100a), fp64.
 *
 * What the library computes (passages: /root/reference/PAPER.md, cited PAPER.md:<line>;
 * formulas (i)-(v) of BASELINE.json:5 `north_star`; discrete readings N1..N22 in DESIGN.md):
 *   PAPER.md:32 (section 2)  one-fluid model: incompressible Navier-Stokes + heat transport +
 *                            ACDI phase-field transport; properties mapped linearly over phi;
 *                            CSF surface tension.
 *   PAPER.md:36 (section 3)  2nd-order finite differences, staggered velocity / cell-centred
 *                            scalars; low-storage three-step Runge-Kutta; pressure correction with
 *                            the Dong-Shen / Dodd-Ferrante splitting -> constant-coefficient
 *                            Poisson equation solved by the FFT direct solver of CaNS; mass-
 *                            momentum consistent regularisation flux in the momentum equation.
 *
 * Layout.  Every field is nx*ny*nz contiguous doubles, x fastest: idx = i + nx*(j + ny*k).
 * u[i,j,k] sits on the x-face between cells i and i+1, v on the y-face between j and j+1,
 * w on the z-face zf[k+1] between cells k and k+1.  x and y are periodic.  z is periodic
 * (z_wall = 0) or bounded by no-slip walls (z_wall = 1; then w[:,:,nz-1] == 0 always).
 * Fluid 1 <-> phi = 1 (dispersed), fluid 2 <-> phi = 0 (carrier).
 *
 * Pointers.  Field pointers given to fizzy_set_fields / fizzy_get_fields / fizzy_poisson_solve
 * may be DEVICE pointers or HOST pointers (pinned or pageable; the copy is a
 * cudaMemcpyAsync(cudaMemcpyDefault) on the context's stream).  `zf` in fizzy_grid is a HOST
 * pointer.  `dev_workspace` is a DEVICE pointer.  The caller owns every buffer it passes; the
 * library owns only the opaque context (host memory) and never calls cudaMalloc for fields.
 *
 * Execution.  All calls enqueue work on the stream given at creation and return without
 * synchronising, except fizzy_gamma (reads one double back) and calls that copy to pageable
 * host memory (CUDA semantics).  No exceptions cross the ABI, no aborts, no global state.
 * There is no CPU fallback: without a CUDA device fizzy_create returns FIZZY_ECUDA.
 */
#ifndef FIZZY_H
#define FIZZY_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fizzy_ctx fizzy_ctx; /* opaque, owned by the library */

/* Version of this interface.  It goes up whenever a call changes what it reads or writes through an unchanged signature:
 *   1  round 1;   2  fizzy_diagnostics writes 8 doubles (was 6: the two Nusselt numbers were added);
 *   3  FIZZY_ENOCONV, fizzy_count_nonfinite_static.
 * A caller built against an older header compares FIZZY_ABI_VERSION (its compile-time value) with fizzy_abi_version() (the
 * loaded library's) before the first call and refuses to run on a mismatch -- e.g. a 6-double buffer handed to a version-2
 * fizzy_diagnostics would be overrun by 16 bytes. */
#define FIZZY_ABI_VERSION 3
int fizzy_abi_version(void);

typedef enum {
    FIZZY_OK = 0,
    FIZZY_EINVAL = 1, /* bad argument (see each call) */
    FIZZY_ENOMEM = 2, /* workspace too small / host allocation failed */
    FIZZY_ECUDA = 3,  /* CUDA runtime error; text via fizzy_last_error */
    FIZZY_ESTATE = 4, /* call out of order (substep before set_fields, stage sequence) */
    FIZZY_ENOCONV = 5 /* pressure solver 1 only: the iterative solve missed rtol within max_iter (no CUDA call failed) */
} fizzy_status;

/* Grid ("3D Cartesian grid").  nx, ny powers of two in [8, 1024]; nz >= 4;
 * nx*ny*nz < 2^31 (the kernels use 32-bit cell offsets).
 * zf == NULL: uniform z.  Otherwise nz+1 HOST doubles, zf[0] = 0, zf[nz] = lz, strictly
 * increasing (stretched grids need z_wall = 1).  Cell centres are face midpoints (N10). */
typedef struct {
    int nx, ny, nz;
    double lx, ly, lz;
    const double *zf;
} fizzy_grid;

/* Boundary conditions: x, y always periodic (all BASELINE.json configs). */
typedef struct {
    int z_wall;        /* 0: periodic z; 1: no-slip, impermeable walls at z = 0 and z = lz */
    double t_wall[2];  /* Dirichlet temperature at the bottom, top wall (heat on) */
} fizzy_bc;

/* Physical parameters.  Index [0] = fluid 1 (phi = 1), [1] = fluid 2 (phi = 0). */
typedef struct {
    double rho[2], mu[2], kth[2], cp[2];
    double sigma;                 /* surface tension coefficient (CSF: sigma*kappa*grad phi) */
    double eps;                   /* interface thickness parameter of ACDI */
    double delta;                 /* regulariser in psi = eps*ln((phi+delta)/(1-phi+delta)); N2: 1e-100;
                                     must be >= 1e-150 so that sqrt(q_a q_b) stays finite (D3) */
    double gamma_rel, gamma_abs;  /* Gamma = gamma_rel*max|u| + gamma_abs, refreshed at stage 0 (N15) */
    double g[3];                  /* gravity */
    double rho_ref;               /* gravity enters as g*(1 - rho_ref/rho_f) (N12) */
    double beta, t_ref;           /* Oberbeck-Boussinesq: -g*beta*(T - t_ref) (N13) */
    double force[3];              /* uniform body acceleration */
    double lin_forcing;           /* Lundgren linear forcing coefficient A: + A*u (N22) */
    int heat;                     /* 1: evolve the temperature equation */
} fizzy_props;

/* Bytes of device workspace fizzy_create needs for this grid / property set (0 on bad input). */
size_t fizzy_workspace_bytes(const fizzy_grid *grid, const fizzy_bc *bc, const fizzy_props *props);

/* Create a context for one grid / boundary set / fluid pair (3-D Cartesian grid, staggered
 * velocity, cell-centred scalars; two fluids with properties mapped over phi; BASELINE.json:7-11 for
 * the boundary sets: x, y periodic, z periodic or walls, uniform or stretched).  `dev_workspace` must hold at least fizzy_workspace_bytes() bytes, be
 * 256-byte aligned and outlive the context.  `cuda_stream` is a cudaStream_t (NULL = default
 * stream).  Builds the 1-D metric tables, FFT twiddles, modified wavenumbers
 * lam_x(l) = -4 sin^2(pi l/nx)/dx^2 (lam_y likewise) and the z-tridiagonal elimination tables.
 * The workspace must be memory of the CUDA device that is current at this call; every later call on the context
 * must find the same device current (FIZZY_ESTATE otherwise).
 * FIZZY_EINVAL: nx, ny not powers of two in [8,1024], nz < 4 or > 65535, nx*ny*nz >= 2^31, lengths <= 0, non-monotone zf,
 * zf given with z_wall = 0, rho <= 0, mu < 0, eps <= 0, delta < 1e-150, cp or kth <= 0 with heat on,
 * misaligned workspace.  FIZZY_ENOMEM: workspace too small. */
fizzy_status fizzy_create(const fizzy_grid *grid, const fizzy_bc *bc, const fizzy_props *props,
                          void *dev_workspace, size_t workspace_bytes, void *cuda_stream,
                          fizzy_ctx **out);

fizzy_status fizzy_destroy(fizzy_ctx *ctx);

/* Load the prognostic fields of the one-fluid model (velocity, pressure, phase indicator phi,
 * temperature; p_prev is the previous substep pressure of the splitting, N7) in the layout above (PAPER.md:36
 * staggered arrangement).  Host or device pointers, N doubles each.  NULL = leave unchanged
 * (the workspace starts zero-filled).  p_prev == NULL sets p_prev := p when p is given.
 * Zeroes the RK history, enforces w[:,:,nz-1] = 0 with walls, recomputes max|u| and the
 * interface quantities of phi, and resets the stage counter to 0. */
fizzy_status fizzy_set_fields(fizzy_ctx *ctx, const double *u, const double *v, const double *w,
                              const double *p, const double *phi, const double *T,
                              const double *p_prev);

/* One RK3 substep, stage = 0, 1, 2 in this order (N1: Wray coefficients gamma = 8/15, 5/12,
 * 3/4; zeta = 0, -17/60, -5/12).  Steps S0-S5 of DESIGN.md: Gamma latch (stage 0), ACDI phi
 * transport, property map, temperature transport (heat on), momentum predictor, Poisson
 * right-hand side + FFT(x,y) + tridiagonal(z) solve, velocity correction and pressure rotation.
 * After stages 0 and 1 the velocity correction is carried out by the first kernel of the NEXT substep (fused with its
 * phi transport); any call that reads or replaces a field in between (fizzy_get_fields, fizzy_set_fields,
 * fizzy_diagnostics, fizzy_stable_dt, fizzy_check_finite, fizzy_poisson_solve) carries it out first, so the state seen
 * through this interface after a substep is always the corrected one (BASELINE.json:5(v)).
 * FIZZY_EINVAL: stage not in {0,1,2} or dt <= 0.  FIZZY_ESTATE: fields not set / wrong stage. */
fizzy_status fizzy_rk3_substep(fizzy_ctx *ctx, int stage, double dt);

/* One full RK3 step = the three substeps above in order ("low-storage three-step Runge-Kutta").
 * With fizzy_graph_enable(ctx, 1) the three substeps (23 kernel launches) are captured once into a CUDA
 * graph per buffer rotation and time step and replayed afterwards -- what matters on the 32^3 .. 128^3
 * configurations, where a substep is launch-bound.  The results are bit-identical to the
 * plain launches.  Graph capture needs a context created on a non-default stream (FIZZY_EINVAL otherwise) and
 * is bypassed while fizzy_timing_enable is on.  FIZZY_ESTATE unless the next stage is 0. */
fizzy_status fizzy_rk3_step(fizzy_ctx *ctx, double dt);
fizzy_status fizzy_graph_enable(fizzy_ctx *ctx, int on);

/* Stable time step of the CURRENT fields, reading N16 of DESIGN.md (BASELINE.json:8 "dt from CFL 0.5"):
 *   dt = cfl * min( 1/max(|u|/dx + |v|/dy + |w|/dzf),  1/(2 nu_max S),  sqrt((rho1+rho2) dmin^3/(4 pi sigma)),
 *                   1/(2 Gamma eps S),  1/(2 a_max S) [heat on] ),   S = 1/dx^2 + 1/dy^2 + 1/dzmin^2,
 * Gamma = gamma_rel*max|u| + gamma_abs.  The two maxima are reduced on the device (one pass over u, v, w); the
 * scalar formula is evaluated on the host.  Synchronises the stream.  *dt = 0 if nothing limits.
 * FIZZY_EINVAL: dt NULL or cfl <= 0.  FIZZY_ESTATE before fizzy_set_fields. */
fizzy_status fizzy_stable_dt(fizzy_ctx *ctx, double cfl, double *dt);

/* Number of non-finite values among u, v, w, p, phi (and T with heat on); one pass, synchronises the stream. */
fizzy_status fizzy_check_finite(fizzy_ctx *ctx, long long *count);

/* Count the non-finite values (Inf, NaN) in up to 8 fields WITHOUT a context, a workspace or any allocation: the health check
 * of fizzy_check_finite (failure detection) for code that is handed field pointers and nothing else.
 * Who needs this: a monitoring or output hook that the solver calls between steps with device pointers to u, v, w, p, phi, T.
 * Such a hook owns no device memory and must not ask for any: the host application has usually given the whole GPU to its own
 * pool allocator (a cudaMalloc from the hook fails, or takes memory the solver counted on), and cudaMalloc / cudaFree
 * synchronise the device, which would stall the solver's streams in the middle of a run.  The same holds inside any loop
 * where an implicit device-wide synchronisation is not acceptable.
 * Scratch: a file-scope __device__ array inside libfizzy.so (256 KiB + 256 B on every GPU that loads the library, held until
 * the process exits) -- one partial count per 4096-value chunk, which is what limits n:
 *     n <= FIZZY_STATIC_MAX_VALUES = 2^27 values per field (a 512^3 grid), nfields <= FIZZY_STATIC_MAX_FIELDS = 8.
 * Larger n is rejected with FIZZY_EINVAL and a message; nothing is launched.  The call makes no cudaMalloc, cudaFree or
 * allocating library call.
 * dev_fields: HOST array of nfields pointers, each to n doubles in memory of the CURRENT device (device or managed memory;
 *             host pointers are rejected -- staging them would need an allocation).  The fields are only read.
 * cuda_stream: cudaStream_t the work is enqueued on (NULL = default stream).  count: HOST pointer, receives the number of
 * non-finite values over all fields.  Synchronises that stream (the count is read back), nothing else.
 * err / err_len: optional HOST buffer for a message when the status is not FIZZY_OK (may be NULL / 0).
 * First call on a device: it also looks up the device address of the built-in array on the current device
 * (cudaGetSymbolAddress, once per device, which may load the library's GPU code there).  Make that first call during
 * start-up, before any stream capture begins.
 * Sharing: every call on a device uses the same array, and the array keeps the last call's contents.  The call clears the two
 * words that must start at zero itself; calls that overlap on the GPU (two streams, two host threads) race on the array and
 * return garbage -- issue them one after another.
 * FIZZY_EINVAL: NULL dev_fields / count / field pointer, nfields or n out of range, a field that is not memory of the
 * current device.  FIZZY_ECUDA: a CUDA runtime call failed (text in err). */
#define FIZZY_STATIC_MAX_VALUES 134217728LL
#define FIZZY_STATIC_MAX_FIELDS 8
fizzy_status fizzy_count_nonfinite_static(const double *const *dev_fields, int nfields, long long n, void *cuda_stream,
                                          long long *count, char *err, size_t err_len);

/* Solve Lap p = rhs with the context's grid and z boundary condition (periodic x, y; periodic
 * or homogeneous Neumann z): FFT in x and y, tridiagonal in z (BASELINE.json:5(iv)).  The
 * singular mean mode follows N17: last row replaced by p_hat(nz-1) = 0, then the dzf-weighted
 * mean is removed.  rhs and p are N doubles, host or device; they may alias. */
fizzy_status fizzy_poisson_solve(fizzy_ctx *ctx, const double *rhs, double *p);

/* the conventional VARIABLE-COEFFICIENT pressure problem that PAPER.md:36 names as Fizzy's alternative to
 * the splitting ("solving the conventional variable-coefficients problem using a geometric multigrid method"):
 *     D( (1/rho_f) d_a p ) = rhs,   rho_f = 1/2 (rho + rho(+1_a)),  rho = rho[1] + (rho[0]-rho[1]) clip(phi,0,1)  (N2, N11),
 * with the context's grid and z boundary condition (periodic x, y; periodic or no-flux walls in z; stretched z allowed).
 * Solved by conjugate gradients preconditioned with one geometric multigrid V-cycle (red-black Gauss-Seidel, levels
 * halving nx, ny, nz while all stay even and >= 4), to  ||rhs' - A p|| <= rtol ||rhs'||  in the dzf-weighted 2-norm, where
 * rhs' = rhs minus its dzf-weighted mean (the operator is singular); p is returned with zero dzf-weighted mean (N17).
 * rhs, p: N doubles, host or device.  phi: N doubles, host or device, or NULL = the context's current phase field.
 * dev_work: caller-owned DEVICE scratch of fizzy_varcoef_workspace_bytes(ctx) bytes, 256-byte aligned (about 10 N
 * doubles); nothing is kept in it between calls.  *iters (may be NULL) = CG iterations used, *relres (may be NULL) = the
 * relative residual reached.  Synchronises the stream (the CG scalars are read on the host).
 * FIZZY_EINVAL: NULL rhs / p / dev_work, rtol <= 0, max_iter < 1, misaligned dev_work.  FIZZY_ENOMEM: work_bytes too small.
 * FIZZY_ESTATE: phi == NULL before fizzy_set_fields.  Not converged within max_iter is NOT an error: check *relres. */
size_t fizzy_varcoef_workspace_bytes(const fizzy_ctx *ctx);

/* Choose the pressure path of fizzy_rk3_substep (PAPER.md:36 offers both):
 *   solver 0 (default): the constant-coefficient splitting, direct FFT / tridiagonal solve (BASELINE.json:5(iv),(v));
 *   solver 1: the variable-coefficient problem  D((1/rho_f) d p_new) = D(u*)/(a dt)  by the multigrid-preconditioned CG above
 *             (to rtol, at most max_iter iterations), then  u = u* - a dt (1/rho_f) d p_new;  no extrapolated pressure, no
 *             reference density.  dev_work: caller-owned DEVICE scratch of fizzy_varcoef_workspace_bytes(ctx) bytes, 256-byte
 *             aligned, which must stay valid while solver 1 is selected.  Every substep then synchronises the stream, CUDA
 *             graph replay is bypassed, and a solve that misses rtol within max_iter makes the substep return FIZZY_ENOCONV.  At
 *             that point phi, T, the RK histories and u** are already those of the new substep but the velocity is not yet
 *             corrected and the stage counter has not moved: the context cannot be retried as it is -- reload it with
 *             fizzy_set_fields (then e.g. raise max_iter).
 *   Going back from solver 1 to solver 0 re-forms p_hat = 2 p - p_prev (N7) from the pressures of the last two substeps.
 * Only between RK3 steps (FIZZY_ESTATE otherwise).  FIZZY_EINVAL / FIZZY_ENOMEM as for fizzy_poisson_solve_varcoef. */
fizzy_status fizzy_set_pressure_solver(fizzy_ctx *ctx, int solver, void *dev_work, size_t work_bytes, double rtol,
                                       int max_iter);
fizzy_status fizzy_poisson_solve_varcoef(fizzy_ctx *ctx, const double *rhs, const double *phi, double *p,
                                         void *dev_work, size_t work_bytes, double rtol, int max_iter,
                                         int *iters, double *relres);

/* Copy the prognostic fields out (same layout and meaning as fizzy_set_fields; host or device pointers); any
 * pointer may be NULL.  Enqueued on the stream like every other call: synchronise before reading host memory. */
fizzy_status fizzy_get_fields(fizzy_ctx *ctx, double *u, double *v, double *w, double *p,
                              double *phi, double *T, double *p_prev);

/* Run-time diagnostics of the current state (definitions in DESIGN.md 10), one pass
 * over the fields and a fixed-order (deterministic) reduction.  `out` = 8 HOST doubles (6 before FIZZY_ABI_VERSION 2),
 * dV = dx*dy*dzf[k]:
 *   out[0] = sum phi dV (volume of fluid 1)        out[1] = 1/2 sum rho(phi) |u_c|^2 dV, u_c = cell-centred mean
 *   out[2] = max over faces of max(|u|,|v|,|w|)    out[3] = max |D(u)|
 *   out[4] = sum |grad phi| dV (central differences: area of the diffuse interface)
 *   out[5] = sum T dV / sum dV (0 with heat off)
 *   out[6], out[7] = Nusselt number at the bottom, top wall: <-dT/dz>_wall * lz/(t_wall[0] - t_wall[1]), the wall
 *            gradient taken through the Dirichlet ghost 2 T_wall - T (0 unless heat on, z_wall = 1, t_wall differ).
 * Synchronises the stream.  FIZZY_ESTATE before fizzy_set_fields. */
fizzy_status fizzy_diagnostics(fizzy_ctx *ctx, double *out);

/* Current Gamma = gamma_rel*max|u| + gamma_abs as latched at the last stage 0 (N15; BASELINE.json:8-11
 * "Gamma = max|u|"); gamma_abs before the first substep.  Synchronises the stream.  NaN if ctx is NULL or
 * its device is not current. */
double fizzy_gamma(const fizzy_ctx *ctx);

/* Number of kernels the library has launched on this context so far (host counter). */
long long fizzy_launch_count(const fizzy_ctx *ctx);

/* Measurement aid (used by bench.py for the roofline object): with timing on, every kernel
 * launch is bracketed by CUDA events recorded on the context's stream.  fizzy_timing_get
 * synchronises the stream, folds the pending events into per-kernel totals and returns the
 * name, accumulated milliseconds and launch count of kernel slot `index` (0-based;
 * FIZZY_EINVAL past the last slot); reset != 0 clears that slot afterwards. */
fizzy_status fizzy_timing_enable(fizzy_ctx *ctx, int on);
fizzy_status fizzy_timing_get(fizzy_ctx *ctx, int index, const char **name, double *total_ms,
                              long long *launches, int reset);

/* Text of the last error on this context ("" if none); static text if ctx is NULL. */
const char *fizzy_last_error(const fizzy_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* FIZZY_H */
