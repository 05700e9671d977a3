// fizzy_api.cu -- host side of libfizzy.so: the C ABI of include/fizzy.h, workspace carving,
// 1-D table construction and the fixed kernel sequence of one RK3 substep.
#include "../../include/fizzy.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "fz_common.cuh"
#include "fz_diag.cuh"
#include "fz_fftx.cuh"
#include "fz_iface.cuh"
#include "fz_momentum.cuh"
#include "fz_stencil.cuh"
#include "fz_spectral.cuh"
#include "fz_mg.cuh"

namespace {

const double RK_GAMMA[3] = {8.0 / 15.0, 5.0 / 12.0, 3.0 / 4.0};   // N1 (Wray)
const double RK_ZETA[3] = {0.0, -17.0 / 60.0, -5.0 / 12.0};

struct Carver {  // hands out 256-byte aligned pieces of the workspace (or just counts)
    char *base;
    size_t off;
    explicit Carver(void *b) : base(static_cast<char *>(b)), off(0) {}
    void *take(size_t bytes)
    {
        void *p = base ? base + off : nullptr;
        off += (bytes + 255) & ~size_t(255);
        return p;
    }
    double *dbl(size_t n) { return static_cast<double *>(take(n * sizeof(double))); }
};

}  // namespace

enum FzKernelId { FZK_LATCH, FZK_PHI, FZK_CORRPHI, FZK_IMARCH, FZK_IPSI, FZK_INHAT, FZK_IFLUX, FZK_TEMP, FZK_MOM, FZK_FFTX_FWD,
                  FZK_SPEC_FWD, FZK_SPEC_BWD, FZK_FFTX_INV, FZK_CORRECT, FZK_OTHER, FZK_MG, FZK_COUNT };
static const char *const FZK_NAME[FZK_COUNT] = {
    "k_latch_gamma", "k_phi_update", "k_corr_phi", "k_iface_march", "k_iface_psi", "k_iface_nhat", "k_iface_flux", "k_temp_update", "k_momentum",
    "k_fftx_fwd", "k_spec_fwd", "k_spec_bwd", "k_fftx_inv", "k_correct", "other", "mg_cg_solve (whole call)"};

struct FzTimed { int id; cudaEvent_t e0, e1; };

struct fizzy_ctx {
    FzP P;
    // optional per-kernel timing (fizzy_timing_enable): CUDA events around every launch
    bool timing = false;
    std::vector<FzTimed> pending;
    std::vector<cudaEvent_t> pool;
    double t_ms[FZK_COUNT] = {0};
    long long t_n[FZK_COUNT] = {0};
    cudaStream_t stream;
    int device;                // CUDA device the context was created on (every later call must find it current)
    bool varrho, varmu, heat, cyclic;
    int log2nx, log2ny;
    long long N, M;
    // fields
    double *u, *v, *w, *us, *vs, *ws, *hu, *hv, *hw;
    double *phi, *phin, *hphi;
    double *p, *pp, *pn;
    double *phat;   // 2p - p_prev (N7), rho1 != rho2 only: written by k_correct, staged by k_momentum_march
    double *T, *Tn, *hT;
    double *kappa, *divrn, *psi, *rr, *nhx, *nhy, *nhz, *rnx, *rny, *rnz;
    double2 *spec;
    CUtensorMap tm_spec;   // the half-spectrum as a rank-3 tensor (2 ny doubles | nxh | nz): input boxes of k_fftx_inv (TMA)
    double2 *twx, *twy;
    double *scal;  // [0] running max|u|, [1] Gamma, [2], [6] gauge mean (two parts), [3..4] dt maxima, [5] non-finite count, [8..15] diagnostics
    double dzmin;  // smallest cell height (N16)
    std::vector<double> hdzf;   // host copy of dzf[0..nz-1] (level tables of fizzy_poisson_solve_varcoef)
    // one RK3 step as a CUDA graph (fizzy_graph_enable): one executable graph per parity of the step counter,
    // because phi/phi_new (and T/T_new) swap three times per step and are back in place after two steps
    bool graph_on = false;
    double *phi0 = nullptr;                       // the buffer phi occupied at creation: selects the graph slot
    cudaGraphExec_t gexec[2] = {nullptr, nullptr};
    double gdt[2] = {0.0, 0.0};
    const double *gkey[2][2] = {{nullptr, nullptr}, {nullptr, nullptr}};   // p, p_prev buffers baked into the graph
    long long glaunches[2] = {0, 0};
    double *dpart; // block partials of k_diag
    FzTri tri;
    int fields_set, next_stage;
    // S5 of stages 0 and 1 is deferred into the first kernel of the next substep (k_corr_phi): until then u, v, w
    // still hold the velocity of the stage start and corr_coef = a dt / rho0 of the pending correction
    bool corr_pending = false;
    double corr_coef = 0.0;
    // pressure path of the substep: 0 = the constant-coefficient splitting (FFT solver), 1 = the variable-coefficient problem
    // by multigrid-preconditioned CG, with the caller's scratch (fizzy_set_pressure_solver)
    int solver = 0;
    void *mg_work = nullptr;
    size_t mg_bytes = 0;
    double mg_rtol = 1e-12;
    int mg_maxit = 200;
    long long launches;
    std::string err;
};

namespace {

bool is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }
int ilog2(int n) { int l = 0; while ((1 << l) < n) ++l; return l; }

bool valid_inputs(const fizzy_grid *g, const fizzy_bc *bc, const fizzy_props *pr)
{
    if (!g || !bc || !pr) return false;
    if (!is_pow2(g->nx) || !is_pow2(g->ny) || g->nx < 8 || g->ny < 8 || g->nx > 1024 || g->ny > 1024) return false;
    if (g->nz < 4 || g->nz > 65535) return false;                          // k rides in gridDim.z
    if ((long long)g->nx * g->ny * g->nz >= (1LL << 31)) return false;   // kernels use 32-bit cell offsets
    if (!(g->lx > 0) || !(g->ly > 0) || !(g->lz > 0)) return false;
    if (bc->z_wall != 0 && bc->z_wall != 1) return false;
    if (g->zf) {
        if (!bc->z_wall) return false;
        if (g->zf[0] != 0.0 || g->zf[g->nz] != g->lz) return false;
        for (int k = 0; k < g->nz; ++k)
            if (!(g->zf[k + 1] > g->zf[k])) return false;
    }
    if (!(pr->rho[0] > 0) || !(pr->rho[1] > 0) || pr->mu[0] < 0 || pr->mu[1] < 0) return false;
    if (!(pr->eps > 0) || !(pr->delta >= 1e-150)) return false;   // D3: sqrt(q_a q_b) must stay finite
    if (pr->heat && (!(pr->cp[0] > 0) || !(pr->cp[1] > 0) || !(pr->kth[0] > 0) || !(pr->kth[1] > 0))) return false;
    return true;
}

// carve (or, with base == NULL, just size) the workspace; fills ctx pointers when c != NULL
size_t layout(fizzy_ctx *c, void *base, const fizzy_grid *g, const fizzy_bc *bc, const fizzy_props *pr,
              double **ztab /*5 tables*/, double **acoef /*a, c*/, double **lam /*lamx, lamy*/)
{
    Carver cv(base);
    const size_t N = (size_t)g->nx * g->ny * g->nz;
    const int nxh = g->nx / 2 + 1;
    const size_t M = (size_t)nxh * g->ny;
    const bool varrho = pr->rho[0] != pr->rho[1];
    const bool cyclic = !bc->z_wall;
    fizzy_ctx dummy;
    fizzy_ctx *x = c ? c : &dummy;
    double **f[] = {&x->u, &x->v, &x->w, &x->us, &x->vs, &x->ws, &x->hu, &x->hv, &x->hw, &x->phi, &x->phin,
                    &x->hphi, &x->p, &x->pp, &x->pn, &x->kappa, &x->divrn, &x->psi, &x->rr, &x->nhx,
                    &x->nhy, &x->nhz};
    for (auto q : f) *q = cv.dbl(N);
    x->rnx = x->rny = x->rnz = x->phat = nullptr;
    if (varrho) { x->rnx = cv.dbl(N); x->rny = cv.dbl(N); x->rnz = cv.dbl(N); x->phat = cv.dbl(N); }
    x->T = x->Tn = x->hT = nullptr;
    if (pr->heat) { x->T = cv.dbl(N); x->Tn = cv.dbl(N); x->hT = cv.dbl(N); }
    x->spec = static_cast<double2 *>(cv.take(M * g->nz * sizeof(double2)));
    x->tri.inv = cv.dbl(M * g->nz);
    x->tri.e = nullptr;
    if (cyclic) x->tri.e = cv.dbl(M * g->nz);
    x->tri.mid = cv.dbl(M * (cyclic ? 4 : 1));
    x->tri.side = static_cast<double2 *>(cv.take(4 * M * sizeof(double2)));
    for (int q = 0; q < 5; ++q) { double *t = cv.dbl(g->nz + 2 * FZ_H); if (ztab) ztab[q] = t; }
    for (int q = 0; q < 2; ++q) { double *t = cv.dbl(g->nz); if (acoef) acoef[q] = t; }
    { double *t = cv.dbl(nxh); if (lam) lam[0] = t; t = cv.dbl(g->ny); if (lam) lam[1] = t; }
    x->twx = static_cast<double2 *>(cv.take(g->nx * sizeof(double2)));
    x->twy = static_cast<double2 *>(cv.take(g->ny * sizeof(double2)));
    x->scal = cv.dbl(16);
    x->dpart = cv.dbl((size_t)FZ_DIAG_BLOCKS * FZ_DIAG_NV);
    return cv.off;
}

fizzy_status fail(fizzy_ctx *c, fizzy_status s, const char *what)
{
    if (c) c->err = what;
    return s;
}

fizzy_status cuda_fail(fizzy_ctx *c, cudaError_t e, const char *where)
{
    if (c) c->err = std::string(where) + ": " + cudaGetErrorString(e);
    return FIZZY_ECUDA;
}

#define FZ_CUDA(call)                                                   \
    do {                                                                \
        cudaError_t e_ = (call);                                        \
        if (e_ != cudaSuccess) return cuda_fail(c, e_, #call);          \
    } while (0)

cudaEvent_t take_event(fizzy_ctx *c)
{
    if (!c->pool.empty()) { cudaEvent_t e = c->pool.back(); c->pool.pop_back(); return e; }
    cudaEvent_t e = nullptr;
    if (cudaEventCreate(&e) != cudaSuccess) { cudaGetLastError(); e = nullptr; }   // no event: this launch goes untimed
    return e;
}

// FZ_TB(id) before a launch, FZ_LAUNCHED(id) after it: counts the launch, checks for a launch
// error and, in timing mode, brackets the kernel with events on the context's stream.
#define FZ_TB(id_)                                                      \
    do {                                                                \
        if (c->timing) {                                                \
            FzTimed t_; t_.id = (id_); t_.e0 = take_event(c); t_.e1 = take_event(c); \
            if (t_.e0) cudaEventRecord(t_.e0, c->stream);               \
            c->pending.push_back(t_);                                   \
        }                                                               \
    } while (0)

#define FZ_LAUNCHED(id_)                                                \
    do {                                                                \
        ++c->launches;                                                  \
        if (c->timing && c->pending.back().e1) cudaEventRecord(c->pending.back().e1, c->stream); \
        cudaError_t e_ = cudaPeekAtLastError();                         \
        if (e_ != cudaSuccess) return cuda_fail(c, e_, FZK_NAME[id_]);  \
    } while (0)

cudaError_t launch_momentum(fizzy_ctx *c, dim3 grid, dim3 block, const FzMomArgs *A);   // defined with the substep

// Planes per z chunk of a marching kernel: a CTA marches KC planes after `ov` planes of pipeline fill, `slots` CTAs run at
// a time.  Cost model: (waves, at least one, + half a wave of tail) x (KC + ov); ties go to the longer chunk.  Large grids
// get 64-128 planes per chunk (measured at 512^3: 4096-8192 CTAs are the flat optimum), small ones short chunks, so
// that a 32^3 grid is not marched by eight CTAs of nineteen plane steps each.
int march_chunk(int nz, int tiles, int slots, int ov)
{
    int best = nz;
    double best_cost = 1e300;
    for (int kc = 4; ; kc *= 2) {
        if (kc > nz) kc = nz;
        const double ctas = (double)tiles * ((nz + kc - 1) / kc);
        double waves = ctas / slots + 0.5;
        if (waves < 1.0) waves = 1.0;
        const double cost = waves * (kc + ov);
        if (cost <= best_cost * 1.0000001) { best_cost = cost; best = kc; }
        if (kc == nz) break;
    }
    return best;
}

void cell_launch(const fizzy_ctx *c, dim3 &grid, dim3 &block)
{
    const int bx = c->P.nx < 64 ? c->P.nx : 64;
    int by = 256 / bx;
    if (by > c->P.ny) by = c->P.ny;
    block = dim3(bx, by, 1);
    grid = dim3(c->P.nx / bx, c->P.ny / by, c->P.nz);
}

}  // namespace

// =====================================================================================
extern "C" size_t fizzy_workspace_bytes(const fizzy_grid *grid, const fizzy_bc *bc, const fizzy_props *props)
{
    if (!valid_inputs(grid, bc, props)) return 0;
    return layout(nullptr, nullptr, grid, bc, props, nullptr, nullptr, nullptr);
}

extern "C" fizzy_status fizzy_create(const fizzy_grid *grid, const fizzy_bc *bc, const fizzy_props *props,
                                     void *dev_workspace, size_t workspace_bytes, void *cuda_stream,
                                     fizzy_ctx **out)
{
    if (!out) return FIZZY_EINVAL;
    *out = nullptr;
    if (!valid_inputs(grid, bc, props)) return FIZZY_EINVAL;
    if (!dev_workspace || (reinterpret_cast<uintptr_t>(dev_workspace) & 255)) return FIZZY_EINVAL;
    if (workspace_bytes < layout(nullptr, nullptr, grid, bc, props, nullptr, nullptr, nullptr)) return FIZZY_ENOMEM;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return FIZZY_ECUDA;  // no CPU fallback
    fizzy_ctx *c = new (std::nothrow) fizzy_ctx();
    if (!c) return FIZZY_ENOMEM;
    *out = c;  // returned even on a CUDA failure below so that fizzy_last_error can be read
    c->stream = static_cast<cudaStream_t>(cuda_stream);
    FZ_CUDA(cudaGetDevice(&c->device));
    {   // the workspace must live on the current device
        cudaPointerAttributes pa;
        if (cudaPointerGetAttributes(&pa, dev_workspace) != cudaSuccess || pa.type != cudaMemoryTypeDevice ||
            pa.device != c->device) {
            cudaGetLastError();
            return fail(c, FIZZY_EINVAL, "dev_workspace is not device memory of the current CUDA device");
        }
    }
    c->fields_set = 0;
    c->next_stage = 0;
    c->launches = 0;

    const int nx = grid->nx, ny = grid->ny, nz = grid->nz;
    double *ztab[5], *acoef[2], *lam[2];
    const size_t used = layout(c, dev_workspace, grid, bc, props, ztab, acoef, lam);
    c->phi0 = c->phi;
    FZ_CUDA(cudaMemsetAsync(dev_workspace, 0, used, c->stream));

    FzP &P = c->P;
    std::memset(&P, 0, sizeof(P));
    P.nx = nx; P.ny = ny; P.nz = nz; P.nxh = nx / 2 + 1;
    P.z_wall = bc->z_wall; P.heat = props->heat ? 1 : 0;
    P.kzf = bc->z_wall ? nz - 1 : nz;
    P.N = (long long)nx * ny * nz; P.sxy = (long long)nx * ny;
    P.dx = grid->lx / nx; P.dy = grid->ly / ny; P.idx = 1.0 / P.dx; P.idy = 1.0 / P.dy; P.lz = grid->lz;
    P.rho1 = props->rho[0]; P.rho2 = props->rho[1]; P.mu1 = props->mu[0]; P.mu2 = props->mu[1];
    P.k1 = props->kth[0]; P.k2 = props->kth[1]; P.cp1 = props->cp[0]; P.cp2 = props->cp[1];
    P.sigma = props->sigma; P.eps = props->eps; P.delta = props->delta;
    P.gamma_rel = props->gamma_rel; P.gamma_abs = props->gamma_abs;
    P.gx = props->g[0]; P.gy = props->g[1]; P.gz = props->g[2];
    P.rho_ref = props->rho_ref; P.beta = props->beta; P.t_ref = props->t_ref;
    P.fx = props->force[0]; P.fy = props->force[1]; P.fz = props->force[2];
    P.a_lin = props->lin_forcing;
    P.t_bot = bc->t_wall[0]; P.t_top = bc->t_wall[1];
    P.rho0 = std::fmin(P.rho1, P.rho2); P.drho = P.rho1 - P.rho2;
    c->N = P.N; c->M = (long long)P.nxh * ny;
    c->varrho = P.rho1 != P.rho2; c->varmu = P.mu1 != P.mu2; c->heat = P.heat != 0; c->cyclic = !bc->z_wall;
    c->log2nx = ilog2(nx); c->log2ny = ilog2(ny);
    // ---- 1-D z metrics with ghosts (walls mirror, periodic wraps), N10: centres = face midpoints
    const int nzt = nz + 2 * FZ_H;
    std::vector<double> dzf(nzt), dzc(nzt, 0.0), idzf(nzt), idzc(nzt, 0.0), igz(nzt, 0.0);
    for (int k = 0; k < nz; ++k) dzf[k + FZ_H] = grid->zf ? grid->zf[k + 1] - grid->zf[k] : grid->lz / nz;
    for (int g = 1; g <= FZ_H; ++g) {
        dzf[FZ_H - g] = bc->z_wall ? dzf[FZ_H + g - 1] : dzf[FZ_H + nz - g];
        dzf[FZ_H + nz - 1 + g] = bc->z_wall ? dzf[FZ_H + nz - g] : dzf[FZ_H + g - 1];
    }
    for (int q = 0; q < nzt - 1; ++q) dzc[q] = 0.5 * (dzf[q] + dzf[q + 1]);
    dzc[nzt - 1] = dzc[nzt - 2];
    for (int q = 0; q < nzt; ++q) { idzf[q] = 1.0 / dzf[q]; idzc[q] = 1.0 / dzc[q]; }
    c->hdzf.assign(dzf.begin() + FZ_H, dzf.begin() + FZ_H + nz);
    c->dzmin = dzf[FZ_H];
    for (int k = 0; k < nz; ++k) c->dzmin = std::fmin(c->dzmin, dzf[k + FZ_H]);
    for (int q = 1; q < nzt; ++q) igz[q] = 1.0 / (dzc[q] + dzc[q - 1]);
    const std::vector<double> *tabs[5] = {&dzf, &dzc, &idzf, &idzc, &igz};
    for (int q = 0; q < 5; ++q)
        FZ_CUDA(cudaMemcpyAsync(ztab[q], tabs[q]->data(), nzt * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    P.dzf = ztab[0] + FZ_H; P.dzc = ztab[1] + FZ_H; P.idzf = ztab[2] + FZ_H; P.idzc = ztab[3] + FZ_H;
    P.igz = ztab[4] + FZ_H;

    // ---- tridiagonal coefficients, modified wavenumbers, twiddles
    std::vector<double> a(nz), cc(nz), lx(P.nxh), ly(ny);
    for (int k = 0; k < nz; ++k) {
        a[k] = 1.0 / (dzf[k + FZ_H] * dzc[k - 1 + FZ_H]);
        cc[k] = 1.0 / (dzf[k + FZ_H] * dzc[k + FZ_H]);
    }
    if (bc->z_wall) { a[0] = 0.0; cc[nz - 1] = 0.0; }
    for (int l = 0; l < P.nxh; ++l) { const double s = std::sin(M_PI * l / nx); lx[l] = -4.0 * s * s / (P.dx * P.dx); }
    for (int m = 0; m < ny; ++m) { const double s = std::sin(M_PI * m / ny); ly[m] = -4.0 * s * s / (P.dy * P.dy); }
    std::vector<double2> twx(nx), twy(ny);
    for (int q = 0; q < nx; ++q) { const double t = -2.0 * M_PI * q / nx; twx[q] = make_double2(std::cos(t), std::sin(t)); }
    for (int q = 0; q < ny; ++q) { const double t = -2.0 * M_PI * q / ny; twy[q] = make_double2(std::cos(t), std::sin(t)); }
    FZ_CUDA(cudaMemcpyAsync(acoef[0], a.data(), nz * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    FZ_CUDA(cudaMemcpyAsync(acoef[1], cc.data(), nz * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    FZ_CUDA(cudaMemcpyAsync(lam[0], lx.data(), P.nxh * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    FZ_CUDA(cudaMemcpyAsync(lam[1], ly.data(), ny * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    FZ_CUDA(cudaMemcpyAsync(c->twx, twx.data(), nx * sizeof(double2), cudaMemcpyHostToDevice, c->stream));
    FZ_CUDA(cudaMemcpyAsync(c->twy, twy.data(), ny * sizeof(double2), cudaMemcpyHostToDevice, c->stream));
    FZ_CUDA(cudaStreamSynchronize(c->stream));  // the host vectors go out of scope below

    c->tri.a = acoef[0]; c->tri.c = acoef[1]; c->tri.lamx = lam[0]; c->tri.lamy = lam[1];
    c->tri.cyclic = c->cyclic ? 1 : 0;
    FZ_TB(FZK_OTHER);
    k_tri_tables<<<(unsigned)((c->M + 127) / 128), 128, 0, c->stream>>>(P, c->tri);
    FZ_LAUNCHED(FZK_OTHER);

    // ---- tensor map of the half-spectrum for the TMA loads of k_fftx_inv (driver entry point through the runtime:
    // libfizzy.so does not link libcuda)
    {
        typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                      const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                      CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        FZ_CUDA(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
        if (!fn || qres != cudaDriverEntryPointSuccess) return fail(c, FIZZY_ECUDA, "cuTensorMapEncodeTiled is not available");
        const FzFxInvGeom G = fx_inv_geom(c->log2nx);
        const cuuint64_t gdim[3] = {(cuuint64_t)2 * ny, (cuuint64_t)P.nxh, (cuuint64_t)nz};
        const cuuint64_t gstr[2] = {(cuuint64_t)ny * 16, (cuuint64_t)P.nxh * ny * 16};
        const cuuint32_t box[3] = {(cuuint32_t)(G.rowb / 8), (cuuint32_t)G.brows, 1};
        const cuuint32_t estr[3] = {1, 1, 1};
        const CUtensorMapSwizzle sw = G.rowb == 128 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_64B;
        const CUresult r = reinterpret_cast<encode_fn>(fn)(&c->tm_spec, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, c->spec, gdim, gstr,
                                                           box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, sw,
                                                           CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return fail(c, FIZZY_ECUDA, "cuTensorMapEncodeTiled failed");
    }

    // dynamic shared memory opt-in of every kernel instantiation this context will launch: once, here,
    // so that a substep is launches only (and can be captured into a CUDA graph)
    FZ_CUDA(cudaFuncSetAttribute(k_iface_march<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)IFACE_SMEM));
    FZ_CUDA(cudaFuncSetAttribute(k_iface_march<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)IFACE_SMEM));
    FZ_CUDA(launch_momentum(c, dim3(), dim3(), nullptr));
    FZ_CUDA(fz_fftx_launch(-1, c->log2nx, P, nullptr, nullptr, nullptr, nullptr, 0.0, nullptr, nullptr, nullptr, nullptr, nullptr, c->stream));
    FZ_CUDA(c->cyclic ? fz_spec_launch<true>(-1, c->log2ny, P, c->tri, nullptr, nullptr, nullptr, c->stream)
                      : fz_spec_launch<false>(-1, c->log2ny, P, c->tri, nullptr, nullptr, nullptr, c->stream));
    return FIZZY_OK;
}

extern "C" fizzy_status fizzy_destroy(fizzy_ctx *c)
{
    if (!c) return FIZZY_EINVAL;
    cudaStreamSynchronize(c->stream);
    for (FzTimed &t : c->pending) { if (t.e0) cudaEventDestroy(t.e0); if (t.e1) cudaEventDestroy(t.e1); }
    for (cudaEvent_t e : c->pool) cudaEventDestroy(e);
    for (cudaGraphExec_t g : c->gexec)
        if (g) cudaGraphExecDestroy(g);
    delete c;
    return FIZZY_OK;
}

extern "C" fizzy_status fizzy_timing_enable(fizzy_ctx *c, int on)
{
    if (!c) return FIZZY_EINVAL;
    c->timing = on != 0;
    return FIZZY_OK;
}

extern "C" fizzy_status fizzy_timing_get(fizzy_ctx *c, int index, const char **name, double *total_ms,
                                         long long *launches, int reset)
{
    if (!c || index < 0 || index >= FZK_COUNT) return FIZZY_EINVAL;
    if (!c->pending.empty()) {
        FZ_CUDA(cudaStreamSynchronize(c->stream));
        for (FzTimed &t : c->pending) {
            float ms = 0.f;
            if (t.e0 && t.e1 && cudaEventElapsedTime(&ms, t.e0, t.e1) == cudaSuccess) { c->t_ms[t.id] += ms; ++c->t_n[t.id]; }
            else cudaGetLastError();   // e.g. an end event never recorded because its call failed midway: not a launch error
            if (t.e0) c->pool.push_back(t.e0);
            if (t.e1) c->pool.push_back(t.e1);
        }
        c->pending.clear();
    }
    if (name) *name = FZK_NAME[index];
    if (total_ms) *total_ms = c->t_ms[index];
    if (launches) *launches = c->t_n[index];
    if (reset) { c->t_ms[index] = 0.0; c->t_n[index] = 0; }
    return FIZZY_OK;
}

extern "C" int fizzy_abi_version(void) { return FIZZY_ABI_VERSION; }
extern "C" const char *fizzy_last_error(const fizzy_ctx *c) { return c ? c->err.c_str() : "null context"; }
extern "C" long long fizzy_launch_count(const fizzy_ctx *c) { return c ? c->launches : 0; }

extern "C" double fizzy_gamma(const fizzy_ctx *c)
{
    if (!c) return NAN;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != c->device) return NAN;
    double g = NAN;
    if (cudaMemcpyAsync(&g, c->scal + 1, sizeof(double), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess) return NAN;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return NAN;
    return g;
}

// =====================================================================================
namespace {

// interface quantities of c->phi -> kappa, divRn (and Rn when rho1 != rho2): kernel group (a).
// with_psi: psi of c->phi is not yet in c->psi (fizzy_set_fields); inside a substep k_phi_update
// has already written it.  r = sqrt(q) is recomputed on chip by the marching sweep; only the
// tiny-grid fallback reads it from c->rr (k_iface_psi writes both).
fizzy_status run_interface(fizzy_ctx *c, bool with_psi)
{
    const FzP &P = c->P;
    dim3 grid, block;
    cell_launch(c, grid, block);
    const bool march = P.nx >= ITX && P.ny >= ITY;
    if (with_psi || !march) {
        FZ_TB(FZK_IPSI);
        k_iface_psi<<<grid, block, 0, c->stream>>>(c->P, c->phi, c->psi, c->rr);
        FZ_LAUNCHED(FZK_IPSI);
    }
    if (march) {   // marching sweep: nhat and r stay on chip
        const int KC = march_chunk(P.nz, (P.nx / ITX) * (P.ny / ITY), 148 * 2, 4);
        const dim3 g(P.nx / ITX, P.ny / ITY, (P.nz + KC - 1) / KC);
        FZ_TB(FZK_IMARCH);
        if (c->varrho)
            k_iface_march<true><<<g, dim3(ITX, ITY), IFACE_SMEM, c->stream>>>(P, c->psi, c->phi, c->kappa, c->divrn,
                                                                              c->rnx, c->rny, c->rnz, KC);
        else
            k_iface_march<false><<<g, dim3(ITX, ITY), IFACE_SMEM, c->stream>>>(P, c->psi, c->phi, c->kappa, c->divrn,
                                                                               nullptr, nullptr, nullptr, KC);
        FZ_LAUNCHED(FZK_IMARCH);
        return FIZZY_OK;
    }
    // tiny grids: one thread per cell, nhat through global memory
    FZ_TB(FZK_INHAT);
    k_iface_nhat<<<grid, block, 0, c->stream>>>(c->P, c->psi, c->nhx, c->nhy, c->nhz);
    FZ_LAUNCHED(FZK_INHAT);
    FZ_TB(FZK_IFLUX);
    if (c->varrho)
        k_iface_flux<true><<<grid, block, 0, c->stream>>>(c->P, c->phi, c->rr, c->nhx, c->nhy, c->nhz, c->kappa,
                                                          c->divrn, c->rnx, c->rny, c->rnz);
    else
        k_iface_flux<false><<<grid, block, 0, c->stream>>>(c->P, c->phi, c->rr, c->nhx, c->nhy, c->nhz, c->kappa,
                                                           c->divrn, nullptr, nullptr, nullptr);
    FZ_LAUNCHED(FZK_IFLUX);
    return FIZZY_OK;
}

// spectral part of S4 on c->spec (forward x-transform already done): fused FFT_y + z elimination,
// back substitution + inverse FFT_y (gauge mean -> scal[2]), inverse x-transform (- gauge shift)
fizzy_status run_spectral_solve(fizzy_ctx *c, double *dst)
{
    const FzP &P = c->P;
    FZ_TB(FZK_SPEC_FWD);
    FZ_CUDA(c->cyclic ? fz_spec_launch<true>(0, c->log2ny, P, c->tri, c->spec, c->twy, c->scal, c->stream)
                      : fz_spec_launch<false>(0, c->log2ny, P, c->tri, c->spec, c->twy, c->scal, c->stream));
    FZ_LAUNCHED(FZK_SPEC_FWD);
    FZ_TB(FZK_SPEC_BWD);
    FZ_CUDA(c->cyclic ? fz_spec_launch<true>(1, c->log2ny, P, c->tri, c->spec, c->twy, c->scal, c->stream)
                      : fz_spec_launch<false>(1, c->log2ny, P, c->tri, c->spec, c->twy, c->scal, c->stream));
    FZ_LAUNCHED(FZK_SPEC_BWD);
    FZ_TB(FZK_FFTX_INV);
    FZ_CUDA(fz_fftx_launch(2, c->log2nx, P, nullptr, nullptr, nullptr, nullptr, 1.0 / ((double)P.nx * (double)P.ny),
                           c->spec, dst, c->twx, c->scal, &c->tm_spec, c->stream));
    FZ_LAUNCHED(FZK_FFTX_INV);
    return FIZZY_OK;
}

// A == NULL: shared-memory opt-in of the variant this context uses (once, at fizzy_create)
template <bool VR, bool VM, bool HT>
cudaError_t launch_momentum3(fizzy_ctx *c, dim3 grid, dim3 block, const FzMomArgs *Ap)
{
    const FzP &P = c->P;
    const size_t smem = (size_t)FzMomFields<VR, HT>::NF * FzMomFields<VR, HT>::RING * MPS * sizeof(double);
    if (!Ap) return cudaFuncSetAttribute(k_momentum_march<VR, VM, HT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    const FzMomArgs &A = *Ap;
    if (P.nx >= MTX && P.ny >= MTY) {   // 2.5-D marching kernel
        const int tiles = (P.nx / MTX) * (P.ny / MTY);
        const int KC = march_chunk(P.nz, tiles, 148 * FzMomFields<VR, HT>::MINB, 3);
        const dim3 g(P.nx / MTX, P.ny / MTY, (P.nz + KC - 1) / KC);
        k_momentum_march<VR, VM, HT><<<g, dim3(MTX, MTY), smem, c->stream>>>(P, A, KC);
    } else {                            // tiny grids: one thread per cell straight from global memory
        k_momentum<VR, VM, HT><<<grid, block, 0, c->stream>>>(P, A);
    }
    return cudaSuccess;
}

template <bool VR, bool VM>
cudaError_t launch_momentum2(fizzy_ctx *c, dim3 grid, dim3 block, const FzMomArgs *A)
{
    return c->heat ? launch_momentum3<VR, VM, true>(c, grid, block, A) : launch_momentum3<VR, VM, false>(c, grid, block, A);
}

cudaError_t launch_momentum(fizzy_ctx *c, dim3 grid, dim3 block, const FzMomArgs *A)
{
    if (c->varrho) return c->varmu ? launch_momentum2<true, true>(c, grid, block, A) : launch_momentum2<true, false>(c, grid, block, A);
    return c->varmu ? launch_momentum2<false, true>(c, grid, block, A) : launch_momentum2<false, false>(c, grid, block, A);
}

// a deferred S5 (see corr_pending): form u, v, w now.  Every entry point that reads or replaces the velocity outside
// a substep calls this first, so the deferral is invisible through the ABI.
fizzy_status flush_correct(fizzy_ctx *c)
{
    if (!c->corr_pending) return FIZZY_OK;
    dim3 grid, block;
    cell_launch(c, grid, block);
    FZ_TB(FZK_CORRECT);
    // the pressures have rotated already: c->p is p_new, c->pp the pressure before it
    k_correct<false><<<grid, block, 0, c->stream>>>(c->P, c->us, c->vs, c->ws, c->p, c->u, c->v, c->w, c->corr_coef,
                                                    c->scal, c->pp, c->phat);
    FZ_LAUNCHED(FZK_CORRECT);
    c->corr_pending = false;
    return FIZZY_OK;
}
#define FZ_FLUSH()                                       \
    do {                                                 \
        const fizzy_status fs_ = flush_correct(c);       \
        if (fs_ != FIZZY_OK) return fs_;                 \
    } while (0)

// every entry point after fizzy_create: the context's device must be the current one
fizzy_status check_device(fizzy_ctx *c)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != c->device)
        return fail(c, FIZZY_ESTATE, "the CUDA device the context was created on is not the current device");
    return FIZZY_OK;
}
#define FZ_DEVICE()                                      \
    do {                                                 \
        const fizzy_status ds_ = check_device(c);        \
        if (ds_ != FIZZY_OK) return ds_;                 \
    } while (0)

}  // namespace

extern "C" fizzy_status fizzy_set_fields(fizzy_ctx *c, const double *u, const double *v, const double *w,
                                         const double *p, const double *phi, const double *T,
                                         const double *p_prev)
{
    if (!c) return FIZZY_EINVAL;
    FZ_DEVICE();
    FZ_FLUSH();
    const size_t B = (size_t)c->N * sizeof(double);
    const double *src[] = {u, v, w, p, phi, c->heat ? T : nullptr};
    double *dst[] = {c->u, c->v, c->w, c->p, c->phi, c->T};
    for (int q = 0; q < 6; ++q)
        if (src[q]) FZ_CUDA(cudaMemcpyAsync(dst[q], src[q], B, cudaMemcpyDefault, c->stream));
    if (p_prev) FZ_CUDA(cudaMemcpyAsync(c->pp, p_prev, B, cudaMemcpyDefault, c->stream));
    else if (p) FZ_CUDA(cudaMemcpyAsync(c->pp, c->p, B, cudaMemcpyDeviceToDevice, c->stream));
    double *hist[] = {c->hphi, c->hu, c->hv, c->hw, c->hT};
    for (double *h : hist)
        if (h) FZ_CUDA(cudaMemsetAsync(h, 0, B, c->stream));
    if (c->P.z_wall) {
        FZ_TB(FZK_OTHER);
        k_zero_plane<<<(unsigned)((c->P.sxy + 255) / 256), 256, 0, c->stream>>>(c->P, c->w);
        FZ_LAUNCHED(FZK_OTHER);
    }
    FZ_TB(FZK_OTHER);
    k_init_scalars<<<1, 1, 0, c->stream>>>(c->P, c->scal);   // running max|u| = 0, Gamma = gamma_abs
    FZ_LAUNCHED(FZK_OTHER);
    FZ_TB(FZK_OTHER);
    k_absmax3<<<148 * 8, 256, 0, c->stream>>>(c->P, c->u, c->v, c->w, c->scal);
    FZ_LAUNCHED(FZK_OTHER);
    if (c->varrho) {   // p_hat = 2p - p_prev of the loaded pressures (N7)
        dim3 grid, block;
        cell_launch(c, grid, block);
        FZ_TB(FZK_OTHER);
        k_phat<<<grid, block, 0, c->stream>>>(c->P, c->p, c->pp, c->phat);
        FZ_LAUNCHED(FZK_OTHER);
    }
    fizzy_status s = run_interface(c, true);
    if (s != FIZZY_OK) return s;
    c->fields_set = 1;
    c->next_stage = 0;
    return FIZZY_OK;
}

extern "C" fizzy_status fizzy_get_fields(fizzy_ctx *c, double *u, double *v, double *w, double *p, double *phi,
                                         double *T, double *p_prev)
{
    if (!c) return FIZZY_EINVAL;
    FZ_DEVICE();
    FZ_FLUSH();
    const size_t B = (size_t)c->N * sizeof(double);
    double *dst[] = {u, v, w, p, phi, c->heat ? T : nullptr, p_prev};
    const double *src[] = {c->u, c->v, c->w, c->p, c->phi, c->T, c->pp};
    for (int q = 0; q < 7; ++q)
        if (dst[q]) FZ_CUDA(cudaMemcpyAsync(dst[q], src[q], B, cudaMemcpyDefault, c->stream));
    return FIZZY_OK;
}

extern "C" fizzy_status fizzy_rk3_substep(fizzy_ctx *c, int stage, double dt)
{
    if (!c) return FIZZY_EINVAL;
    FZ_DEVICE();
    if (stage < 0 || stage > 2 || !(dt > 0.0)) return fail(c, FIZZY_EINVAL, "stage must be 0,1,2 and dt > 0");
    if (!c->fields_set) return fail(c, FIZZY_ESTATE, "fizzy_set_fields has not been called");
    if (stage != c->next_stage) return fail(c, FIZZY_ESTATE, "stages must be called in the order 0,1,2");
    const FzP &P = c->P;
    const double gs = RK_GAMMA[stage], zs = RK_ZETA[stage], as = gs + zs;
    dim3 grid, block;
    cell_launch(c, grid, block);
    fizzy_status s;

    // S0: latch Gamma = gamma_rel * max|u| + gamma_abs (N15)
    if (stage == 0) {
        FZ_TB(FZK_LATCH);
        k_latch_gamma<<<1, 1, 0, c->stream>>>(P, c->scal);
        FZ_LAUNCHED(FZK_LATCH);
    }
    // S1: phi transport (divRn holds D(R/Gamma) of the current phi); with the S5 of the previous substep still
    // pending it is fused in front (k_corr_phi)
    if (c->corr_pending) {
        FZ_TB(FZK_CORRPHI);
        k_corr_phi<<<grid, block, 0, c->stream>>>(P, c->us, c->vs, c->ws, c->p, c->pp, c->phat, c->u, c->v, c->w, c->phi,
                                                  c->divrn, c->hphi, c->phin, c->psi, c->scal, c->corr_coef, dt, gs, zs,
                                                  stage != 2);
        FZ_LAUNCHED(FZK_CORRPHI);
        c->corr_pending = false;
    } else {
        FZ_TB(FZK_PHI);
        k_phi_update<<<grid, block, 0, c->stream>>>(P, c->phi, c->u, c->v, c->w, c->divrn, c->hphi, c->phin, c->psi, c->scal, dt, gs, zs, stage != 2);
        FZ_LAUNCHED(FZK_PHI);
    }
    std::swap(c->phi, c->phin);
    // interface quantities of phi_new (N6): used by S3 now and by S1 of the next substep
    if ((s = run_interface(c, false)) != FIZZY_OK) return s;
    // S2b: temperature
    if (c->heat) {
        FZ_TB(FZK_TEMP);
        k_temp_update<<<grid, block, 0, c->stream>>>(P, c->T, c->phi, c->u, c->v, c->w, c->hT, c->Tn, dt, gs, zs, stage != 2);
        FZ_LAUNCHED(FZK_TEMP);
        std::swap(c->T, c->Tn);
    }
    // S2 + S3: property map on the fly, momentum predictor -> u**
    FzMomArgs A;
    A.u = c->u; A.v = c->v; A.w = c->w; A.phi = c->phi; A.kappa = c->kappa;
    A.rnx = c->rnx; A.rny = c->rny; A.rnz = c->rnz; A.p = c->p; A.pp = c->pp; A.phat = c->phat; A.T = c->T;
    A.us = c->us; A.vs = c->vs; A.ws = c->ws; A.hu = c->hu; A.hv = c->hv; A.hw = c->hw;
    A.scal = c->scal; A.dt = dt; A.gs = gs; A.zs = zs; A.keep_h = stage != 2;
    A.adt = c->solver == 1 ? 0.0 : as * dt;   // the p_hat part of the splitting rides in the predictor (D2); none with solver 1
    FZ_TB(FZK_MOM);
    FZ_CUDA(launch_momentum(c, grid, block, &A));
    FZ_LAUNCHED(FZK_MOM);
    if (c->solver == 1) {
        // S4', S5': D((1/rho_f) d p_new) = D(u*)/(a dt) by multigrid-preconditioned CG, then
        // u = u* - a dt (1/rho_f) d p_new.  No p_hat, no deferred correction; the solve synchronises the stream.
        FZ_TB(FZK_OTHER);
        k_div_rhs<<<grid, block, 0, c->stream>>>(P, c->us, c->vs, c->ws, 1.0 / (as * dt), c->pn);
        FZ_LAUNCHED(FZK_OTHER);
        int iters = 0;
        double relres = 0.0;
        s = fizzy_poisson_solve_varcoef(c, c->pn, nullptr, c->pn, c->mg_work, c->mg_bytes, c->mg_rtol, c->mg_maxit, &iters, &relres);
        if (s != FIZZY_OK) return s;
        // (the solve stops on rr <= rtol^2 bb; relres is sqrt(rr/bb): one rounding of slack so that the two tests agree)
        if (!(relres <= c->mg_rtol * (1.0 + 1e-12)))
            return fail(c, FIZZY_ENOCONV, "fizzy_rk3_substep: the variable-coefficient pressure solve did not reach rtol within max_iter; "
                                          "the context is part-way through the substep: reload it with fizzy_set_fields");
        FZ_TB(FZK_CORRECT);
        if (stage == 2)
            k_correct_var<true><<<grid, block, 0, c->stream>>>(P, c->us, c->vs, c->ws, c->pn, c->phi, c->u, c->v, c->w, as * dt, c->scal);
        else
            k_correct_var<false><<<grid, block, 0, c->stream>>>(P, c->us, c->vs, c->ws, c->pn, c->phi, c->u, c->v, c->w, as * dt, c->scal);
        FZ_LAUNCHED(FZK_CORRECT);
        double *old = c->pp;
        c->pp = c->p;
        c->p = c->pn;
        c->pn = old;
        c->next_stage = (stage + 1) % 3;
        return FIZZY_OK;
    }
    // S4: b = rho0/(a dt) D(u**), FFT x (fused), FFT y, tridiagonal z, inverse
    FZ_TB(FZK_FFTX_FWD);
    FZ_CUDA(fz_fftx_launch(0, c->log2nx, P, nullptr, c->us, c->vs, c->ws, P.rho0 / (as * dt), c->spec, nullptr,
                           c->twx, c->scal, nullptr, c->stream));
    FZ_LAUNCHED(FZK_FFTX_FWD);
    if ((s = run_spectral_solve(c, c->pn)) != FIZZY_OK) return s;
    // S5: correction, pressure rotation
    // (rho1 != rho2: it also forms p_hat = 2 p_new - p for the next substep's predictor, N7)
    // after stages 0 and 1 it is deferred into the first kernel of the next substep (corr_pending)
    if (stage == 2) {
        FZ_TB(FZK_CORRECT);
        k_correct<true><<<grid, block, 0, c->stream>>>(P, c->us, c->vs, c->ws, c->pn, c->u, c->v, c->w,
                                                       as * dt / P.rho0, c->scal, c->p, c->phat);
        FZ_LAUNCHED(FZK_CORRECT);
    } else {
        c->corr_pending = true;
        c->corr_coef = as * dt / P.rho0;
    }
    double *old_pp = c->pp;
    c->pp = c->p;
    c->p = c->pn;
    c->pn = old_pp;
    c->next_stage = (stage + 1) % 3;
    return FIZZY_OK;
}

extern "C" fizzy_status fizzy_diagnostics(fizzy_ctx *c, double *out)
{
    if (!c) return FIZZY_EINVAL;
    FZ_DEVICE();
    if (!out) return fail(c, FIZZY_EINVAL, "out must be non-NULL");
    if (!c->fields_set) return fail(c, FIZZY_ESTATE, "fizzy_set_fields has not been called");
    FZ_FLUSH();
    FZ_TB(FZK_OTHER);
    k_diag<<<FZ_DIAG_BLOCKS, 256, 0, c->stream>>>(c->P, c->u, c->v, c->w, c->phi, c->T, c->dpart);
    FZ_LAUNCHED(FZK_OTHER);
    FZ_TB(FZK_OTHER);
    k_diag_final<<<1, 256, 0, c->stream>>>(c->P, c->dpart, FZ_DIAG_BLOCKS, c->scal + 8);
    FZ_LAUNCHED(FZK_OTHER);
    FZ_CUDA(cudaMemcpyAsync(out, c->scal + 8, 8 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    FZ_CUDA(cudaStreamSynchronize(c->stream));
    return FIZZY_OK;
}

extern "C" fizzy_status fizzy_poisson_solve(fizzy_ctx *c, const double *rhs, double *p)
{
    if (!c) return FIZZY_EINVAL;
    FZ_DEVICE();
    if (!rhs || !p) return fail(c, FIZZY_EINVAL, "rhs and p must be non-NULL");
    FZ_FLUSH();   // c->pn is the scratch of this call
    const FzP &P = c->P;
    const size_t B = (size_t)c->N * sizeof(double);
    FZ_CUDA(cudaMemcpyAsync(c->pn, rhs, B, cudaMemcpyDefault, c->stream));
    FZ_TB(FZK_FFTX_FWD);
    FZ_CUDA(fz_fftx_launch(1, c->log2nx, P, c->pn, nullptr, nullptr, nullptr, 1.0, c->spec, nullptr, c->twx, c->scal,
                           nullptr, c->stream));
    FZ_LAUNCHED(FZK_FFTX_FWD);
    fizzy_status s = run_spectral_solve(c, c->pn);
    if (s != FIZZY_OK) return s;
    FZ_CUDA(cudaMemcpyAsync(p, c->pn, B, cudaMemcpyDefault, c->stream));
    return FIZZY_OK;
}

extern "C" fizzy_status fizzy_check_finite(fizzy_ctx *c, long long *count)
{
    if (!c) return FIZZY_EINVAL;
    FZ_DEVICE();
    if (!count) return fail(c, FIZZY_EINVAL, "count must be non-NULL");
    FZ_FLUSH();
    unsigned long long *cnt = reinterpret_cast<unsigned long long *>(c->scal + 5);
    FZ_CUDA(cudaMemsetAsync(cnt, 0, sizeof(*cnt), c->stream));
    FZ_TB(FZK_OTHER);
    k_count_nonfinite<<<148 * 8, 256, 0, c->stream>>>(c->N, c->u, c->v, c->w, c->p, c->phi, c->heat ? c->T : nullptr, cnt);
    FZ_LAUNCHED(FZK_OTHER);
    unsigned long long h = 0;
    FZ_CUDA(cudaMemcpyAsync(&h, cnt, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    FZ_CUDA(cudaStreamSynchronize(c->stream));
    *count = (long long)h;
    return FIZZY_OK;
}

extern "C" fizzy_status fizzy_stable_dt(fizzy_ctx *c, double cfl, double *dt)
{
    if (!c) return FIZZY_EINVAL;
    FZ_DEVICE();
    if (!dt || !(cfl > 0.0)) return fail(c, FIZZY_EINVAL, "dt must be non-NULL and cfl > 0");
    if (!c->fields_set) return fail(c, FIZZY_ESTATE, "fizzy_set_fields has not been called");
    FZ_FLUSH();
    const FzP &P = c->P;
    FZ_CUDA(cudaMemsetAsync(c->scal + 3, 0, 2 * sizeof(double), c->stream));
    FZ_TB(FZK_OTHER);
    k_dt_reduce<<<148 * 8, 256, 0, c->stream>>>(P, c->u, c->v, c->w, c->scal + 3);
    FZ_LAUNCHED(FZK_OTHER);
    double red[2] = {0.0, 0.0};
    FZ_CUDA(cudaMemcpyAsync(red, c->scal + 3, sizeof(red), cudaMemcpyDeviceToHost, c->stream));
    FZ_CUDA(cudaStreamSynchronize(c->stream));
    // N16: the limits are scalars of the parameters and of the two maxima just reduced on the device
    const double S = 1.0 / (P.dx * P.dx) + 1.0 / (P.dy * P.dy) + 1.0 / (c->dzmin * c->dzmin);
    const double dmin = std::fmin(P.dx, std::fmin(P.dy, c->dzmin));
    const double gam = P.gamma_rel * red[1] + P.gamma_abs;
    const double nu = std::fmax(P.mu1 / P.rho1, P.mu2 / P.rho2);
    double lim = INFINITY;
    if (red[0] > 0.0) lim = std::fmin(lim, 1.0 / red[0]);
    if (nu > 0.0) lim = std::fmin(lim, 1.0 / (2.0 * nu * S));
    if (P.sigma > 0.0) lim = std::fmin(lim, std::sqrt((P.rho1 + P.rho2) * dmin * dmin * dmin / (4.0 * M_PI * P.sigma)));
    if (gam > 0.0) lim = std::fmin(lim, 1.0 / (2.0 * gam * P.eps * S));
    if (P.heat) lim = std::fmin(lim, 1.0 / (2.0 * std::fmax(P.k1 / (P.rho1 * P.cp1), P.k2 / (P.rho2 * P.cp2)) * S));
    *dt = std::isinf(lim) ? 0.0 : cfl * lim;
    return FIZZY_OK;
}

extern "C" fizzy_status fizzy_graph_enable(fizzy_ctx *c, int on)
{
    if (!c) return FIZZY_EINVAL;
    if (on && (c->stream == nullptr || c->stream == cudaStreamLegacy || c->stream == cudaStreamPerThread))
        return fail(c, FIZZY_EINVAL, "CUDA graph capture needs a context created on a non-default stream");
    c->graph_on = on != 0;
    return FIZZY_OK;
}

extern "C" fizzy_status fizzy_rk3_step(fizzy_ctx *c, double dt)
{
    if (!c) return FIZZY_EINVAL;
    FZ_DEVICE();
    if (!(dt > 0.0)) return fail(c, FIZZY_EINVAL, "dt must be > 0");
    if (!c->fields_set) return fail(c, FIZZY_ESTATE, "fizzy_set_fields has not been called");
    if (c->next_stage != 0) return fail(c, FIZZY_ESTATE, "fizzy_rk3_step must start at stage 0");
    fizzy_status s = FIZZY_OK;
    if (!c->graph_on || c->timing || c->solver == 1) {   // plain launches (per-kernel events cannot be recorded into a replayed graph)
        for (int stage = 0; stage < 3 && s == FIZZY_OK; ++stage) s = fizzy_rk3_substep(c, stage, dt);
        return s;
    }
    const int par = c->phi == c->phi0 ? 0 : 1;
    if (!c->gexec[par] || c->gdt[par] != dt || c->gkey[par][0] != c->p || c->gkey[par][1] != c->pp) {   // (re)capture: the kernel arguments bake in dt and the buffer rotation
        if (c->gexec[par]) { cudaGraphExecDestroy(c->gexec[par]); c->gexec[par] = nullptr; }
        // the capture itself executes nothing: remember the buffer rotation, capture, restore, then replay below
        double *sv[] = {c->phi, c->phin, c->p, c->pp, c->pn, c->T, c->Tn};
        const bool sv_pending = c->corr_pending;   // false here (a full step ends with k_correct<true>), and false again
        const double sv_coef = c->corr_coef;       // after three captured substeps; restored for a capture that fails midway
        const long long l0 = c->launches;
        cudaGraph_t g = nullptr;
        FZ_CUDA(cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal));
        for (int stage = 0; stage < 3 && s == FIZZY_OK; ++stage) s = fizzy_rk3_substep(c, stage, dt);
        const cudaError_t ce = cudaStreamEndCapture(c->stream, &g);
        c->glaunches[par] = c->launches - l0;
        c->launches = l0;
        c->phi = sv[0]; c->phin = sv[1]; c->p = sv[2]; c->pp = sv[3]; c->pn = sv[4]; c->T = sv[5]; c->Tn = sv[6];
        c->next_stage = 0;
        c->corr_pending = sv_pending;
        c->corr_coef = sv_coef;
        if (s != FIZZY_OK) { if (g) cudaGraphDestroy(g); return s; }
        if (ce != cudaSuccess) return cuda_fail(c, ce, "cudaStreamEndCapture");
        const cudaError_t ie = cudaGraphInstantiate(&c->gexec[par], g, 0);
        cudaGraphDestroy(g);
        if (ie != cudaSuccess) { c->gexec[par] = nullptr; return cuda_fail(c, ie, "cudaGraphInstantiate"); }
        c->gdt[par] = dt;
        c->gkey[par][0] = c->p;
        c->gkey[par][1] = c->pp;
    }
    FZ_CUDA(cudaGraphLaunch(c->gexec[par], c->stream));
    // the host-side buffer rotation of three substeps: phi and T swap three times, the pressures rotate back
    std::swap(c->phi, c->phin);
    if (c->heat) std::swap(c->T, c->Tn);
    c->launches += c->glaunches[par];
    return FIZZY_OK;
}

// =====================================================================================
// variable-coefficient pressure Poisson problem, multigrid-preconditioned CG (fz_mg.cuh)
namespace {

struct MgPlan {
    int nlev;
    int nx[FZ_MG_MAXLEV], ny[FZ_MG_MAXLEV], nz[FZ_MG_MAXLEV];
    size_t doubles;   // workspace, in doubles
};

// levels halve nx, ny, nz together while all three stay even and the coarse grid keeps >= 4 cells per direction
MgPlan mg_plan(const fizzy_ctx *c)
{
    MgPlan m;
    m.nlev = 1;
    m.nx[0] = c->P.nx; m.ny[0] = c->P.ny; m.nz[0] = c->P.nz;
    while (m.nlev < FZ_MG_MAXLEV) {
        const int q = m.nlev - 1;
        if ((m.nx[q] | m.ny[q] | m.nz[q]) & 1) break;
        if (m.nx[q] < 8 || m.ny[q] < 8 || m.nz[q] < 8) break;
        m.nx[m.nlev] = m.nx[q] / 2; m.ny[m.nlev] = m.ny[q] / 2; m.nz[m.nlev] = m.nz[q] / 2;
        ++m.nlev;
    }
    size_t d = 9 * (size_t)c->N;   // sol, res, d, q | level 0: x, r, bx, by, bz (its b is res)
    for (int q = 1; q < m.nlev; ++q) d += 6 * (size_t)m.nx[q] * m.ny[q] * m.nz[q];
    for (int q = 0; q < m.nlev; ++q) d += 3 * (size_t)m.nz[q] + 32;
    d += FZ_MG_RBLOCKS + 64;
    m.doubles = d + 64 * (size_t)(6 * m.nlev + 16);   // 256-byte alignment slack of every piece
    return m;
}

void mg_grid(const FzMgLevel &L, dim3 &grid, dim3 &block)
{
    block = dim3(32, 8, 1);
    grid = dim3((L.nx + 31) / 32, (L.ny + 7) / 8, L.nz);
}

}  // namespace

extern "C" fizzy_status fizzy_set_pressure_solver(fizzy_ctx *c, int solver, void *dev_work, size_t work_bytes, double rtol,
                                                  int max_iter)
{
    if (!c) return FIZZY_EINVAL;
    FZ_DEVICE();
    if (solver != 0 && solver != 1) return fail(c, FIZZY_EINVAL, "solver must be 0 (splitting) or 1 (variable-coefficient multigrid)");
    FZ_FLUSH();
    if (c->next_stage != 0) return fail(c, FIZZY_ESTATE, "the pressure solver can only be changed between RK3 steps");
    if (solver == 1) {
        if (!dev_work || (reinterpret_cast<uintptr_t>(dev_work) & 255) || !(rtol > 0.0) || max_iter < 1)
            return fail(c, FIZZY_EINVAL, "solver 1 needs 256-byte aligned dev_work, rtol > 0, max_iter >= 1");
        if (work_bytes < mg_plan(c).doubles * sizeof(double)) return fail(c, FIZZY_ENOMEM, "dev_work is smaller than fizzy_varcoef_workspace_bytes");
        c->mg_work = dev_work; c->mg_bytes = work_bytes; c->mg_rtol = rtol; c->mg_maxit = max_iter;
    }
    if (c->solver == 1 && solver == 0 && c->varrho && c->fields_set) {
        // the solver-1 substeps rotate p and p_prev but never write p_hat; the splitting's predictor reads it from
        // c->phat (N7), so form 2 p - p_prev of the current pressures before the first splitting substep
        dim3 grid, block;
        cell_launch(c, grid, block);
        FZ_TB(FZK_OTHER);
        k_phat<<<grid, block, 0, c->stream>>>(c->P, c->p, c->pp, c->phat);
        FZ_LAUNCHED(FZK_OTHER);
    }
    c->solver = solver;
    return FIZZY_OK;
}

extern "C" size_t fizzy_varcoef_workspace_bytes(const fizzy_ctx *c)
{
    return c ? mg_plan(c).doubles * sizeof(double) : 0;
}

extern "C" fizzy_status fizzy_poisson_solve_varcoef(fizzy_ctx *c, const double *rhs, const double *phi, double *p,
                                                    void *dev_work, size_t work_bytes, double rtol, int max_iter,
                                                    int *iters, double *relres)
{
    if (!c) return FIZZY_EINVAL;
    FZ_DEVICE();
    if (!rhs || !p || !dev_work || !(rtol > 0.0) || max_iter < 1) return fail(c, FIZZY_EINVAL, "rhs, p, dev_work must be non-NULL, rtol > 0, max_iter >= 1");
    if (reinterpret_cast<uintptr_t>(dev_work) & 255) return fail(c, FIZZY_EINVAL, "dev_work must be 256-byte aligned");
    const MgPlan plan = mg_plan(c);
    if (work_bytes < plan.doubles * sizeof(double)) return fail(c, FIZZY_ENOMEM, "dev_work is smaller than fizzy_varcoef_workspace_bytes");
    if (!phi && !c->fields_set) return fail(c, FIZZY_ESTATE, "phi == NULL needs fizzy_set_fields first");
    const FzP &P = c->P;
    const int n = (int)c->N;
    cudaStream_t st = c->stream;
    // timing mode: ONE event pair around the whole solve (its kernels are launched from lambdas, outside FZ_TB); the
    // time includes the host round trips of the CG scalars
    FZ_TB(FZK_MG);
    const size_t mg_slot = c->pending.size();   // 0 when timing is off
    Carver cv(dev_work);
    double *sol = cv.dbl(n), *res = cv.dbl(n), *dir = cv.dbl(n), *q = cv.dbl(n);
    FzMgLevel L[FZ_MG_MAXLEV];
    std::vector<double> tab;
    for (int l = 0; l < plan.nlev; ++l) {
        const size_t nl = (size_t)plan.nx[l] * plan.ny[l] * plan.nz[l];
        L[l].nx = plan.nx[l]; L[l].ny = plan.ny[l]; L[l].nz = plan.nz[l]; L[l].z_wall = P.z_wall;
        const double dx = P.dx * (1 << l), dy = P.dy * (1 << l);
        L[l].cx = 1.0 / (dx * dx); L[l].cy = 1.0 / (dy * dy);
        L[l].x = cv.dbl(nl);
        L[l].b = l == 0 ? res : cv.dbl(nl);
        L[l].r = cv.dbl(nl);
        L[l].bx = cv.dbl(nl); L[l].by = cv.dbl(nl); L[l].bz = cv.dbl(nl);
    }
    // 1-D z tables of every level: dzf (sum of the two children), centre spacings from face midpoints (N10)
    // (all levels in one host vector: one copy and one synchronisation instead of one per level)
    std::vector<double> dz = c->hdzf;
    size_t tab_off[FZ_MG_MAXLEV], tab_len = 0;
    for (int l = 0; l < plan.nlev; ++l) { tab_off[l] = tab_len; tab_len += (3 * (size_t)plan.nz[l] + 31) & ~size_t(31); }   // 256-byte pieces
    tab.assign(tab_len, 0.0);
    for (int l = 0; l < plan.nlev; ++l) {
        const int nzl = plan.nz[l];
        if (l > 0) { std::vector<double> cz(nzl); for (int k = 0; k < nzl; ++k) cz[k] = dz[2 * k] + dz[2 * k + 1]; dz.swap(cz); }
        double *t = tab.data() + tab_off[l];
        for (int k = 0; k < nzl; ++k) {
            const int kp = k + 1 == nzl ? 0 : k + 1, km = k == 0 ? nzl - 1 : k - 1;
            const double dzc_p = 0.5 * (dz[k] + dz[kp]), dzc_m = 0.5 * (dz[km] + dz[k]);
            t[k] = dz[k];
            t[nzl + k] = (P.z_wall && k == nzl - 1) ? 0.0 : 1.0 / (dzc_p * dz[k]);
            t[2 * nzl + k] = (P.z_wall && k == 0) ? 0.0 : 1.0 / (dzc_m * dz[k]);
        }
    }
    {
        double *dt = cv.dbl(tab_len);
        FZ_CUDA(cudaMemcpyAsync(dt, tab.data(), tab_len * sizeof(double), cudaMemcpyHostToDevice, st));
        FZ_CUDA(cudaStreamSynchronize(st));   // pageable source: the copy has left the host vector
        for (int l = 0; l < plan.nlev; ++l) {
            const int nzl = plan.nz[l];
            L[l].wz = dt + tab_off[l]; L[l].czh = L[l].wz + nzl; L[l].czl = L[l].wz + 2 * nzl;
        }
    }
    double *partial = cv.dbl(FZ_MG_RBLOCKS), *scalar = cv.dbl(8);
    dim3 grid, block;

    // face coefficients of every level
    const double *dphi = c->phi;
    if (phi) {   // a caller-supplied phase field: stage it in `q` (free until the CG loop)
        FZ_CUDA(cudaMemcpyAsync(q, phi, (size_t)n * sizeof(double), cudaMemcpyDefault, st));
        dphi = q;
    }
    mg_grid(L[0], grid, block);
    k_mg_beta<<<grid, block, 0, st>>>(L[0], dphi, P.rho2, P.drho);
    ++c->launches;
    for (int l = 1; l < plan.nlev; ++l) {
        mg_grid(L[l], grid, block);
        k_mg_coarsen_beta<<<grid, block, 0, st>>>(L[l], L[l - 1]);
        ++c->launches;
    }
    FZ_CUDA(cudaPeekAtLastError());

    const int plane = P.nx * P.ny;
    auto dotw = [&](const double *a, const double *b, double *out) -> cudaError_t {
        k_mg_dot<<<FZ_MG_RBLOCKS, 256, 0, st>>>(a, b, L[0].wz, plane, n, partial);
        k_mg_dot_final<<<1, 256, 0, st>>>(partial, FZ_MG_RBLOCKS, scalar);
        c->launches += 2;
        cudaError_t e = cudaMemcpyAsync(out, scalar, sizeof(double), cudaMemcpyDeviceToHost, st);
        return e == cudaSuccess ? cudaStreamSynchronize(st) : e;
    };
    // flat cells between walls (dx or dy > 1.5 dz_min: the tanh-stretched channel grids): zebra z-line relaxation, exact
    // along z; otherwise red-black points (a line sweep is one thread per column and 3x slower per sweep at 256^3)
    const bool zline = P.z_wall != 0 && std::fmax(P.dx, P.dy) > 1.5 * c->dzmin;
    auto smooth = [&](const FzMgLevel &lev, int sweeps, bool forward) {
        dim3 g2, b2;
        mg_grid(lev, g2, b2);
        for (int s = 0; s < sweeps; ++s) {
            if (zline) {
                const dim3 gl(g2.x, g2.y, 1);
                k_mg_zline<<<gl, b2, 0, st>>>(lev, forward ? 0 : 1);
                k_mg_zline<<<gl, b2, 0, st>>>(lev, forward ? 1 : 0);
            } else {
                k_mg_gs<<<g2, b2, 0, st>>>(lev, forward ? 0 : 1);
                k_mg_gs<<<g2, b2, 0, st>>>(lev, forward ? 1 : 0);
            }
            c->launches += 2;
        }
    };
    // z = V-cycle approximation of A^-1 res, into L[0].x
    auto vcycle = [&]() {
        dim3 g2, b2;
        k_mg_fill<<<FZ_MG_RBLOCKS, 256, 0, st>>>(L[0].x, 0.0, n);
        ++c->launches;
        for (int l = 0; l < plan.nlev - 1; ++l) {
            smooth(L[l], FZ_MG_NU, true);
            mg_grid(L[l], g2, b2);
            k_mg_residual<<<g2, b2, 0, st>>>(L[l]);
            mg_grid(L[l + 1], g2, b2);
            k_mg_restrict<<<g2, b2, 0, st>>>(L[l + 1], L[l]);
            c->launches += 2;
        }
        smooth(L[plan.nlev - 1], FZ_MG_COARSE, true);
        smooth(L[plan.nlev - 1], FZ_MG_COARSE, false);
        for (int l = plan.nlev - 2; l >= 0; --l) {
            mg_grid(L[l], g2, b2);
            k_mg_prolong<<<g2, b2, 0, st>>>(L[l], L[l + 1]);
            ++c->launches;
            smooth(L[l], FZ_MG_NU, false);
        }
    };

    // res = rhs - (dzf-weighted mean of rhs); sol = 0
    FZ_CUDA(cudaMemcpyAsync(res, rhs, (size_t)n * sizeof(double), cudaMemcpyDefault, st));
    double s1 = 0.0, vol = 0.0, bb = 0.0;
    k_mg_fill<<<FZ_MG_RBLOCKS, 256, 0, st>>>(sol, 1.0, n);
    FZ_CUDA(dotw(sol, nullptr, &vol));
    FZ_CUDA(dotw(res, nullptr, &s1));
    k_mg_shift<<<FZ_MG_RBLOCKS, 256, 0, st>>>(res, res, -s1 / vol, n);
    k_mg_fill<<<FZ_MG_RBLOCKS, 256, 0, st>>>(sol, 0.0, n);
    c->launches += 3;
    FZ_CUDA(dotw(res, res, &bb));
    int it = 0;
    double rr = bb;
    if (bb > 0.0) {
        double rz = 0.0, rz_new = 0.0, dq = 0.0;
        vcycle();
        FZ_CUDA(cudaMemcpyAsync(dir, L[0].x, (size_t)n * sizeof(double), cudaMemcpyDeviceToDevice, st));
        FZ_CUDA(dotw(res, L[0].x, &rz));
        mg_grid(L[0], grid, block);
        for (it = 1; it <= max_iter; ++it) {
            k_mg_apply<<<grid, block, 0, st>>>(L[0], dir, q);
            ++c->launches;
            FZ_CUDA(dotw(dir, q, &dq));
            if (!(dq != 0.0) || !std::isfinite(dq)) return fail(c, FIZZY_ECUDA, "fizzy_poisson_solve_varcoef: breakdown (d, A d) = 0 or not finite");
            const double alpha = rz / dq;
            k_mg_axpby<<<FZ_MG_RBLOCKS, 256, 0, st>>>(sol, dir, alpha, 1.0, n);
            k_mg_axpby<<<FZ_MG_RBLOCKS, 256, 0, st>>>(res, q, -alpha, 1.0, n);
            c->launches += 2;
            FZ_CUDA(dotw(res, res, &rr));
            if (rr <= rtol * rtol * bb) break;
            vcycle();
            FZ_CUDA(dotw(res, L[0].x, &rz_new));
            k_mg_axpby<<<FZ_MG_RBLOCKS, 256, 0, st>>>(dir, L[0].x, 1.0, rz_new / rz, n);
            ++c->launches;
            rz = rz_new;
        }
        if (it > max_iter) it = max_iter;
    }
    // gauge N17: remove the dzf-weighted mean, copy out
    FZ_CUDA(dotw(sol, nullptr, &s1));
    k_mg_shift<<<FZ_MG_RBLOCKS, 256, 0, st>>>(sol, sol, -s1 / vol, n);
    ++c->launches;
    FZ_CUDA(cudaPeekAtLastError());
    FZ_CUDA(cudaMemcpyAsync(p, sol, (size_t)n * sizeof(double), cudaMemcpyDefault, st));
    if (c->timing && mg_slot && c->pending[mg_slot - 1].e1) cudaEventRecord(c->pending[mg_slot - 1].e1, st);
    if (iters) *iters = it;
    if (relres) *relres = bb > 0.0 ? std::sqrt(rr / bb) : 0.0;
    return FIZZY_OK;
}
