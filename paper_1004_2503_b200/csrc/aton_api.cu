// C ABI of the ATON hot path (include/aton.h): context, uploads/downloads, source lists, the step
// loop and the diagnostics.  The host only drives; every step of the path runs in
// the kernels of aton_step_v5.cuh (product), aton_step_v4.cuh / aton_step_fused.cuh (fallbacks for grids it cannot tile),
// aton_fixup.cuh, aton_step_hll2.cuh / aton_step_hll.cuh (the HLL flux), aton_step_ref.cuh (cross-checks) and aton_reduce.cuh.
#include "aton_ctx.cuh"
#include "aton_reduce.cuh"
#include "aton_step_fused.cuh"
#include "aton_step_hll.cuh"
#include "aton_step_hll2.cuh"
#include "aton_step_v4.cuh"
#include "aton_step_v5.cuh"

using namespace aton;

namespace aton {
char g_init_error[512] = "";
}

namespace {

int flags_of(const aton_params_t &p) {
    return (p.recomb_case == 0 ? F_CASE_A : 0) | (p.cooling ? F_COOL : 0) | (p.coll_ion ? F_COLL : 0);
}

StepConst make_step_const(const aton_ctx *ctx, double dt) {
    const aton_params_t &p = ctx->p;
    const double kb15 = 1.5 * K_BOLTZ;
    StepConst s{};
    const double h = ctx->c * dt / (2.0 * ctx->dx);
    s.h = (float)h;
    s.keep = (float)(1.0 - 6.0 * h);
    s.dt = (float)dt;
    s.cs = (float)(ctx->c * p.sigma_n);
    s.heat_K = (float)((p.e_photon_eV * p.sigma_e / p.sigma_n - E0_EV) * EV_ERG / kb15);
    s.heat_rate_K = (float)(ctx->c * (p.e_photon_eV * p.sigma_e - E0_EV * p.sigma_n) * EV_ERG / kb15);
    s.l2_zrec0 = (float)std::log2((p.recomb_case == 0 ? 1.778e-29 : 3.435e-30) / kb15);
    s.zff0 = (float)(1.42e-27 / kb15);
    s.zexc0 = (float)(7.5e-19 / kb15);
    s.l2_zci0 = (float)std::log2(E0_EV * EV_ERG * 21.11 / kb15);
    s.zci_over_beta = (float)(E0_EV * EV_ERG / kb15);
    const double zp1 = 1.0 + p.redshift;
    s.compton0 = p.redshift >= 0.0 ? (float)(5.65e-36 * zp1 * zp1 * zp1 * zp1 / kb15) : 0.0f;
    s.t_cmb = (float)(2.726 * zp1);
    s.eps_sub = (float)p.eps_sub;
    s.max_sub = p.max_sub;
    s.clump_model = p.clump_model;
    if (p.clump_model == 1) {
        s.clump_k0 = (float)(p.clump_a - p.clump_b);
        s.clump_k1 = (float)(p.clump_b / ctx->nH_mean);
    } else {
        s.clump_k0 = (float)p.clump_a;
        s.clump_k1 = (float)p.clump_b;
    }
    s.ci_k0 = p.clump_i_a > 0.0 ? (float)p.clump_i_a : 0.0f;
    s.ci_k1 = (float)p.clump_i_b;
    s.inj_scale = 0.0f;
    // when the fp32 sub-cycling hands a cell to the fp64 path (chemistry<.., BAIL>; thresholds measured against the
    // 1-step bar at 256^3 / 512^3 / 1024^3: profiles/r02_b_fixup.md)
    s.stiff_kappa = 1.0f / 64.0f;
    s.stiff_sens = 8.0f;
    s.stiff_nsub = 1 << 30;
    return s;
}

StepConstD make_step_const_d(const aton_ctx *ctx, double dt) {
    const aton_params_t &p = ctx->p;
    const double kb15 = 1.5 * K_BOLTZ;
    StepConstD s{};
    s.dt = dt;
    s.cs = ctx->c * p.sigma_n;
    s.heat_K = (p.e_photon_eV * p.sigma_e / p.sigma_n - E0_EV) * EV_ERG / kb15;
    s.heat_rate_K = ctx->c * (p.e_photon_eV * p.sigma_e - E0_EV * p.sigma_n) * EV_ERG / kb15;
    s.zrec0 = (p.recomb_case == 0 ? 1.778e-29 : 3.435e-30) / kb15;
    s.zff0 = 1.42e-27 / kb15;
    s.zexc0 = 7.5e-19 / kb15;
    s.zci_over_beta = E0_EV * EV_ERG / kb15;
    const double zp1 = 1.0 + p.redshift;
    s.compton0 = p.redshift >= 0.0 ? 5.65e-36 * zp1 * zp1 * zp1 * zp1 / kb15 : 0.0;
    s.t_cmb = 2.726 * zp1;
    s.eps_sub = p.eps_sub;
    s.max_sub = p.max_sub;
    s.clump_model = p.clump_model;
    if (p.clump_model == 1) {
        s.clump_k0 = p.clump_a - p.clump_b;
        s.clump_k1 = p.clump_b / ctx->nH_mean;
    } else {
        s.clump_k0 = p.clump_a;
        s.clump_k1 = p.clump_b;
    }
    s.ci_k0 = p.clump_i_a > 0.0 ? p.clump_i_a : 0.0;
    s.ci_k1 = p.clump_i_b;
    return s;
}

// which fused kernel a step launches: 5 (row-wide warps; nx % 128 == 0, ny % 8 == 0), else 4 (32 x 4 / 64 x 2 warp
// tiles), else 2 (the fallback that tiles anything); variant 0 is the one-thread-per-cell kernel
int step_kernel_of(const aton_ctx *ctx) {
    if (ctx->variant == 0) return 0;
    if (ctx->variant == 5 && v5_pick_w(ctx->g, ctx->tile_y)) return 5;
    if (ctx->variant == 5 && v4_pick_wxq(ctx->g, 0)) return 4;
    if (ctx->variant == 4 && v4_pick_wxq(ctx->g, ctx->tile_y)) return 4;
    return 2;
}

FieldsIO make_io(const aton_ctx *ctx, int cur) {
    FieldsIO f{};
    const int a = cur, b = 1 - cur;
    f.N = ctx->rad[a][0]; f.Gx = ctx->rad[a][1]; f.Gy = ctx->rad[a][2]; f.Gz = ctx->rad[a][3];
    f.N1 = ctx->rad[b][0]; f.Gx1 = ctx->rad[b][1]; f.Gy1 = ctx->rad[b][2]; f.Gz1 = ctx->rad[b][3];
    f.x = ctx->x; f.T = ctx->T; f.nH = ctx->nH;
    f.src_mask = ctx->src_mask; f.src_cell = ctx->src_cell; f.src_rho = ctx->src_rho; f.src_rho_d = ctx->src_rho_d;
    f.n_src = ctx->n_src;
    f.stats = ctx->stats;
    f.defer_mask = ctx->defer_mask;
    f.src_bits = ctx->src_bits;
    f.stiff_q = ctx->stiff_q; f.stiff_n = ctx->stiff_n; f.stiff_cap = ctx->stiff_cap;
    f.fix_inject = step_kernel_of(ctx) >= 4 ? 1 : 0;
    return f;
}

__global__ void write_fixargs_kernel(FixArgs a0, FixArgs a1, FixArgs *dst) { dst[0] = a0; dst[1] = a1; }

// aton_set_timing: an event right before / after the dominant kernel of a step
void time_mark(aton_ctx *ctx) {
    if (!ctx->timing) return;
    cudaEvent_t e;
    if (cudaEventCreate(&e) != cudaSuccess) return;
    cudaEventRecord(e, ctx->stream);
    ctx->ev.push_back(e);
}

void fix_mark(aton_ctx *ctx) {
    if (!ctx->timing) return;
    cudaEvent_t e;
    if (cudaEventCreate(&e) != cudaSuccess) return;
    cudaEventRecord(e, ctx->stream);
    ctx->ev_fix.push_back(e);
}

void stiff_mark(aton_ctx *ctx) {
    if (!ctx->timing) return;
    cudaEvent_t e;
    if (cudaEventCreate(&e) != cudaSuccess) return;
    cudaEventRecord(e, ctx->stream);
    ctx->ev_stiff.push_back(e);
}

template <int FLAGS>
cudaError_t launch_one(aton_ctx *ctx, const FieldsIO &f, int zb, int ze) {
    const StepConst &sc = ctx->sc;
    const StepConstD &scd = ctx->scd;
    // HLL intercell flux: the tiled kernel where a kernel variant 4 / 5 context's grid allows it (nx % 32 == 0,
    // ny % 8 == 0; it shares their second half: mask, fix-up, fp64), else one thread per cell with the chemistry in place
    const bool hll_tiled = ctx->p.flux == 1 && step_kernel_of(ctx) >= 4 && hll_tiled_grid_ok(ctx->g);
    if (ctx->p.flux == 1 && !hll_tiled) {
        if (ctx->slab) return cudaErrorNotSupported;          // checked with a message in aton_init_slab
        const int threads = 256;
        const unsigned blocks = (unsigned)((ctx->nalloc + threads - 1) / threads);
        time_mark(ctx);
        step_hll_kernel<FLAGS><<<blocks, threads, 0, ctx->stream>>>(f, ctx->g, sc, scd);
        time_mark(ctx);
        return cudaGetLastError();
    }
    if (ctx->variant == 0) {
        const int threads = 256;
        const unsigned blocks = (unsigned)((ctx->nalloc + threads - 1) / threads);
        time_mark(ctx);
        step_ref_kernel<FLAGS><<<blocks, threads, 0, ctx->stream>>>(f, ctx->g, sc, scd);
        time_mark(ctx);
        return cudaGetLastError();
    }
    // variant 5 needs nx % 128 == 0 and ny % 8 == 0, variant 4 nx % 32 == 0 and ny % 4 == 0 (or nx % 64 == 0 and
    // ny % 2 == 0); other grids run the variant-2 kernel.  All flag the cells that sub-cycle for step_fixup_kernel;
    // variants 4 and 5 also flag their source cells (the fix-up injects), variant 2 injects in the step kernel.
    const int kern = step_kernel_of(ctx);
    const int wxq4 = kern == 4 ? v4_pick_wxq(ctx->g, ctx->variant == 4 ? ctx->tile_y : 0) : (kern == 5 ? -1 : 0);
    if (ctx->slab && !wxq4) return cudaErrorNotSupported;    // checked with a message in aton_step
    ctx->fast_subcycles += (long long)ctx->plane * (ze - zb);
    cudaError_t e;
    time_mark(ctx);
    if (hll_tiled)      // two cells per thread on the packed forms where nx % 64 == 0, else one
        e = hll_pk_grid_ok(ctx->g) ? launch_step_hll_pk<FLAGS>(f, ctx->g, sc, ctx->stream, zb, ze)
                                   : launch_step_hll_tiled<FLAGS>(f, ctx->g, sc, ctx->stream, zb, ze);
    else if (kern == 5)
        e = launch_step_v5<FLAGS>(f, ctx->g, sc, v5_pick_w(ctx->g, ctx->tile_y), ctx->tile_z, ctx->stream, zb, ze);
    else if (kern == 4)
        e = launch_step_v4<FLAGS>(f, ctx->g, sc, wxq4, ctx->variant == 4 ? ctx->tile_z : 0, ctx->stream, zb, ze);
    else
        e = launch_step_fused<FLAGS>(f, ctx->g, sc, ctx->variant == 2 ? ctx->tile_y : 0, ctx->variant == 2 ? ctx->tile_z : 0,
                                     ctx->stream);
    time_mark(ctx);
    // the second half of a step: cells that sub-cycle (cooling on) and, for variant 4, the source cells
    if (e != cudaSuccess || !((FLAGS & F_COOL) || (wxq4 && ctx->n_src > 0))) return e;
    (void)scd;
    fix_mark(ctx);
    ctx->launches++;
    const bool inline64 = (long)ctx->nalloc <= FIXUP_INLINE64_CELLS;      // small grid: the fp64 redo happens in the fix-up kernel
    e = launch_step_fixup<FLAGS>(ctx->fixargs + ctx->cur, (long)ctx->plane * zb, (long)ctx->plane * ze, inline64, ctx->stream);
    fix_mark(ctx);
    if (e == cudaSuccess && (FLAGS & F_COOL) && !inline64) {   // without cooling nothing sub-cycles: no cell can be stiff
        ctx->launches++;
        stiff_mark(ctx);
        e = launch_step_stiff<FLAGS>(ctx->fixargs + ctx->cur, ctx->stream);
        stiff_mark(ctx);
    }
    return e;
}

cudaError_t launch_step(aton_ctx *ctx, int zb, int ze) {
    const FieldsIO f = make_io(ctx, ctx->cur);
    ctx->launches++;
    switch (flags_of(ctx->p)) {
        case 0: return launch_one<0>(ctx, f, zb, ze);
        case 1: return launch_one<1>(ctx, f, zb, ze);
        case 2: return launch_one<2>(ctx, f, zb, ze);
        case 3: return launch_one<3>(ctx, f, zb, ze);
        case 4: return launch_one<4>(ctx, f, zb, ze);
        case 5: return launch_one<5>(ctx, f, zb, ze);
        case 6: return launch_one<6>(ctx, f, zb, ze);
        default: return launch_one<7>(ctx, f, zb, ze);
    }
}

int scale_into(aton_ctx *ctx, const float *in, float *out, float s) {
    const int nquad = (int)(ctx->ncell / 4);
    const int blocks = std::min((nquad + 255) / 256, 148 * 16);
    scale_kernel<<<blocks, 256, 0, ctx->stream>>>((const float4 *)in, (float4 *)out, s, nquad);
    ctx->launches++;
    CU(ctx, cudaGetLastError());
    return ATON_OK;
}

}  // namespace

namespace aton {

int check_dt(aton_ctx *ctx, double *dt, const char *who) {
    if (!(*dt > 0.0)) *dt = aton_courant_dt(ctx, 0.8);
    const double mu = ctx->c * *dt / ctx->dx;
    if (!(mu <= (1.0 / 3.0) * (1.0 + 1e-12)) || !std::isfinite(mu))
        return fail(ctx, ATON_EINVAL, "%s: c*dt/dx = %g > 1/3 is unstable for the unsplit 3-D LF scheme", who, mu);
    return ATON_OK;
}

// Step constants for dt, and the arguments variant 4's cold paths (v4_fix_drain, step_fixup_kernel, step_stiff_kernel)
// read from global memory: rewritten (stream-ordered, no host synchronisation) only when something they hold changed.
cudaError_t prepare_step(aton_ctx *ctx, double dt) {
    if (!ctx->fix_dirty && ctx->fix_dt == dt) return cudaSuccess;
    if (ctx->step_graph) {             // the captured pair of steps holds the old constants
        cudaGraphExecDestroy(ctx->step_graph);
        ctx->step_graph = nullptr;
    }
    ctx->sc = make_step_const(ctx, dt);
    ctx->scd = make_step_const_d(ctx, dt);
    FixArgs a[2];
    for (int cur = 0; cur < 2; cur++) { a[cur].f = make_io(ctx, cur); a[cur].c = ctx->sc; a[cur].cd = ctx->scd; }
    write_fixargs_kernel<<<1, 1, 0, ctx->stream>>>(a[0], a[1], ctx->fixargs);
    ctx->launches++;
    ctx->fix_dirty = false;
    ctx->fix_dt = dt;
    return cudaGetLastError();
}

cudaError_t launch_step_planes(aton_ctx *ctx, int zb, int ze) { return launch_step(ctx, zb, ze); }

// raw sums of the context's own cells in the order of aton_reduce_sums (include/aton.h)
void sums_from_reduce(aton_ctx *ctx, const double *r, const unsigned long long *st, double *sums) {
    sums[0] = (double)ctx->ncell; sums[1] = r[R_X]; sums[2] = r[R_XM]; sums[3] = r[R_M]; sums[4] = r[R_N];
    sums[5] = r[R_NM]; sums[6] = r[R_T]; sums[7] = r[R_HALF]; sums[8] = r[R_BAD];
    sums[9] = (double)((long long)st[0] + ctx->fast_subcycles); sums[10] = (double)st[2];
    sums[11] = std::sqrt(r[R_F2MAX]); sums[12] = (double)std::max((long long)st[1], ctx->fast_subcycles > 0 ? 1LL : 0LL);
    sums[13] = r[R_NMIN]; sums[14] = (double)st[3];
}

// the diagnostics of PAPER.md:L149 / L303-305 / Eq.15 from (possibly all-reduced) raw sums
void diag_from_sums(const aton_ctx *ctx, const double *s, aton_diag_t *out) {
    const double n = s[0], cs = ctx->c * ctx->p.sigma_n;
    out->x_vol = s[1] / n;
    out->x_mass = s[2] / s[3];
    out->gamma_vol = cs * s[4] / n;
    out->gamma_mass = cs * s[5] / s[3];
    out->photons_total = s[4] * ctx->dx * ctx->dx * ctx->dx;
    out->T_vol = s[6] / n;
    out->f_max = s[11];
    out->N_min = s[13];
    out->frac_x_half = s[7] / n;
    out->n_nonfinite = (long long)s[8];
    out->subcycles_total = (long long)s[9];
    out->subcycles_max = (long long)s[12];
    out->cells_subcycled = (long long)s[10];
    out->cells_fp64 = (long long)s[14];
    out->steps_done = ctx->steps_done;
    out->time_s = ctx->time_s;
}

// run the two-pass reduction; host_out[R_COUNT]
int run_reduce(aton_ctx *ctx, bool full, double *host_out) {
    const int nquad = (int)(ctx->ncell / 4);
    const int blocks = std::min((nquad + 255) / 256, REDUCE_BLOCKS);
    float **r = ctx->rad[ctx->cur];
    const size_t o = ctx->off;             // the slab's own planes start one plane in
    reduce_pass1<<<blocks, 256, 0, ctx->stream>>>(
        full ? (const float4 *)(r[0] + o) : nullptr, (const float4 *)(r[1] + o), (const float4 *)(r[2] + o),
        (const float4 *)(r[3] + o), (const float4 *)(ctx->x + o), (const float4 *)(ctx->T + o),
        (const float4 *)(ctx->nH + o), nquad, ctx->partials);
    CU(ctx, cudaGetLastError());
    double *out = ctx->partials + (size_t)REDUCE_BLOCKS * R_COUNT;
    reduce_pass2<<<1, 32, 0, ctx->stream>>>(ctx->partials, blocks, out);
    CU(ctx, cudaGetLastError());
    ctx->launches += 2;
    CU(ctx, cudaMemcpyAsync(host_out, out, sizeof(double) * R_COUNT, cudaMemcpyDeviceToHost, ctx->stream));
    CU(ctx, cudaStreamSynchronize(ctx->stream));
    return ATON_OK;
}

}  // namespace aton

extern "C" {

static int init_common(aton_t **out, const aton_grid_t *grid, const aton_box_t *box, const aton_params_t *params,
                       void *cuda_stream, bool slab, int z_begin, int nz_local) {
    if (out) *out = nullptr;
    if (!out || !grid || !box || !params) return fail(nullptr, ATON_EINVAL, "aton_init: NULL argument");
    if (grid->nx < 4 || grid->nx % 4 != 0 || grid->ny < 1 || grid->nz < 1)
        return fail(nullptr, ATON_EINVAL, "aton_init: need nx %% 4 == 0, nx >= 4, ny, nz >= 1 (got %d %d %d)",
                    grid->nx, grid->ny, grid->nz);
    if (slab && (z_begin < 0 || nz_local < 1 || z_begin + nz_local > grid->nz))
        return fail(nullptr, ATON_EINVAL, "aton_init_slab: planes [%d, %d) are not inside nz = %d", z_begin,
                    z_begin + nz_local, grid->nz);
    if (slab && !v4_grid_ok(Grid{grid->nx, grid->ny, nz_local + 2}))
        return fail(nullptr, ATON_EINVAL, "aton_init_slab: needs nx %% 32 == 0 and ny %% 4 == 0 (kernel variant 4)");
    const int nz_own = slab ? nz_local : grid->nz, nz_alloc = slab ? nz_local + 2 : grid->nz;
    const double nalloc_d = (double)grid->nx * grid->ny * nz_alloc;
    if (nalloc_d >= 2147483648.0) return fail(nullptr, ATON_EINVAL, "aton_init: nx*ny*nz must be < 2^31");
    if (!(box->lx_cm > 0.0)) return fail(nullptr, ATON_EINVAL, "aton_init: lx_cm must be > 0");
    if (!(params->sigma_n > 0.0) || !(params->sigma_e > 0.0) || !(params->e_photon_eV > 0.0))
        return fail(nullptr, ATON_EINVAL, "aton_init: sigma_n, sigma_e, e_photon_eV must be > 0");
    if (params->clump_model < 0 || params->clump_model > 2 || params->c_cm_s < 0.0 || params->eps_sub < 0.0 ||
        params->max_sub < 0 || params->flux < 0 || params->flux > 1)
        return fail(nullptr, ATON_EINVAL, "aton_init: bad clump_model / c / eps_sub / max_sub / flux");
    if (slab && params->flux != 0 && !(grid->nx % 32 == 0 && grid->ny % 8 == 0))
        return fail(nullptr, ATON_EINVAL, "aton_init_slab: the HLL flux on a slab needs nx %% 32 == 0 and ny %% 8 == 0 (the tiled kernels)");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(nullptr, ATON_ECUDA, "aton_init: no CUDA device (there is no CPU fallback)");
    }
    aton_ctx *ctx = new (std::nothrow) aton_ctx();
    if (!ctx) return fail(nullptr, ATON_ENOMEM, "aton_init: host allocation failed");
    ctx->g = Grid{grid->nx, grid->ny, nz_alloc};
    ctx->plane = (size_t)grid->nx * grid->ny;
    ctx->ncell = ctx->plane * nz_own;
    ctx->nalloc = (size_t)nalloc_d;
    ctx->slab = slab;
    ctx->off = slab ? ctx->plane : 0;
    ctx->z_begin = slab ? z_begin : 0;
    ctx->nz_local = nz_own;
    ctx->nz_global = grid->nz;
    ctx->p = *params;
    ctx->c = params->c_cm_s > 0.0 ? params->c_cm_s : 2.99792458e10;
    if (ctx->p.eps_sub == 0.0) ctx->p.eps_sub = 0.1;
    if (ctx->p.max_sub == 0) ctx->p.max_sub = 1 << 14;
    ctx->dx = box->lx_cm / grid->nx;
    ctx->stream = (cudaStream_t)cuda_stream;
    cudaGetDevice(&ctx->device);
    const size_t bytes = ctx->nalloc * sizeof(float);
    cudaError_t e = cudaSuccess;
    float **slots[11] = {&ctx->rad[0][0], &ctx->rad[0][1], &ctx->rad[0][2], &ctx->rad[0][3], &ctx->rad[1][0],
                         &ctx->rad[1][1], &ctx->rad[1][2], &ctx->rad[1][3], &ctx->x, &ctx->T, &ctx->nH};
    for (int i = 0; i < 11 && e == cudaSuccess; i++) e = cudaMalloc((void **)slots[i], bytes);
    for (int i = 0; i < 11 && e == cudaSuccess && slab; i++) e = cudaMemsetAsync(*slots[i], 0, bytes, ctx->stream);
    if (e == cudaSuccess) e = cudaMalloc((void **)&ctx->stats, N_STATS * sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMalloc((void **)&ctx->partials, sizeof(double) * (REDUCE_BLOCKS + 1) * R_COUNT);
    if (e == cudaSuccess) e = cudaMalloc((void **)&ctx->src_mask, sizeof(unsigned) * (ctx->nalloc / 1024 + 1));
    const size_t defer_bytes = sizeof(unsigned) * (ctx->nalloc / 32 + 1);
    if (e == cudaSuccess) e = cudaMalloc((void **)&ctx->defer_mask, defer_bytes);
    if (e == cudaSuccess) e = cudaMemsetAsync(ctx->defer_mask, 0, defer_bytes, ctx->stream);
    ctx->stiff_cap = (unsigned)std::max<size_t>(ctx->nalloc / 16, 4096);
    if (e == cudaSuccess) e = cudaMalloc((void **)&ctx->stiff_q, sizeof(int) * (size_t)ctx->stiff_cap);
    if (e == cudaSuccess) e = cudaMalloc((void **)&ctx->stiff_n, 4 * sizeof(unsigned));
    if (e == cudaSuccess) e = cudaMemsetAsync(ctx->stiff_n, 0, 4 * sizeof(unsigned), ctx->stream);
    if (e == cudaSuccess) e = cudaMalloc((void **)&ctx->fixargs, 2 * sizeof(FixArgs));
    if (e == cudaSuccess) e = cudaMalloc((void **)&ctx->src_bits, defer_bytes);
    if (e == cudaSuccess) e = cudaMemsetAsync(ctx->src_bits, 0, defer_bytes, ctx->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(ctx->stats, 0, N_STATS * sizeof(unsigned long long), ctx->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(ctx->src_mask, 0, sizeof(unsigned) * (ctx->nalloc / 1024 + 1), ctx->stream);
    if (e != cudaSuccess) {
        int code = fail(nullptr, e == cudaErrorMemoryAllocation ? ATON_ENOMEM : ATON_ECUDA,
                        "aton_init: device allocation failed: %s", cudaGetErrorString(e));
        cudaGetLastError();
        aton_free(ctx);
        return code;
    }
    *out = ctx;
    return ATON_OK;
}

int aton_init(aton_t **out, const aton_grid_t *grid, const aton_box_t *box, const aton_params_t *params,
              void *cuda_stream) {
    return init_common(out, grid, box, params, cuda_stream, false, 0, 0);
}

int aton_init_slab(aton_t **out, const aton_grid_t *global_grid, const aton_box_t *box, const aton_params_t *params,
                   void *cuda_stream, int z_begin, int nz_local) {
    return init_common(out, global_grid, box, params, cuda_stream, true, z_begin, nz_local);
}

void aton_free(aton_t *ctx) {
    if (!ctx) return;
    cudaSetDevice(ctx->device);
    slab_comm_free(ctx);
    if (ctx->step_graph) cudaGraphExecDestroy(ctx->step_graph);
    for (cudaEvent_t e : ctx->ev) cudaEventDestroy(e);
    for (cudaEvent_t e : ctx->ev_fix) cudaEventDestroy(e);
    for (cudaEvent_t e : ctx->ev_stiff) cudaEventDestroy(e);
    for (int b = 0; b < 2; b++)
        for (int v = 0; v < 4; v++) cudaFree(ctx->rad[b][v]);
    cudaFree(ctx->x); cudaFree(ctx->T); cudaFree(ctx->nH);
    cudaFree(ctx->src_mask); cudaFree(ctx->src_cell); cudaFree(ctx->src_rho); cudaFree(ctx->src_rho_d);
    cudaFree(ctx->stiff_q); cudaFree(ctx->stiff_n); cudaFree(ctx->fixargs);
    cudaFree(ctx->stats); cudaFree(ctx->partials); cudaFree(ctx->defer_mask); cudaFree(ctx->src_bits);
    delete ctx;
}

const char *aton_last_error(const aton_t *ctx) { return ctx ? ctx->err : g_init_error; }

long long aton_launch_count(const aton_t *ctx) { return ctx ? ctx->launches : 0; }

int aton_set_kernel(aton_t *ctx, int variant, int tile_y, int tile_z) {
    if (!ctx) return ATON_EINVAL;
    if (variant != 0 && variant != 2 && variant != 4 && variant != 5)
        return fail(ctx, ATON_EINVAL, "aton_set_kernel: variant must be 0, 2, 4 or 5");
    if ((variant == 2 && !fused_shape_ok(tile_y, tile_z)) || (variant == 4 && !v4_shape_ok(tile_y, tile_z)) ||
        (variant == 5 && !v5_shape_ok(tile_y, tile_z)))
        return fail(ctx, ATON_EINVAL, "aton_set_kernel: unsupported tile shape %d x %d", tile_y, tile_z);
    ctx->variant = variant; ctx->tile_y = tile_y; ctx->tile_z = tile_z;
    ctx->fix_dirty = true;
    return ATON_OK;
}

int aton_set_timing(aton_t *ctx, int on) {
    if (!ctx) return ATON_EINVAL;
    for (cudaEvent_t e : ctx->ev) cudaEventDestroy(e);
    for (cudaEvent_t e : ctx->ev_fix) cudaEventDestroy(e);
    for (cudaEvent_t e : ctx->ev_stiff) cudaEventDestroy(e);
    ctx->ev.clear();
    ctx->ev_fix.clear();
    ctx->ev_stiff.clear();
    ctx->timing = on != 0;
    return ATON_OK;
}

int aton_kernel_time(aton_t *ctx, double *ms_total, long long *n_launches) {
    if (!ctx || !ms_total || !n_launches) return ATON_EINVAL;
    CU(ctx, cudaStreamSynchronize(ctx->stream));
    double tot = 0.0;
    for (size_t i = 0; i + 1 < ctx->ev.size(); i += 2) {
        float ms = 0.0f;
        CU(ctx, cudaEventElapsedTime(&ms, ctx->ev[i], ctx->ev[i + 1]));
        tot += ms;
    }
    *ms_total = tot;
    *n_launches = (long long)(ctx->ev.size() / 2);
    return ATON_OK;
}

int aton_fixup_time(aton_t *ctx, double *ms_fixup, double *ms_stiff, long long *n_launches) {
    if (!ctx || !ms_fixup || !ms_stiff || !n_launches) return ATON_EINVAL;
    CU(ctx, cudaStreamSynchronize(ctx->stream));
    double tot[2] = {0.0, 0.0};
    const std::vector<cudaEvent_t> *lists[2] = {&ctx->ev_fix, &ctx->ev_stiff};
    for (int k = 0; k < 2; k++)
        for (size_t i = 0; i + 1 < lists[k]->size(); i += 2) {
            float ms = 0.0f;
            CU(ctx, cudaEventElapsedTime(&ms, (*lists[k])[i], (*lists[k])[i + 1]));
            tot[k] += ms;
        }
    *ms_fixup = tot[0];
    *ms_stiff = tot[1];
    *n_launches = (long long)(ctx->ev_fix.size() / 2);
    return ATON_OK;
}

int aton_set_fields(aton_t *ctx, const float *nH, const float *x, const float *T, const float *N, const float *Fx,
                    const float *Fy, const float *Fz, int on_device) {
    if (!ctx) return ATON_EINVAL;
    if (!nH || !x || !T) return fail(ctx, ATON_EINVAL, "aton_set_fields: nH, x and T are required");
    const size_t bytes = ctx->ncell * sizeof(float);
    const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    ctx->have_fields = false;
    ctx->halo_valid = false;
    ctx->cur = 0;
    const size_t o = ctx->off;             // a slab's own planes start one (ghost) plane in
    CU(ctx, cudaMemcpyAsync(ctx->nH + o, nH, bytes, kind, ctx->stream));
    CU(ctx, cudaMemcpyAsync(ctx->x + o, x, bytes, kind, ctx->stream));
    CU(ctx, cudaMemcpyAsync(ctx->T + o, T, bytes, kind, ctx->stream));
    const float *rad_in[4] = {N, Fx, Fy, Fz};
    const float inv_c = (float)(1.0 / ctx->c);
    for (int v = 0; v < 4; v++) {
        float *dst = ctx->rad[0][v] + o;
        if (ctx->slab) CU(ctx, cudaMemsetAsync(ctx->rad[0][v], 0, ctx->nalloc * sizeof(float), ctx->stream));
        if (!rad_in[v]) {
            CU(ctx, cudaMemsetAsync(dst, 0, bytes, ctx->stream));
        } else {
            CU(ctx, cudaMemcpyAsync(dst, rad_in[v], bytes, kind, ctx->stream));
            if (v > 0) {   // the device carries G = F/c
                int rc = scale_into(ctx, dst, dst, inv_c);
                if (rc) return rc;
            }
        }
    }
    CU(ctx, cudaMemsetAsync(ctx->stats, 0, N_STATS * sizeof(unsigned long long), ctx->stream));
    double red[R_COUNT];
    int rc = run_reduce(ctx, false, red);
    if (rc) return rc;
    if (!(red[R_NHMIN] > 0.0) || !std::isfinite(red[R_M]))
        return fail(ctx, ATON_EINVAL, "aton_set_fields: n_H must be finite and > 0 everywhere (min %g)", red[R_NHMIN]);
    if (!ctx->mean_set) ctx->nH_mean = red[R_M] / (double)ctx->ncell;
    ctx->fix_dirty = true;
    CU(ctx, cudaMemsetAsync(ctx->stiff_n, 0, 4 * sizeof(unsigned), ctx->stream));
    ctx->steps_done = 0;
    ctx->fast_subcycles = 0;
    ctx->time_s = 0.0;
    ctx->have_fields = true;
    return ATON_OK;
}

int aton_set_sources(aton_t *ctx, long long n, const float *pos, const double *rate, int on_device) {
    if (!ctx) return ATON_EINVAL;
    if (n < 0 || (n > 0 && (!pos || !rate))) return fail(ctx, ATON_EINVAL, "aton_set_sources: bad arguments");
    std::vector<float> hpos;
    std::vector<double> hrate;
    if (n > 0 && on_device) {
        hpos.resize(3 * n); hrate.resize(n);
        CU(ctx, cudaMemcpyAsync(hpos.data(), pos, sizeof(float) * 3 * n, cudaMemcpyDeviceToHost, ctx->stream));
        CU(ctx, cudaMemcpyAsync(hrate.data(), rate, sizeof(double) * n, cudaMemcpyDeviceToHost, ctx->stream));
        CU(ctx, cudaStreamSynchronize(ctx->stream));
        pos = hpos.data(); rate = hrate.data();
    }
    // NGP binning: cell = floor(pos*n) mod n; merge sources sharing a cell (fp64)
    std::vector<std::pair<int, double>> cells;
    cells.reserve((size_t)n);
    const int dims[3] = {ctx->g.nx, ctx->g.ny, ctx->nz_global};     // positions refer to the global box
    for (long long s = 0; s < n; s++) {
        int ijk[3];
        for (int a = 0; a < 3; a++) {
            const double q = (double)pos[3 * s + a];
            if (!(q >= 0.0 && q <= 1.0)) return fail(ctx, ATON_EINVAL, "aton_set_sources: position %lld outside [0,1]", s);
            long long v = (long long)std::floor(q * dims[a]);
            ijk[a] = (int)(v % dims[a]);
        }
        if (!(rate[s] >= 0.0) || !std::isfinite(rate[s]))
            return fail(ctx, ATON_EINVAL, "aton_set_sources: rate %lld must be finite and >= 0", s);
        int k = ijk[2];
        if (ctx->slab) {       // keep the sources of this slab; local plane index counts the ghost plane below
            if (k < ctx->z_begin || k >= ctx->z_begin + ctx->nz_local) continue;
            k = k - ctx->z_begin + 1;
        }
        cells.push_back({ijk[0] + ctx->g.nx * (ijk[1] + ctx->g.ny * k), rate[s]});
    }
    std::stable_sort(cells.begin(), cells.end(), [](const auto &a, const auto &b) { return a.first < b.first; });
    std::vector<int> ucell;
    std::vector<double> urate;
    for (const auto &cr : cells) {
        if (!ucell.empty() && ucell.back() == cr.first) urate.back() += cr.second;
        else { ucell.push_back(cr.first); urate.push_back(cr.second); }
    }
    const size_t nu = ucell.size();
    const size_t nwords = ctx->nalloc / 1024 + 1;
    std::vector<unsigned> mask(nwords, 0u);
    std::vector<float> rho(nu);
    std::vector<double> rho_d(nu);
    const double inv_vol = 1.0 / (ctx->dx * ctx->dx * ctx->dx);
    for (size_t s = 0; s < nu; s++) {
        const unsigned seg = (unsigned)ucell[s] >> 5;
        mask[seg >> 5] |= 1u << (seg & 31);
        rho_d[s] = urate[s] * inv_vol;
        rho[s] = (float)rho_d[s];
    }
    CU(ctx, cudaStreamSynchronize(ctx->stream));
    cudaFree(ctx->src_cell); cudaFree(ctx->src_rho); cudaFree(ctx->src_rho_d);
    ctx->src_cell = nullptr; ctx->src_rho = nullptr; ctx->src_rho_d = nullptr; ctx->n_src = 0;
    ctx->fix_dirty = true;
    CU(ctx, cudaMemcpyAsync(ctx->src_mask, mask.data(), sizeof(unsigned) * nwords, cudaMemcpyHostToDevice, ctx->stream));
    CU(ctx, cudaMemsetAsync(ctx->src_bits, 0, sizeof(unsigned) * (ctx->nalloc / 32 + 1), ctx->stream));
    if (nu > 0) {
        CU(ctx, cudaMalloc((void **)&ctx->src_cell, sizeof(int) * nu));
        CU(ctx, cudaMalloc((void **)&ctx->src_rho, sizeof(float) * nu));
        CU(ctx, cudaMalloc((void **)&ctx->src_rho_d, sizeof(double) * nu));
        CU(ctx, cudaMemcpyAsync(ctx->src_rho_d, rho_d.data(), sizeof(double) * nu, cudaMemcpyHostToDevice, ctx->stream));
        CU(ctx, cudaMemcpyAsync(ctx->src_cell, ucell.data(), sizeof(int) * nu, cudaMemcpyHostToDevice, ctx->stream));
        CU(ctx, cudaMemcpyAsync(ctx->src_rho, rho.data(), sizeof(float) * nu, cudaMemcpyHostToDevice, ctx->stream));
        source_bits_kernel<<<(unsigned)((nu + 255) / 256), 256, 0, ctx->stream>>>(ctx->src_cell, (int)nu, ctx->src_bits);
        ctx->launches++;
        CU(ctx, cudaGetLastError());
    }
    CU(ctx, cudaStreamSynchronize(ctx->stream));
    ctx->n_src = (int)nu;
    return ATON_OK;
}

double aton_courant_dt(const aton_t *ctx, double courant) {
    if (!ctx) return -1.0;
    return courant * ctx->dx / (3.0 * ctx->c);
}

int aton_step(aton_t *ctx, double dt, int n_steps) {
    if (!ctx) return ATON_EINVAL;
    if (!ctx->have_fields) return fail(ctx, ATON_ESTATE, "aton_step: call aton_set_fields first");
    if (n_steps < 0) return fail(ctx, ATON_EINVAL, "aton_step: n_steps < 0");
    if (int rc = check_dt(ctx, &dt, "aton_step")) return rc;
    if (ctx->slab && ctx->variant != 4 && ctx->variant != 5)
        return fail(ctx, ATON_ESTATE, "aton_step: a slab context runs kernel variants 4 and 5 only");
    if (ctx->slab && n_steps > 1)
        return fail(ctx, ATON_EINVAL, "aton_step: a slab context advances one step per call (exchange the halo planes first, or use aton_step_slab)");
    if (n_steps > 0) CU(ctx, prepare_step(ctx, dt));
    const int zb = ctx->slab ? 1 : 0, ze = ctx->slab ? ctx->nz_local + 1 : ctx->g.nz;
    int s = 0;
    // Small grids (configs 1-2) are launch bound: three launches per step, each a few microseconds of work (SURVEY
    // 3(iii), H7).  Capture one ping-pong pair of steps in a CUDA graph once and replay it.
    if (!ctx->slab && !ctx->timing && !ctx->graph_failed && ctx->ncell <= ((size_t)1 << 22) && n_steps >= 4) {
        if (ctx->cur == 1) {           // the captured pair starts from buffer 0
            CU(ctx, launch_step_planes(ctx, zb, ze));
            ctx->cur = 0; ctx->steps_done++; ctx->time_s += dt; s++;
        }
        if (!ctx->step_graph) {
            const long long l0 = ctx->launches, f0 = ctx->fast_subcycles;
            cudaGraph_t graph = nullptr;
            cudaError_t e = cudaStreamBeginCapture(ctx->stream, cudaStreamCaptureModeThreadLocal);
            if (e == cudaSuccess) {
                e = launch_step_planes(ctx, zb, ze);
                ctx->cur = 1;
                if (e == cudaSuccess) e = launch_step_planes(ctx, zb, ze);
                ctx->cur = 0;
                const cudaError_t e2 = cudaStreamEndCapture(ctx->stream, &graph);
                if (e == cudaSuccess) e = e2;
            }
            if (e == cudaSuccess) e = cudaGraphInstantiate(&ctx->step_graph, graph, 0);
            if (graph) cudaGraphDestroy(graph);
            ctx->graph_launches = ctx->launches - l0;
            ctx->graph_fast = ctx->fast_subcycles - f0;
            ctx->launches = l0;            // capturing launched nothing
            ctx->fast_subcycles = f0;
            if (e != cudaSuccess) {
                cudaGetLastError();
                ctx->step_graph = nullptr;
                ctx->graph_failed = true;
            }
        }
        while (ctx->step_graph && n_steps - s >= 2) {
            CU(ctx, cudaGraphLaunch(ctx->step_graph, ctx->stream));
            ctx->launches += ctx->graph_launches;
            ctx->fast_subcycles += ctx->graph_fast;
            ctx->steps_done += 2;
            ctx->time_s += 2 * dt;
            s += 2;
        }
    }
    for (; s < n_steps; s++) {
        CU(ctx, launch_step_planes(ctx, zb, ze));
        ctx->cur = 1 - ctx->cur;
        ctx->steps_done++;
        ctx->time_s += dt;
    }
    ctx->halo_valid = false;
    return ATON_OK;
}

int aton_set_mean_density(aton_t *ctx, double nH_mean) {
    if (!ctx) return ATON_EINVAL;
    if (!(nH_mean > 0.0) || !std::isfinite(nH_mean)) return fail(ctx, ATON_EINVAL, "aton_set_mean_density: must be > 0");
    ctx->nH_mean = nH_mean;
    ctx->mean_set = true;
    ctx->fix_dirty = true;
    return ATON_OK;
}

// halo planes of a slab: [4 fields][ny][nx] each, fields in the order N, Gx, Gy, Gz (G = F/c, as carried)
int aton_halo_pack(aton_t *ctx, float *send_lo, float *send_hi) {
    if (!ctx || !send_lo || !send_hi) return ATON_EINVAL;
    if (!ctx->slab) return fail(ctx, ATON_ESTATE, "aton_halo_pack: not a slab context");
    if (!ctx->have_fields) return fail(ctx, ATON_ESTATE, "aton_halo_pack: no fields set");
    const size_t pb = ctx->plane * sizeof(float);
    for (int v = 0; v < 4; v++) {
        const float *a = ctx->rad[ctx->cur][v];
        CU(ctx, cudaMemcpyAsync(send_lo + v * ctx->plane, a + ctx->plane, pb, cudaMemcpyDeviceToDevice, ctx->stream));
        CU(ctx, cudaMemcpyAsync(send_hi + v * ctx->plane, a + (size_t)ctx->nz_local * ctx->plane, pb,
                                cudaMemcpyDeviceToDevice, ctx->stream));
    }
    return ATON_OK;
}

int aton_halo_unpack(aton_t *ctx, const float *recv_lo, const float *recv_hi) {
    if (!ctx || !recv_lo || !recv_hi) return ATON_EINVAL;
    if (!ctx->slab) return fail(ctx, ATON_ESTATE, "aton_halo_unpack: not a slab context");
    if (!ctx->have_fields) return fail(ctx, ATON_ESTATE, "aton_halo_unpack: no fields set");
    const size_t pb = ctx->plane * sizeof(float);
    for (int v = 0; v < 4; v++) {
        float *a = ctx->rad[ctx->cur][v];
        CU(ctx, cudaMemcpyAsync(a, recv_lo + v * ctx->plane, pb, cudaMemcpyDeviceToDevice, ctx->stream));
        CU(ctx, cudaMemcpyAsync(a + (size_t)(ctx->nz_local + 1) * ctx->plane, recv_hi + v * ctx->plane, pb,
                                cudaMemcpyDeviceToDevice, ctx->stream));
    }
    return ATON_OK;
}

int aton_reduce_sums(aton_t *ctx, double *sums, int n) {
    if (!ctx || !sums) return ATON_EINVAL;
    if (n != ATON_NSUMS) return fail(ctx, ATON_EINVAL, "aton_reduce_sums: n must be ATON_NSUMS (%d)", ATON_NSUMS);
    if (!ctx->have_fields) return fail(ctx, ATON_ESTATE, "aton_reduce_sums: no fields set");
    double r[R_COUNT];
    int rc = run_reduce(ctx, true, r);
    if (rc) return rc;
    unsigned long long st[N_STATS];
    CU(ctx, cudaMemcpyAsync(st, ctx->stats, sizeof(st), cudaMemcpyDeviceToHost, ctx->stream));
    CU(ctx, cudaStreamSynchronize(ctx->stream));
    sums_from_reduce(ctx, r, st, sums);
    return ATON_OK;
}

int aton_diag_from_sums(aton_t *ctx, const double *sums, int n, aton_diag_t *out) {
    if (!ctx || !sums || !out) return ATON_EINVAL;
    if (n != ATON_NSUMS) return fail(ctx, ATON_EINVAL, "aton_diag_from_sums: n must be ATON_NSUMS (%d)", ATON_NSUMS);
    if (!(sums[0] > 0.0) || !(sums[3] > 0.0)) return fail(ctx, ATON_EINVAL, "aton_diag_from_sums: no cells / no mass in the sums");
    diag_from_sums(ctx, sums, out);
    return ATON_OK;
}

int aton_set_mean_from_sums(aton_t *ctx, const double *sums, int n) {
    if (!ctx || !sums) return ATON_EINVAL;
    if (n != ATON_NSUMS) return fail(ctx, ATON_EINVAL, "aton_set_mean_from_sums: n must be ATON_NSUMS (%d)", ATON_NSUMS);
    if (!(sums[0] > 0.0)) return fail(ctx, ATON_EINVAL, "aton_set_mean_from_sums: no cells in the sums");
    return aton_set_mean_density(ctx, sums[3] / sums[0]);
}

int aton_get_fields(aton_t *ctx, float *nH, float *x, float *T, float *N, float *Fx, float *Fy, float *Fz,
                    int on_device) {
    if (!ctx) return ATON_EINVAL;
    if (!ctx->have_fields) return fail(ctx, ATON_ESTATE, "aton_get_fields: no fields set");
    const size_t bytes = ctx->ncell * sizeof(float);
    const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    const size_t o = ctx->off;
    if (nH) CU(ctx, cudaMemcpyAsync(nH, ctx->nH + o, bytes, kind, ctx->stream));
    if (x) CU(ctx, cudaMemcpyAsync(x, ctx->x + o, bytes, kind, ctx->stream));
    if (T) CU(ctx, cudaMemcpyAsync(T, ctx->T + o, bytes, kind, ctx->stream));
    if (N) CU(ctx, cudaMemcpyAsync(N, ctx->rad[ctx->cur][0] + o, bytes, kind, ctx->stream));
    float *outs[3] = {Fx, Fy, Fz};
    for (int v = 0; v < 3; v++) {
        if (!outs[v]) continue;
        const float *G = ctx->rad[ctx->cur][1 + v] + o;
        if (on_device) {
            int rc = scale_into(ctx, G, outs[v], (float)ctx->c);
            if (rc) return rc;
        } else {   // F = c G staged in the idle ping-pong buffer
            float *stage = ctx->rad[1 - ctx->cur][1 + v] + o;
            int rc = scale_into(ctx, G, stage, (float)ctx->c);
            if (rc) return rc;
            CU(ctx, cudaMemcpyAsync(outs[v], stage, bytes, kind, ctx->stream));
        }
    }
    CU(ctx, cudaStreamSynchronize(ctx->stream));
    return ATON_OK;
}

int aton_reduce(aton_t *ctx, aton_diag_t *out) {
    if (!ctx || !out) return ATON_EINVAL;
    double sums[ATON_NSUMS];
    int rc = aton_reduce_sums(ctx, sums, ATON_NSUMS);
    if (rc) return rc;
    diag_from_sums(ctx, sums, out);
    return ATON_OK;
}

}  // extern "C"
