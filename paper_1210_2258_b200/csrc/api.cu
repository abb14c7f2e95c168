// api.cu -- the C ABI of include/sgp.h: argument checks, plan life cycle, one-shot and host-pointer wrappers.
#include <new>
#include "plan.cuh"

namespace sgpk {

thread_local std::string g_last_cuda_error;

int validate_options(const sgp_options *o)
{
    if (!o) return SGP_ERR_ARG;
    if (!(o->beta > 0 && o->beta < 1 && o->theta > 0 && o->theta < 1)) return SGP_ERR_ARG;
    if (!(o->alpha_min > 0 && o->alpha_min < o->alpha_max)) return SGP_ERR_ARG;
    if (!(o->alpha0 > 0) || !(o->tau1 > 0)) return SGP_ERR_ARG;
    if (o->m_alpha < 1 || o->m_alpha > SGP_MAX_MALPHA) return SGP_ERR_ARG;
    if (o->armijo_memory < 1 || o->armijo_memory > SGP_MAX_ARMIJO_MEMORY) return SGP_ERR_ARG;
    if (o->max_iter < 0 || o->max_backtracks < 0 || o->alt_start < 0) return SGP_ERR_ARG;
    if (!o->adaptive_L && !(o->L1 > 0 && o->L1 < o->L2)) return SGP_ERR_ARG;
    if (o->stop_rule < SGP_STOP_MAXIT || o->stop_rule > SGP_STOP_MINERR) return SGP_ERR_ARG;
    if (o->init < SGP_INIT_USER || o->init > SGP_INIT_CONST_SMOOTH) return SGP_ERR_ARG;
    if (o->init == SGP_INIT_CONST_SMOOTH && !(o->init_sigma > 0.0)) return SGP_ERR_ARG;
    if (o->flux_constraint != 0 && o->flux_constraint != 1) return SGP_ERR_ARG;
    if (o->psf_origin != SGP_PSF_CENTER && o->psf_origin != SGP_PSF_CORNER) return SGP_ERR_ARG;
    if (o->check_every < 0 || o->refresh_every < 0) return SGP_ERR_ARG;
    if (!(o->rl_relax > 0.0) || !(o->rl_linear > 0.0)) return SGP_ERR_ARG;
    if (o->rl_relax != 1.0 && o->rl_linear != 1.0) return SGP_ERR_ARG;      // Eq.3 and Eq.4 are alternatives
    return SGP_OK;
}

static int floor_pow2(int v) { int r = 1; while (r * 2 <= v) r *= 2; return r; }
static bool is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }

static int elems_per_thread(int L, int dtype, bool col)
{
    if (dtype == SGP_F64) return col ? fft_E_col<double>(L) : fft_E<double>(L);
    return col ? fft_E_col<float>(L) : fft_E<float>(L);
}
static int pad_len(int L, int E) { return L + (L >> (E == 32 ? 5 : 4)); }
static int row_len(int L, int E) { return (pad_len(L, E) + 1) & ~1; }      // fft_core.cuh: row_stride

// Spectrum tile width C (columns per CTA of the column kernel) and rows per CTA of the row kernels.
int choose_tiles(int ny, int nx, int dtype, const sgp_options *opt, int *C_out, int *RB_out, int nb)
{
    const int esz = dtype == SGP_F64 ? 16 : 8;                     // bytes per complex number
    const int Lr = nx / 2, Lc = ny;
    const int Ec = elems_per_thread(Lc, dtype, true), Er = elems_per_thread(Lr, dtype, false);
    const int TFc = Lc / Ec, TFr = Lr / Er;
    // column kernel: 256 threads per CTA when a thread holds 32 elements (two CTAs per SM), else up to 512;
    // at most ~100 KB of shared memory per CTA
    const int col_max = Ec == 32 ? 256 : 512;
    int C = floor_pow2(col_max / TFc > 1 ? col_max / TFc : 1);
    if (C > 32) C = 32;
    while (C > 1 && (size_t)C * pad_len(Lc, Ec) * esz > 72 * 1024) C /= 2;
    while (C > 1 && Lr % C != 0) C /= 2;
    // small grids: at least 32 tiles as long as a tile keeps 8 columns (full 64-byte pieces of a spectrum row in fp32) -- a 256^2
    // problem on 4 CTAs of 32 columns is latency-bound on 4 of 148 SMs (measured, 256^2: K2 / K5 14.9 / 14.2 -> 10.8 / 10.7 us;
    // same rule in col.cuh: col_default_C, for square grids)
    while (C > 8 && Lr / C < 32) C /= 2;
    if (opt && opt->tile_cols > 0) {
        if (!is_pow2(opt->tile_cols) || Lr % opt->tile_cols != 0) return SGP_ERR_ARG;
        C = opt->tile_cols;
    }
    if (C * TFc > col_max || (size_t)C * pad_len(Lc, Ec) * esz > 227 * 1024) return SGP_ERR_ARG;
    if (((size_t)C * pad_len(Lc, Ec) * esz) % 16 != 0) return SGP_ERR_ARG;        // the landing zones of the bulk copies follow the exchange buffer
    // row kernels: 256 threads per CTA; rows whose threads span several warps use one named barrier each (ids 1..15);
    // the 5-smooth lengths pad a row's thread group to a synchronisable size (fft_core.cuh: group_threads)
    const int TFg = group_threads(TFr);
    int RB = floor_pow2(256 / TFg > 1 ? 256 / TFg : 1);
    if (RB > 32) RB = 32;
    // small grids: enough row CTAs for two per SM (148 SMs) over all nb problems, as long as a CTA keeps 8 rows (one 256^2 problem:
    // 8 CTAs of 32 rows -> 32 of 8, with the tile rule above 19.7 -> 27.6 kit/s; 512^2: 18.3 -> 22.8 kit/s); a batched plan of 64
    // problems fills the GPU through blockIdx.z and keeps the larger CTAs (RB = 8 there: -6 %).  Sums are per CTA, so a batched and an
    // ordinary plan agree bit for bit only when their rows_per_block are equal (set it explicitly where that matters).
    while (RB > 8 && (long long)nb * (ny / RB) < 296 && ((RB / 2) * TFg) % 32 == 0) RB /= 2;
    if (opt && opt->rows_per_block > 0) {
        if (!is_pow2(opt->rows_per_block)) return SGP_ERR_ARG;
        RB = opt->rows_per_block;
    }
    while (RB > 1 && ny % RB != 0) RB /= 2;
    if (RB * TFg > 256 || (RB * TFg) % 32 != 0 || (TFg > 32 && RB > 15)) return SGP_ERR_ARG;
    {   // rows + the shared-memory copies of the twiddle tables (row_fwd.cuh) must leave room for two CTAs per SM
        const size_t tables = dtype == SGP_F64 ? row_table_entries<double>(Lr) : row_table_entries<float>(Lr);
        while (RB > 1 && ((size_t)RB * row_len(Lr, Er) + tables) * esz > 113 * 1024 && (RB / 2) * TFg % 32 == 0) RB /= 2;
        if (((size_t)RB * row_len(Lr, Er) + tables) * esz > 113 * 1024) return SGP_ERR_ARG;
    }
    *C_out = C; *RB_out = RB;
    return SGP_OK;
}

size_t workspace_bytes(int kind, int p, int ny, int nx, int dtype)
{
    if (p < 1 || p > SGP_MAX_IMAGES || !size_supported(ny) || !size_supported(nx)) return 0;
    const size_t r = dtype == SGP_F64 ? 8 : 4;
    const size_t n = (size_t)ny * nx;
    size_t planes = 7 * (size_t)p + 4;                 // khat, spec, g, b, q (two buffers), u per image; f, grad, d, scratch
    size_t b = planes * n * r;
    if (kind == SGP_KIND_BOUNDARY) b += (2 + (size_t)p) * n * r + n;     // alphaR, alpha, alpha_j on R (OSEM, Eq.22), M_R
    // twiddle tables (row passes, real<->complex, two column plans), pack line, companion lines of the transfer functions
    b += ((size_t)nx * 2 + 3 * (size_t)ny + (size_t)ny * (p + 1) + 64) * 2 * r;
    // per-CTA partial sums (one row of the grid per CTA at worst), per-chunk partials of the backtracking / flux kernels, set-up partials
    b += ((size_t)ny * (6 + 2 * p) + 2 * (n * p / 4096 + 2) + 1024 * (size_t)p + 2 * 1184 + 4096) * sizeof(double);
    b += sizeof(Ctrl) + 2048 /* BtInfo */ + 2 * 96 * sizeof(unsigned int);
    b += 64 * 256;                                     // every piece is rounded up to 256 bytes
    return b;
}

}  // namespace sgpk

using namespace sgpk;

struct sgp_plan { PlanBase *impl; };

extern "C" {

void sgp_options_default(sgp_options *o)
{
    if (!o) return;
    memset(o, 0, sizeof(*o));
    o->beta = 1e-4; o->theta = 0.4;
    o->alpha0 = 1.3; o->alpha_min = 1e-5; o->alpha_max = 1e5;
    o->tau1 = 0.5; o->m_alpha = 3;
    o->alt_start = 20;
    o->armijo_memory = 1;
    o->L1 = 1e-10; o->L2 = 1e10; o->adaptive_L = 1;
    o->max_iter = 100; o->stop_rule = SGP_STOP_MAXIT; o->tol = 1e-5;
    o->disc_threshold = 1.0; o->sigma_R = 1e-2; o->max_backtracks = 30;
    o->psf_origin = SGP_PSF_CENTER; o->init = SGP_INIT_CONST;
    o->refresh_every = 0; o->strict = 0; o->check_every = 0;
    o->flux_constraint = 0; o->flux_value = 0.0; o->init_sigma = 2.0;
    o->tile_cols = 0; o->rows_per_block = 0; o->use_graph = 1; o->rl_relax = 1.0; o->rl_linear = 1.0;
}

void sgp_result_init(sgp_result *r) { if (r) memset(r, 0, sizeof(*r)); }

const char *sgp_strerror(int s)
{
    switch (s) {
    case SGP_OK: return "ok";
    case SGP_ERR_ARG: return "invalid argument (null pointer, p out of range, unsupported grid size or option value)";
    case SGP_ERR_PSF: return "PSF sum is not positive or not finite";
    case SGP_ERR_DATA: return "invalid data (non-finite or negative image values, negative start image, no positive value for the scaling bounds)";
    case SGP_ERR_ALLOC: return "allocation failed";
    case SGP_ERR_CUDA: return "CUDA error (see sgp_last_cuda_error)";
    case SGP_ERR_LINESEARCH: return "line search failed: max_backtracks reductions without Armijo acceptance";
    case SGP_ERR_NONFINITE: return "objective J0 is not finite";
    case SGP_ERR_UNSUPPORTED: return "option combination not supported by this build";
    default: return "unknown status";
    }
}

const char *sgp_version(void) { return "sgp-b200 0.1.0 (sm_100a)"; }
const char *sgp_last_cuda_error(void) { return g_last_cuda_error.c_str(); }

size_t sgp_workspace_bytes(int kind, int p, int ny, int nx, int dtype) { return workspace_bytes(kind, p, ny, nx, dtype); }
size_t sgp_plan_workspace_bytes(const sgp_plan *plan);

int sgp_plan_create(sgp_plan **plan, int kind, int p, int ny, int nx, int oy, int ox, int sy, int sx, int dtype,
                    const sgp_options *opt)
{
    return sgp_plan_create_batched(plan, 1, kind, p, ny, nx, oy, ox, sy, sx, dtype, opt);
}

int sgp_plan_create_batched(sgp_plan **plan, int nb, int kind, int p, int ny, int nx, int oy, int ox, int sy, int sx, int dtype,
                            const sgp_options *opt)
{
    if (!plan) return SGP_ERR_ARG;
    if (nb < 1 || nb > 65535) { *plan = nullptr; return SGP_ERR_ARG; }
    *plan = nullptr;
    sgp_options o;
    if (opt) o = *opt; else sgp_options_default(&o);
    int rc = validate_options(&o);
    if (rc) return rc;
    if (dtype != SGP_F32 && dtype != SGP_F64) return SGP_ERR_ARG;
    if (kind < SGP_KIND_SINGLE || kind > SGP_KIND_BOUNDARY) return SGP_ERR_ARG;
    if (p < 1 || p > SGP_MAX_IMAGES || (kind == SGP_KIND_SINGLE && p != 1)) return SGP_ERR_ARG;
    if (!size_supported(ny) || !size_supported(nx)) return SGP_ERR_ARG;
    if (kind == SGP_KIND_BOUNDARY) {
        if (oy < 0 || ox < 0 || sy < 1 || sx < 1 || oy + sy > ny || ox + sx > nx) return SGP_ERR_ARG;
        if (!(o.sigma_R > 0)) return SGP_ERR_ARG;
    } else { oy = 0; ox = 0; sy = ny; sx = nx; }
    PlanBase *b = dtype == SGP_F32 ? make_plan_f32() : make_plan_f64();
    if (!b) return SGP_ERR_ALLOC;
    b->kind = kind; b->p = p; b->ny = ny; b->nx = nx; b->dtype = dtype; b->opt = o; b->nb = nb;
    b->G.ny = ny; b->G.nx = nx; b->G.oy = oy; b->G.ox = ox; b->G.sy = sy; b->G.sx = sx;
    b->G.masked = kind == SGP_KIND_BOUNDARY ? 1 : 0; b->G.p = p;
    rc = b->init();
    if (rc) { delete b; return rc; }
    sgp_plan *pl = new (std::nothrow) sgp_plan;
    if (!pl) { delete b; return SGP_ERR_ALLOC; }
    pl->impl = b;
    *plan = pl;
    return SGP_OK;
}

size_t sgp_plan_workspace_bytes(const sgp_plan *plan) { return plan ? plan->impl->bytes_allocated : 0; }

void sgp_plan_destroy(sgp_plan *plan)
{
    if (!plan) return;
    delete plan->impl;
    delete plan;
}

int sgp_plan_set_psf(sgp_plan *plan, const void *const *psf, void *stream)
{
    if (!plan || !psf) return SGP_ERR_ARG;
    return plan->impl->set_psf(psf, (cudaStream_t)stream);
}

int sgp_plan_run(sgp_plan *plan, int algorithm, const void *const *g, const void *const *b_arr, const double *b_const,
                 const void *f0, void *f_out, const sgp_options *opt, sgp_result *res, void *stream)
{
    if (!plan) return SGP_ERR_ARG;
    return plan->impl->run(algorithm, g, b_arr, b_const, f0, f_out, opt, res, (cudaStream_t)stream);
}

int sgp_plan_run_batched(sgp_plan *plan, int algorithm, const void *const *g, const void *const *b_arr, const double *b_const,
                         const void *const *f0, void *const *f_out, const sgp_options *opt, sgp_result *res, void *stream)
{
    if (!plan) return SGP_ERR_ARG;
    return plan->impl->run_batched(algorithm, g, b_arr, b_const, f0, f_out, opt, res, (cudaStream_t)stream);
}

int sgp_plan_apply_A(sgp_plan *plan, int j, const void *x, void *out, void *stream)
{
    if (!plan) return SGP_ERR_ARG;
    return plan->impl->apply(false, j, x, out, (cudaStream_t)stream);
}
int sgp_plan_apply_AT(sgp_plan *plan, int j, const void *y, void *out, void *stream)
{
    if (!plan) return SGP_ERR_ARG;
    return plan->impl->apply(true, j, y, out, (cudaStream_t)stream);
}
int sgp_plan_get_mask(sgp_plan *plan, unsigned char *maskR_out, void *alpha_out, long *nR, void *stream)
{
    if (!plan) return SGP_ERR_ARG;
    return plan->impl->get_mask(maskR_out, alpha_out, nR, (cudaStream_t)stream);
}
int sgp_plan_rfft2(sgp_plan *plan, const void *x, void *spec_out, void *stream)
{
    if (!plan) return SGP_ERR_ARG;
    return plan->impl->rfft2(x, spec_out, (cudaStream_t)stream);
}
int sgp_plan_irfft2(sgp_plan *plan, const void *spec_in, void *x_out, void *stream)
{
    if (!plan) return SGP_ERR_ARG;
    return plan->impl->irfft2(spec_in, x_out, (cudaStream_t)stream);
}

int sgp_plan_set_profiling(sgp_plan *plan, int on)
{
    if (!plan) return SGP_ERR_ARG;
    plan->impl->profiling = on != 0;
    return SGP_OK;
}
int sgp_plan_get_kernel_ms(sgp_plan *plan, double *ms_sum, long *launches)
{
    if (!plan || !ms_sum || !launches) return SGP_ERR_ARG;
    for (int i = 0; i < SGP_PROF_SLOTS; ++i) { ms_sum[i] = plan->impl->prof_ms[i]; launches[i] = plan->impl->prof_count[i]; }
    return SGP_OK;
}

// ---- one-shot calls: find or create a plan, set the PSFs, run.
// The plan of the last one-shot call of this host thread is kept (workspace, twiddles, the instantiated CUDA graph) and used
// again when the next call has the same geometry, dtype, device and plan-time options; a call with another key replaces it.
// sgp_release_cached_plans() frees it; so does the end of the thread.  The PSFs are transformed again in every call.
struct PlanKey {
    int dev, kind, p, ny, nx, oy, ox, sy, sx, dtype, tile_cols, rows_per_block, use_graph, psf_origin;
    int nb;            // problems of a batched plan (sgp_mosaic); 0 for the ordinary plans of the one-shot calls
    double sigma_R;
    bool operator==(const PlanKey &o) const
    {
        return dev == o.dev && kind == o.kind && p == o.p && ny == o.ny && nx == o.nx && oy == o.oy && ox == o.ox && sy == o.sy &&
               sx == o.sx && dtype == o.dtype && tile_cols == o.tile_cols && rows_per_block == o.rows_per_block &&
               use_graph == o.use_graph && psf_origin == o.psf_origin && nb == o.nb && sigma_R == o.sigma_R;
    }
};
struct PlanCache {
    sgp_plan *plan = nullptr;
    PlanKey key{};
    void clear() { if (plan) { sgp_plan_destroy(plan); plan = nullptr; } }
    ~PlanCache() { clear(); }
};
static thread_local PlanCache g_plan_cache;
static thread_local PlanCache g_mosaic_cache;      // the batched sub-domain plan of this thread's last sgp_mosaic call, kept the same way

static void release_host_bufs();
void sgp_release_cached_plans(void) { g_plan_cache.clear(); g_mosaic_cache.clear(); release_host_bufs(); }

static int one_shot(int algorithm, int kind, int p, const void *const *g, const void *const *psf, const void *const *b_arr,
                    const double *b_const, int oy, int ox, int sy, int sx, int ny, int nx, const void *f0, void *f_out,
                    unsigned char *maskR_out, int dtype, const sgp_options *opt, sgp_result *res, void *stream)
{
    if (!g || !psf || !f_out || !res || !opt) return SGP_ERR_ARG;
    PlanKey key{};
    if (cudaGetDevice(&key.dev) != cudaSuccess) { (void)cudaGetLastError(); key.dev = -1; }
    key.kind = kind; key.p = p; key.ny = ny; key.nx = nx; key.dtype = dtype;
    const bool bnd = kind == SGP_KIND_BOUNDARY;
    key.oy = bnd ? oy : 0; key.ox = bnd ? ox : 0; key.sy = bnd ? sy : ny; key.sx = bnd ? sx : nx;
    key.tile_cols = opt->tile_cols; key.rows_per_block = opt->rows_per_block; key.use_graph = opt->use_graph & ~1;
    key.psf_origin = opt->psf_origin; key.sigma_R = bnd ? opt->sigma_R : 0.0;
    PlanCache &pc = g_plan_cache;
    int rc;
    if (!pc.plan || !(pc.key == key)) {
        pc.clear();
        rc = sgp_plan_create(&pc.plan, kind, p, ny, nx, oy, ox, sy, sx, dtype, opt);
        if (rc) { pc.plan = nullptr; return rc; }
        pc.key = key;
    }
    sgp_plan *pl = pc.plan;
    const long l0 = pl->impl->launches;
    rc = sgp_plan_set_psf(pl, psf, stream);
    if (!rc) rc = sgp_plan_run(pl, algorithm, g, b_arr, b_const, f0, f_out, opt, res, stream);
    if (maskR_out && (rc == SGP_OK || rc == SGP_ERR_LINESEARCH)) {
        int r2 = sgp_plan_get_mask(pl, maskR_out, nullptr, nullptr, stream);
        if (!rc) rc = r2;
    }
    res->kernel_launches = pl->impl->launches - l0;
    if (rc == SGP_ERR_CUDA || rc == SGP_ERR_ALLOC) pc.clear();          // do not keep a plan whose device state is unknown
    return rc;
}

int sgp_single(const void *g, const void *psf, const void *b_arr, double b_const, const void *f0, void *f_out, int ny, int nx,
               int dtype, const sgp_options *opt, sgp_result *res, void *stream)
{
    const void *gg[1] = {g}, *pp[1] = {psf}, *bb[1] = {b_arr};
    return one_shot(SGP_ALG_SGP, SGP_KIND_SINGLE, 1, gg, pp, b_arr ? bb : nullptr, &b_const, 0, 0, ny, nx, ny, nx, f0, f_out, nullptr,
                    dtype, opt, res, stream);
}
int rl_single(const void *g, const void *psf, const void *b_arr, double b_const, const void *f0, void *f_out, int ny, int nx,
              int dtype, const sgp_options *opt, sgp_result *res, void *stream)
{
    const void *gg[1] = {g}, *pp[1] = {psf}, *bb[1] = {b_arr};
    return one_shot(SGP_ALG_RL, SGP_KIND_SINGLE, 1, gg, pp, b_arr ? bb : nullptr, &b_const, 0, 0, ny, nx, ny, nx, f0, f_out, nullptr,
                    dtype, opt, res, stream);
}
int sgp_multi(int p, const void *const *g, const void *const *psf, const void *const *b_arr, const double *b_const,
              const void *f0, void *f_out, int ny, int nx, int dtype, const sgp_options *opt, sgp_result *res, void *stream)
{
    return one_shot(SGP_ALG_SGP, SGP_KIND_MULTI, p, g, psf, b_arr, b_const, 0, 0, ny, nx, ny, nx, f0, f_out, nullptr, dtype, opt, res, stream);
}
int rl_multi(int p, const void *const *g, const void *const *psf, const void *const *b_arr, const double *b_const,
             const void *f0, void *f_out, int ny, int nx, int dtype, const sgp_options *opt, sgp_result *res, void *stream)
{
    return one_shot(SGP_ALG_RL, SGP_KIND_MULTI, p, g, psf, b_arr, b_const, 0, 0, ny, nx, ny, nx, f0, f_out, nullptr, dtype, opt, res, stream);
}
int sgp_boundary(int p, const void *const *g, const void *const *psf, const void *const *b_arr, const double *b_const,
                 int oy, int ox, int sy, int sx, int ny, int nx, const void *f0, void *f_out, unsigned char *maskR_out,
                 int dtype, const sgp_options *opt, sgp_result *res, void *stream)
{
    return one_shot(SGP_ALG_SGP, SGP_KIND_BOUNDARY, p, g, psf, b_arr, b_const, oy, ox, sy, sx, ny, nx, f0, f_out, maskR_out, dtype, opt, res, stream);
}
int rl_boundary(int p, const void *const *g, const void *const *psf, const void *const *b_arr, const double *b_const,
                int oy, int ox, int sy, int sx, int ny, int nx, const void *f0, void *f_out, unsigned char *maskR_out,
                int dtype, const sgp_options *opt, sgp_result *res, void *stream)
{
    return one_shot(SGP_ALG_RL, SGP_KIND_BOUNDARY, p, g, psf, b_arr, b_const, oy, ox, sy, sx, ny, nx, f0, f_out, maskR_out, dtype, opt, res, stream);
}

int osem_multi(int p, const void *const *g, const void *const *psf, const void *const *b_arr, const double *b_const,
               const void *f0, void *f_out, int ny, int nx, int dtype, const sgp_options *opt, sgp_result *res, void *stream)
{
    return one_shot(SGP_ALG_OSEM, SGP_KIND_MULTI, p, g, psf, b_arr, b_const, 0, 0, ny, nx, ny, nx, f0, f_out, nullptr, dtype, opt, res, stream);
}
int osem_boundary(int p, const void *const *g, const void *const *psf, const void *const *b_arr, const double *b_const,
                  int oy, int ox, int sy, int sx, int ny, int nx, const void *f0, void *f_out, unsigned char *maskR_out,
                  int dtype, const sgp_options *opt, sgp_result *res, void *stream)
{
    return one_shot(SGP_ALG_OSEM, SGP_KIND_BOUNDARY, p, g, psf, b_arr, b_const, oy, ox, sy, sx, ny, nx, f0, f_out, maskR_out, dtype, opt, res, stream);
}

// ---- host-pointer variants: stage through device buffers (pinned staging is the caller's choice)
struct DevBufs {      // one device allocation, carved into 256-byte aligned pieces
    unsigned char *base = nullptr;
    size_t cap = 0, used = 0;
    ~DevBufs() { cudaFree(base); }
    static size_t al(size_t b) { return (b + 255) & ~(size_t)255; }
    int dev = -1;
    int reserve(size_t bytes)         // grow-only when the object is kept across calls (host_shot); starts an empty carve
    {
        int d = 0;
        SGP_CUDA_TRY(cudaGetDevice(&d));
        used = 0;
        if (base && d == dev && bytes <= cap) return SGP_OK;
        release();
        SGP_CUDA_TRY(cudaMalloc((void **)&base, bytes ? bytes : 256));
        cap = bytes; dev = d;
        return SGP_OK;
    }
    void release() { if (base) { cudaFree(base); (void)cudaGetLastError(); } base = nullptr; cap = 0; used = 0; }
    int blank(size_t bytes, void **dev)
    {
        if (used + al(bytes) > cap) return SGP_ERR_ALLOC;
        *dev = base + used; used += al(bytes);
        return SGP_OK;
    }
    int up(const void *host, size_t bytes, cudaStream_t st, void **dev)
    {
        *dev = nullptr;
        if (!host) return SGP_OK;
        int rc = blank(bytes, dev);
        if (rc) return rc;
        SGP_CUDA_TRY(cudaMemcpyAsync(*dev, host, bytes, cudaMemcpyHostToDevice, st));
        return SGP_OK;
    }
};

static thread_local DevBufs g_host_bufs;      // staging of the *_host calls of this thread, kept like the plan
static thread_local DevBufs g_mosaic_bufs;    // sub-images and sub-domain reconstructions of sgp_mosaic
static void release_host_bufs() { g_host_bufs.release(); g_mosaic_bufs.release(); }

static int host_shot(int algorithm, int kind, int p, const void *const *g, const void *const *psf, const void *const *b_arr,
                     const double *b_const, int oy, int ox, int sy, int sx, int ny, int nx, const void *f0, void *f_out,
                     unsigned char *maskR_out, int dtype, const sgp_options *opt, sgp_result *res, void *stream)
{
    if (!g || !psf || !f_out || !res || !opt || p < 1 || p > SGP_MAX_IMAGES) return SGP_ERR_ARG;
    if (dtype != SGP_F32 && dtype != SGP_F64) return SGP_ERR_ARG;
    if (ny < 1 || nx < 1 || sy < 1 || sx < 1) return SGP_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t r = dtype == SGP_F64 ? 8 : 4;
    const size_t nb = (size_t)ny * nx * r, sb = (size_t)sy * sx * r;
    DevBufs &D = g_host_bufs;
    const void *dg[SGP_MAX_IMAGES], *dk[SGP_MAX_IMAGES], *db[SGP_MAX_IMAGES];
    int rc;
    bool have_b = false;
    if ((rc = D.reserve((size_t)p * (2 * DevBufs::al(sb) + DevBufs::al(nb)) + 2 * DevBufs::al(nb) + DevBufs::al((size_t)ny * nx)))) return rc;
    for (int j = 0; j < p; ++j) {
        if (!g[j] || !psf[j]) return SGP_ERR_ARG;
        void *t;
        if ((rc = D.up(g[j], sb, st, &t))) return rc; dg[j] = t;
        if ((rc = D.up(psf[j], nb, st, &t))) return rc; dk[j] = t;
        if ((rc = D.up(b_arr ? b_arr[j] : nullptr, sb, st, &t))) return rc; db[j] = t;
        if (t) have_b = true;
    }
    void *df0 = nullptr, *dout = nullptr, *dmask = nullptr;
    if ((rc = D.up(f0, nb, st, &df0))) return rc;
    if ((rc = D.blank(nb, &dout))) return rc;
    if (maskR_out && (rc = D.blank((size_t)ny * nx, &dmask))) return rc;
    rc = one_shot(algorithm, kind, p, dg, dk, have_b ? db : nullptr, b_const, oy, ox, sy, sx, ny, nx, df0, dout,
                  (unsigned char *)dmask, dtype, opt, res, stream);
    if (rc == SGP_OK || rc == SGP_ERR_LINESEARCH) {
        SGP_CUDA_TRY(cudaMemcpyAsync(f_out, dout, nb, cudaMemcpyDeviceToHost, st));
        if (maskR_out) SGP_CUDA_TRY(cudaMemcpyAsync(maskR_out, dmask, (size_t)ny * nx, cudaMemcpyDeviceToHost, st));
        SGP_CUDA_TRY(cudaStreamSynchronize(st));
    }
    return rc;
}

int sgp_single_host(const void *g, const void *psf, const void *b_arr, double b_const, const void *f0, void *f_out, int ny,
                    int nx, int dtype, const sgp_options *opt, sgp_result *res, void *stream)
{
    const void *gg[1] = {g}, *pp[1] = {psf}, *bb[1] = {b_arr};
    return host_shot(SGP_ALG_SGP, SGP_KIND_SINGLE, 1, gg, pp, b_arr ? bb : nullptr, &b_const, 0, 0, ny, nx, ny, nx, f0, f_out, nullptr,
                     dtype, opt, res, stream);
}
int rl_single_host(const void *g, const void *psf, const void *b_arr, double b_const, const void *f0, void *f_out, int ny,
                   int nx, int dtype, const sgp_options *opt, sgp_result *res, void *stream)
{
    const void *gg[1] = {g}, *pp[1] = {psf}, *bb[1] = {b_arr};
    return host_shot(SGP_ALG_RL, SGP_KIND_SINGLE, 1, gg, pp, b_arr ? bb : nullptr, &b_const, 0, 0, ny, nx, ny, nx, f0, f_out, nullptr,
                     dtype, opt, res, stream);
}
int sgp_multi_host(int p, const void *const *g, const void *const *psf, const void *const *b_arr, const double *b_const,
                   const void *f0, void *f_out, int ny, int nx, int dtype, const sgp_options *opt, sgp_result *res, void *stream)
{
    return host_shot(SGP_ALG_SGP, SGP_KIND_MULTI, p, g, psf, b_arr, b_const, 0, 0, ny, nx, ny, nx, f0, f_out, nullptr, dtype, opt, res, stream);
}
int rl_multi_host(int p, const void *const *g, const void *const *psf, const void *const *b_arr, const double *b_const,
                  const void *f0, void *f_out, int ny, int nx, int dtype, const sgp_options *opt, sgp_result *res, void *stream)
{
    return host_shot(SGP_ALG_RL, SGP_KIND_MULTI, p, g, psf, b_arr, b_const, 0, 0, ny, nx, ny, nx, f0, f_out, nullptr, dtype, opt, res, stream);
}
int osem_multi_host(int p, const void *const *g, const void *const *psf, const void *const *b_arr, const double *b_const,
                    const void *f0, void *f_out, int ny, int nx, int dtype, const sgp_options *opt, sgp_result *res, void *stream)
{
    return host_shot(SGP_ALG_OSEM, SGP_KIND_MULTI, p, g, psf, b_arr, b_const, 0, 0, ny, nx, ny, nx, f0, f_out, nullptr, dtype, opt, res, stream);
}
int osem_boundary_host(int p, const void *const *g, const void *const *psf, const void *const *b_arr, const double *b_const,
                       int oy, int ox, int sy, int sx, int ny, int nx, const void *f0, void *f_out, unsigned char *maskR_out,
                       int dtype, const sgp_options *opt, sgp_result *res, void *stream)
{
    return host_shot(SGP_ALG_OSEM, SGP_KIND_BOUNDARY, p, g, psf, b_arr, b_const, oy, ox, sy, sx, ny, nx, f0, f_out, maskR_out, dtype, opt, res, stream);
}
int sgp_boundary_host(int p, const void *const *g, const void *const *psf, const void *const *b_arr, const double *b_const,
                      int oy, int ox, int sy, int sx, int ny, int nx, const void *f0, void *f_out, unsigned char *maskR_out,
                      int dtype, const sgp_options *opt, sgp_result *res, void *stream)
{
    return host_shot(SGP_ALG_SGP, SGP_KIND_BOUNDARY, p, g, psf, b_arr, b_const, oy, ox, sy, sx, ny, nx, f0, f_out, maskR_out, dtype, opt, res, stream);
}
int rl_boundary_host(int p, const void *const *g, const void *const *psf, const void *const *b_arr, const double *b_const,
                     int oy, int ox, int sy, int sx, int ny, int nx, const void *f0, void *f_out, unsigned char *maskR_out,
                     int dtype, const sgp_options *opt, sgp_result *res, void *stream)
{
    return host_shot(SGP_ALG_RL, SGP_KIND_BOUNDARY, p, g, psf, b_arr, b_const, oy, ox, sy, sx, ny, nx, f0, f_out, maskR_out, dtype, opt, res, stream);
}

// ---- mosaic of sub-domain reconstructions: one batched boundary plan over the ty x tx sub-images
static int mosaic_start(int t, int N, int T, int s) { int h = N / T, o = t * h - (s - h) / 2; return o < 0 ? 0 : (o > N - s ? N - s : o); }

int sgp_mosaic(int algorithm, int p, const void *const *g, const void *const *psf, const double *b_const, int Ny, int Nx,
               int ty, int tx, int sy, int sx, int ny, int nx, void *f_out, int dtype, const sgp_options *opt,
               sgp_result *res, void *stream)
{
    if (!g || !psf || !b_const || !f_out || !opt || !res || p < 1 || p > SGP_MAX_IMAGES) return SGP_ERR_ARG;
    if (dtype != SGP_F32 && dtype != SGP_F64) return SGP_ERR_ARG;
    if (ty < 1 || tx < 1 || Ny % ty || Nx % tx || sy < Ny / ty || sx < Nx / tx || sy > Ny || sx > Nx || sy > ny || sx > nx) return SGP_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t r = dtype == SGP_F64 ? 8 : 4;
    const int nb = ty * tx, hy = Ny / ty, hx = Nx / tx, oy = (ny - sy) / 2, ox = (nx - sx) / 2;
    // the sub-domain plan (workspace, tables, boundary weights' buffers) and the sub-image buffers are kept between calls of the same
    // geometry, like the plan of the one-shot calls (creating and freeing them was 6 of the 8.4 ms of a 2 x 2 mosaic of 160^2-in-256^2
    // sub-domains, 100 iterations each); the PSFs are transformed and the weights recomputed in every call
    PlanKey key{};
    if (cudaGetDevice(&key.dev) != cudaSuccess) { (void)cudaGetLastError(); key.dev = -1; }
    key.kind = SGP_KIND_BOUNDARY; key.p = p; key.ny = ny; key.nx = nx; key.dtype = dtype; key.oy = oy; key.ox = ox; key.sy = sy; key.sx = sx;
    key.tile_cols = opt->tile_cols; key.rows_per_block = opt->rows_per_block; key.use_graph = opt->use_graph & ~1;
    key.psf_origin = opt->psf_origin; key.sigma_R = opt->sigma_R; key.nb = nb;
    PlanCache &pc = g_mosaic_cache;
    int rc;
    if (!pc.plan || !(pc.key == key)) {
        pc.clear();
        rc = sgp_plan_create_batched(&pc.plan, nb, SGP_KIND_BOUNDARY, p, ny, nx, oy, ox, sy, sx, dtype, opt);
        if (rc) { pc.plan = nullptr; return rc; }
        pc.key = key;
    }
    sgp_plan *pl = pc.plan;
    DevBufs &D = g_mosaic_bufs;       // the sub-images (contiguous sy x sx copies of windows of g_j) and the nb reconstructions
    const size_t sb = (size_t)sy * sx * r, nbytes = (size_t)ny * nx * r;
    std::vector<const void *> gs((size_t)nb * p);
    std::vector<void *> fo((size_t)nb);
    std::vector<double> bc((size_t)nb * p);
    rc = D.reserve((size_t)nb * p * DevBufs::al(sb) + (size_t)nb * DevBufs::al(nbytes));
    for (int t = 0; t < nb && !rc; ++t) {
        const int yi = mosaic_start(t / tx, Ny, ty, sy), xi = mosaic_start(t % tx, Nx, tx, sx);
        for (int j = 0; j < p && !rc; ++j) {
            void *sub = nullptr;
            if (!g[j]) { rc = SGP_ERR_ARG; break; }
            rc = D.blank(sb, &sub);
            if (rc) break;
            const unsigned char *src = static_cast<const unsigned char *>(g[j]) + ((size_t)yi * Nx + xi) * r;
            if (cudaMemcpy2DAsync(sub, (size_t)sx * r, src, (size_t)Nx * r, (size_t)sx * r, (size_t)sy, cudaMemcpyDeviceToDevice, st) != cudaSuccess) rc = SGP_ERR_CUDA;
            gs[(size_t)t * p + j] = sub; bc[(size_t)t * p + j] = b_const[j];
        }
        if (!rc) rc = D.blank(nbytes, &fo[t]);
    }
    if (!rc) rc = sgp_plan_set_psf(pl, psf, stream);
    if (!rc) rc = sgp_plan_run_batched(pl, algorithm, gs.data(), nullptr, bc.data(), nullptr, fo.data(), opt, res, stream);
    if (rc == SGP_OK || rc == SGP_ERR_LINESEARCH) {
        for (int t = 0; t < nb; ++t) {
            const int iy = t / tx, ix = t % tx;
            const int yi = mosaic_start(iy, Ny, ty, sy), xi = mosaic_start(ix, Nx, tx, sx);
            const int ys = iy * hy - yi + oy, xs = ix * hx - xi + ox;        // the non-overlapping part inside S-bar
            const unsigned char *src = static_cast<const unsigned char *>(fo[t]) + ((size_t)ys * nx + xs) * r;
            unsigned char *dst = static_cast<unsigned char *>(f_out) + ((size_t)iy * hy * Nx + (size_t)ix * hx) * r;
            if (cudaMemcpy2DAsync(dst, (size_t)Nx * r, src, (size_t)nx * r, (size_t)hx * r, (size_t)hy, cudaMemcpyDeviceToDevice, st) != cudaSuccess && !rc) rc = SGP_ERR_CUDA;
        }
        if (cudaStreamSynchronize(st) != cudaSuccess && !rc) rc = SGP_ERR_CUDA;
    }
    if (rc == SGP_ERR_CUDA || rc == SGP_ERR_ALLOC) pc.clear();          // do not keep a plan whose device state is unknown
    return rc;
}

int sgp_mosaic_host(int algorithm, int p, const void *const *g, const void *const *psf, const double *b_const, int Ny, int Nx,
                    int ty, int tx, int sy, int sx, int ny, int nx, void *f_out, int dtype, const sgp_options *opt,
                    sgp_result *res, void *stream)
{
    if (!g || !psf || !f_out || p < 1 || p > SGP_MAX_IMAGES || Ny < 1 || Nx < 1 || ny < 1 || nx < 1) return SGP_ERR_ARG;
    if (dtype != SGP_F32 && dtype != SGP_F64) return SGP_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t r = dtype == SGP_F64 ? 8 : 4;
    const size_t ib = (size_t)Ny * Nx * r, kb = (size_t)ny * nx * r;
    DevBufs D;
    int rc = D.reserve((size_t)p * (DevBufs::al(ib) + DevBufs::al(kb)) + DevBufs::al(ib));
    if (rc) return rc;
    const void *dg[SGP_MAX_IMAGES], *dk[SGP_MAX_IMAGES];
    for (int j = 0; j < p; ++j) {
        if (!g[j] || !psf[j]) return SGP_ERR_ARG;
        void *t;
        if ((rc = D.up(g[j], ib, st, &t))) return rc; dg[j] = t;
        if ((rc = D.up(psf[j], kb, st, &t))) return rc; dk[j] = t;
    }
    void *dout = nullptr;
    if ((rc = D.blank(ib, &dout))) return rc;
    rc = sgp_mosaic(algorithm, p, dg, dk, b_const, Ny, Nx, ty, tx, sy, sx, ny, nx, dout, dtype, opt, res, stream);
    if (rc == SGP_OK || rc == SGP_ERR_LINESEARCH) {
        SGP_CUDA_TRY(cudaMemcpyAsync(f_out, dout, ib, cudaMemcpyDeviceToHost, st));
        SGP_CUDA_TRY(cudaStreamSynchronize(st));
    }
    return rc;
}

}  // extern "C"
