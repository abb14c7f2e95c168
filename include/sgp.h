/*
 * sgp.h -- C ABI of libsgp_b200: scaled gradient projection (SGP) and Richardson-Lucy (RL)
 * deconvolution of Poisson images on one NVIDIA B200 (sm_100a).
 *
 * Method: Prato, Cavicchioli, Zanni, Boccacci, Bertero, "Efficient deconvolution methods for
 * astronomical imaging: algorithms and IDL-GPU codes" (arXiv:1210.2258).  Citations below are
 * PAPER.md:<line> + equation / algorithm; "A<n>" are the readings listed in DESIGN.md section 3.
 *
 *   minimise   J0(f) = sum_j sum_{m in S} { g_j ln( g_j / (A_j f + b_j) ) + A_j f + b_j - g_j }    (Eq.2 / Eq.12)
 *   subject to f >= 0,
 *   A_j f   = M_S o (K_j * (M_R o f))                                   (Eq.16)
 *   A_j^T y = M_R o (K_j corr (M_S o y))                                (Eq.17)
 *
 * by Algorithm 1 with the scaling D_k = (M_R/alpha) o clip(f, L1, L2) (Eq.10 / Eq.23),
 * the alternating Barzilai-Borwein step lengths (Eq.7-9) and Armijo backtracking on
 * A f + lambda A d (Alg.1 steps 4-5), or by the RL iteration f <- (M_R/alpha) o f o sum_j A_j^T(g_j/(A_j f + b_j))
 * (Eq.1 / Eq.13 / Eq.21).  Every step of the iteration runs in CUDA kernels of this library; there
 * is no CPU fallback.
 *
 * Conventions
 *   - Arrays are row-major and contiguous: element (y, x) of an ny x nx array is a[y*nx + x].
 *   - Entry points WITHOUT the _host suffix take DEVICE pointers (cudaMalloc'ed or a torch CUDA
 *     tensor's data_ptr); the *_host variants take HOST pointers and copy to / from the device inside
 *     the call.  Arrays of pointers (g[], psf[], b_arr[]) are always HOST arrays holding p pointers.
 *   - `dtype` selects the element type of every array argument: SGP_F32 = float, SGP_F64 = double.
 *     All reductions (J0, dot products) are accumulated in double in both modes.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  The calls are
 *     synchronous with respect to the host: they return after the work has completed on `stream`.
 *   - Ownership: the caller owns every input and output; inputs are never modified; f_out may alias
 *     f0.  The library owns only the plan's workspace, freed by sgp_plan_destroy.
 *   - Errors: every entry point returns 0 (SGP_OK) or a negative sgp_status.  Nothing is printed, no
 *     exception crosses the ABI.  After an error inside the iteration f_out holds the last accepted
 *     iterate.  sgp_last_cuda_error() gives the text of the last CUDA error seen by this thread.
 *   - Grid sizes: ny, nx (independently) of the form 2^a 5^b within 64...4096 that are a power of two or a multiple of
 *     40: 64 80 128 160 200 256 320 400 512 640 800 1000 1024 1280 1600 2000 2048 2560 3200 4000 4096; any other size
 *     returns SGP_ERR_ARG (500, 625, 1250, 2500, 3125 have no radix plan; pad the grid).
 *   - A plan is not thread-safe; different plans may be used from different threads.
 */
#ifndef SGP_B200_H
#define SGP_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SGP_MAX_IMAGES 16
#define SGP_MAX_MALPHA 16
#define SGP_MAX_ARMIJO_MEMORY 64

typedef enum { SGP_F32 = 0, SGP_F64 = 1 } sgp_dtype;
/* stopping rules, PAPER.md:279-298 (Sect.3.3); max_iter is always an additional cap */
typedef enum { SGP_STOP_MAXIT = 0, SGP_STOP_RELJ = 1, SGP_STOP_DISCREPANCY = 2,
               SGP_STOP_MINERR = 3 /* Eq.25: needs sgp_result.truth; DESIGN reading A27 */ } sgp_stop;
/* initial guess, PAPER.md:260-267 (Sect.3.1) */
typedef enum { SGP_INIT_USER = 0, SGP_INIT_CONST = 1, SGP_INIT_ZERO = 2, SGP_INIT_G = 3,
               SGP_INIT_CONST_SMOOTH = 4 /* the constant image convolved with a Gaussian (reading A28) */ } sgp_init;
/* where the PSF centre sits in the input array (A18) */
typedef enum { SGP_PSF_CENTER = 0, SGP_PSF_CORNER = 1 } sgp_psf_origin;
/* problem kind of a plan */
typedef enum { SGP_KIND_SINGLE = 0, SGP_KIND_MULTI = 1, SGP_KIND_BOUNDARY = 2 } sgp_kind;
/* algorithm run by sgp_plan_run */
typedef enum { SGP_ALG_SGP = 0, SGP_ALG_RL = 1, SGP_ALG_OSEM = 2 } sgp_algorithm;

typedef enum {
    SGP_OK = 0,
    SGP_ERR_ARG = -1,        /* null pointer, p out of range, unsupported size, bad option value */
    SGP_ERR_PSF = -2,        /* PSF sum <= 0 or non-finite */
    SGP_ERR_DATA = -3,       /* non-finite g, negative g in strict mode, negative user f0, no positive value for the adaptive bounds */
    SGP_ERR_ALLOC = -4,      /* device or host allocation failed */
    SGP_ERR_CUDA = -5,       /* a CUDA call failed; see sgp_last_cuda_error() */
    SGP_ERR_LINESEARCH = -6, /* max_backtracks reductions of lambda without Armijo acceptance (A16) */
    SGP_ERR_NONFINITE = -7,  /* J0 of the start point is not finite */
    SGP_ERR_UNSUPPORTED = -8 /* option combination not available in this build */
} sgp_status;

/* stop_reason values in sgp_result */
typedef enum { SGP_REASON_NONE = 0, SGP_REASON_MAXIT = 1, SGP_REASON_RELJ = 2, SGP_REASON_DISCREPANCY = 3,
               SGP_REASON_MINERR = 4 } sgp_reason;

/* Options; sgp_options_default() fills the paper's values. */
typedef struct sgp_options {
    double beta, theta;                          /* Armijo: 1e-4, 0.4 */
    double alpha0, alpha_min, alpha_max, tau1;   /* 1.3, 1e-5, 1e5, 0.5 */
    int m_alpha;                                 /* memory of the BB2 minimum, Eq.9: 3 */
    int alt_start;                               /* alternation only after this many iterations: 20 (A9) */
    int armijo_memory;                           /* M >= 1; 1 = monotone line search, the paper     (A15) */
    double L1, L2;                               /* scaling bounds of Eq.10 when adaptive_L = 0 */
    int adaptive_L;                              /* 1: bounds from one RL step */
    int max_iter;                                /* iteration cap (always active) */
    int stop_rule;                               /* sgp_stop */
    double tol;                                  /* Eq.24 */
    double disc_threshold;                       /* Eq.26: stop at the first k with 2 J0/(p #S) <= this (A6, A7) */
    double sigma_R;                              /* Eq.20 threshold defining R (A13) */
    int max_backtracks;                          /* A16 */
    int psf_origin;                              /* sgp_psf_origin */
    int init;                                    /* sgp_init */
    int refresh_every;                           /* A21 (sgp_* only): recompute A_j f and J0 from f after every n-th iteration; 0 = never */
    int strict;                                  /* A17: 1 = negative g is SGP_ERR_DATA instead of being clamped to 0 */
    int check_every;                             /* iterations enqueued between two host reads of the device status; 0 = auto */
    int tile_cols;                               /* tuning: spectrum tile width in columns (power of 2); 0 = auto */
    int rows_per_block;                          /* tuning: rows per CTA in the row-FFT kernels (power of 2); 0 = auto (depends on the grid and, for small
                                                    grids, on the number of problems of a batched plan; reductions are summed per CTA, so two plans agree
                                                    bit for bit only with equal rows_per_block) */
    int use_graph;                               /* bit 0 (default 1) = replay the iterations as CUDA graphs of 10 (kept across runs of a plan), else
                                                    plain stream launches; the only bit that may differ per run.  Experiment switches (plan level):
                                                    bit 1 = persistent column kernel, bit 2 / bit 3 = force the separate / the fused line-search
                                                    kernel (default: chosen by working set vs L2), bit 4 = never use the two-CTAs-per-SM column
                                                    kernel, bit 6 = RL / OSEM on the six separate launches of round 1 instead of the fused four,
                                                    bit 7 = never use the one-cluster-per-problem kernel of the small grids (sgp_*, one image,
                                                    128^2 / 256^2, constant background: the whole iteration in one kernel, csrc/small.cuh) */
    double rl_relax;                             /* rl_* only: exponent of the multiplicative relaxation, Eq.3:
                                                    f <- f o (W o sum_j A_j^T(g_j/(A_j f + b_j)))^rl_relax; 1 (default) = plain RL */
    double rl_linear;                            /* rl_* only: constant lambda_k of the linear relaxation, Eq.4:
                                                    f <- max(0, f - rl_linear f o (1 - W o sum_j A_j^T(g_j/(A_j f + b_j)))), the max being the paper's
                                                    non-negativity constraint (DESIGN reading A25); 1 (default) = plain RL; rl_relax and rl_linear both != 1 is SGP_ERR_ARG */
    int flux_constraint;                         /* sgp_* only: 1 = project on { f >= 0, sum_R f = c } in the metric D^-1 (Bonettini et al. 2009, cited
                                                    PAPER.md:60, :68; the paper itself uses f >= 0 only): y_i = max(0, x_i - mu D_i), mu by Newton steps on
                                                    the piecewise-linear equation sum y = c, each one reduction over f and the gradient, no FFT.  f(0) is
                                                    rescaled to the flux c (DESIGN reading A26).  0 (default) = off */
    double flux_value;                           /* c; <= 0 (default): c = (1/p) sum_j sum_S (g_j - b_j), clipped at 0 */
    double init_sigma;                           /* SGP_INIT_CONST_SMOOTH: standard deviation of the Gaussian in pixels (default 2) */
} sgp_options;

/* Result of a run.  The trace pointers are optional caller-allocated HOST arrays of max_iter+1 entries
 * (NULL = not wanted): trace_J[k] = J0(f(k)) for k = 0..iterations; trace_alpha[k], trace_lambda[k],
 * trace_rule[k] (0 = alpha0, 1 = BB1, 2 = Eq.9 minimum of BB2), trace_backtracks[k] describe the step
 * f(k) -> f(k+1).  RL fills trace_J only; OSEM evaluates J0 at the final iterate only (J0_final) and leaves trace_J zero.
 * force_alpha / force_lambda (HOST arrays of max_iter doubles, NaN = not forced, NULL = off) are a
 * TEST-ONLY replay mode: alpha_k / lambda_k are taken from them instead of the BB rules / Armijo loop. */
typedef struct sgp_result {
    int iterations;
    int stop_reason;            /* sgp_reason */
    double J0_final;
    double discrepancy_final;   /* 2 J0 / (p #S), Eq.26 */
    int total_backtracks;
    double L1_used, L2_used;
    long n_fft2;                /* 2-D transforms executed inside the iteration loop, COUNTED on the device by the column passes
                                   (2p+2 per SGP iteration and RL step, 4p per OSEM cycle, p+1 per refresh) */
    double setup_ms, loop_ms;   /* device time of the start-point phase and of the iteration loop (CUDA events) */
    long kernel_launches;       /* kernels of this library launched by the call */
    int fused_linesearch;       /* 1: the run used the fused line-search + ratio kernel; 2: the whole iteration ran inside the one-cluster-per-problem
                                   kernel of the small grids (csrc/small.cuh) */
    int status;                 /* sgp_status of THIS problem (batched runs return the first error; every problem reports its own here) */
    double *trace_J, *trace_alpha, *trace_lambda;
    int *trace_rule, *trace_backtracks;
    const double *force_alpha, *force_lambda;
    /* Eq.25: truth = the object f~ used to generate the data, a DEVICE array ny x nx in the dtype of the call
     * (input; NULL = not given).  When given, trace_err[k] = ||f(k) - f~||_2 / ||f~||_2 for k = 0..iterations (optional HOST array
     * of max_iter + 2 doubles; entry iterations + 1 holds the error of the discarded step after a SGP_STOP_MINERR stop) and
     * err_final = the error of the returned iterate.  SGP_STOP_MINERR stops at the first k whose next step would increase the
     * error and returns f(k) (sgp_*, rl_* and, per cycle, osem_*; DESIGN reading A27). */
    const void *truth;
    double *trace_err;
    double err_final;
} sgp_result;

typedef struct sgp_plan sgp_plan;

/* Kernel slots of the per-kernel timing (sgp_plan_set_profiling).  One SGP iteration is the seven launches
 * K1..K7 (SURVEY.md 8(d) schedule A), one RL round the six launches R1..R6. */
typedef enum {
    SGP_PROF_K1 = 0,  /* a10(q)+a1: lazy q_j += lambda u_j, ratio g/(Af+b) fused into the forward row FFT, p images */
    SGP_PROF_K2 = 1,  /* a2: column FFT -> sum_j conj(K^_j) x -> inverse column FFT                            */
    SGP_PROF_K3 = 2,  /* a10(f)+a3+a5+a6: inverse row FFT -> lazy f += lambda d, gradient, BB sums, step length  */
    SGP_PROF_K4 = 3,  /* a4+a7: scaling, projection, d, grad'd fused into the forward row FFT of d             */
    SGP_PROF_K5 = 4,  /* a8: column FFT -> x K^_j -> p inverse column FFTs                                      */
    SGP_PROF_K6 = 5,  /* a8+a9+a11: inverse row FFTs -> u_j = A_j d, J(lambda = 1), Armijo test, book-keeping    */
    SGP_PROF_K7 = 6,  /* a9 backtracks (elementwise; returns at once when lambda = 1 was accepted)                */
    SGP_PROF_R1 = 7,  /* RL: forward row FFT of f                                                               */
    SGP_PROF_R2 = 8,  /* RL: column pass x K^_j                                                                 */
    SGP_PROF_R3 = 9,  /* RL: inverse row FFTs -> q_j = A_j f, J0(f), stopping rules                             */
    SGP_PROF_R4 = 10, /* RL: ratio fused into the forward row FFTs                                              */
    SGP_PROF_R5 = 11, /* RL: column pass sum_j conj(K^_j)                                                       */
    SGP_PROF_R6 = 12, /* RL: inverse row FFT -> multiplicative update, Eq.1/13/21                               */
    SGP_PROF_SLOTS = 13
} sgp_prof_slot;

void sgp_options_default(sgp_options *opt);
void sgp_result_init(sgp_result *res);           /* zero everything, NULL traces */
const char *sgp_strerror(int status);
const char *sgp_version(void);
const char *sgp_last_cuda_error(void);
/* upper bound of the device workspace a plan of this shape allocates at creation (0 for unsupported arguments); the
 * per-run trace block (56 bytes per iteration of max_iter) comes on top.  sgp_plan_workspace_bytes: what a plan did allocate. */
size_t sgp_workspace_bytes(int kind, int p, int ny, int nx, int dtype);
size_t sgp_plan_workspace_bytes(const sgp_plan *plan);

/* ---- one-shot entry points: DEVICE pointers ------------------------------------------------------
 * g: detected image(s), psf: PSF(s) on the object grid (any positive scale; normalised to unit sum
 * inside), b_arr: background array(s) or NULL to use the constant(s) b_const,
 * f0: initial image (required for SGP_INIT_USER, else may be NULL), f_out: ny x nx result.
 * Each host thread keeps the plan of its last one-shot call (device workspace, twiddle tables, the instantiated
 * CUDA graph; the *_host calls also keep their staging buffer) and uses it again when the next call has the same
 * device, kind, p, grid, window, dtype and plan-time options (tile_cols, rows_per_block, use_graph, psf_origin,
 * sigma_R); the PSFs are transformed again in every call.  sgp_mosaic keeps its batched sub-domain plan and its
 * sub-image buffers the same way (a second slot, keyed also by the number of sub-domains).  sgp_release_cached_plans()
 * frees what the calling thread holds (the end of the thread does too); a call with another key frees the old plan first. */
void sgp_release_cached_plans(void);
int sgp_single(const void *g, const void *psf, const void *b_arr, double b_const, const void *f0,
               void *f_out, int ny, int nx, int dtype, const sgp_options *opt, sgp_result *res,
               void *stream);
int sgp_multi(int p, const void *const *g, const void *const *psf, const void *const *b_arr,
              const double *b_const, const void *f0, void *f_out, int ny, int nx, int dtype,
              const sgp_options *opt, sgp_result *res, void *stream);
/* Boundary-effect correction (Sect.2.4): g[j], b_arr[j] are sy x sx detected images occupying
 * S = [oy,oy+sy) x [ox,ox+sx) of the ny x nx object grid S-bar; psf[j], f0, f_out are ny x nx;
 * maskR_out (optional, ny*nx bytes, device) receives M_R of Eq.20; f_out is zero outside R. */
int sgp_boundary(int p, const void *const *g, const void *const *psf, const void *const *b_arr,
                 const double *b_const, int oy, int ox, int sy, int sx, int ny, int nx,
                 const void *f0, void *f_out, unsigned char *maskR_out, int dtype,
                 const sgp_options *opt, sgp_result *res, void *stream);
/* Richardson-Lucy on the same kernels (Eq.1 / Eq.13 / Eq.21); uses only the stopping fields,
 * init, psf_origin, sigma_R, strict and the tuning fields of opt. */
int rl_single(const void *g, const void *psf, const void *b_arr, double b_const, const void *f0,
              void *f_out, int ny, int nx, int dtype, const sgp_options *opt, sgp_result *res,
              void *stream);
int rl_multi(int p, const void *const *g, const void *const *psf, const void *const *b_arr,
             const double *b_const, const void *f0, void *f_out, int ny, int nx, int dtype,
             const sgp_options *opt, sgp_result *res, void *stream);
int rl_boundary(int p, const void *const *g, const void *const *psf, const void *const *b_arr,
                const double *b_const, int oy, int ox, int sy, int sx, int ny, int nx,
                const void *f0, void *f_out, unsigned char *maskR_out, int dtype,
                const sgp_options *opt, sgp_result *res, void *stream);
/* OSEM, Algorithm 2 of the paper: one iteration is a cycle over the p images,
 *   h <- h o A_j^T( g_j / (A_j h + b_j) ), j = 1..p (Eq.15);  boundary form: h <- (M_R/alpha_j) o h o ... (Eq.22),
 * 4p two-dimensional FFTs per iteration, on the kernels of rl_*.  Same arguments as rl_multi /
 * rl_boundary (device pointers).  opt->max_iter cycles are run: stop_rule must be SGP_STOP_MAXIT or -- the way the paper
 * stops OSEM, by the reconstruction error of Eq.25, which needs the true object in res->truth --
 * SGP_STOP_MINERR (the error is evaluated after every cycle; the first cycle that would increase it is discarded and the
 * iterate before it returned), else SGP_ERR_UNSUPPORTED.  J0 (Eq.12) is evaluated once, at the returned iterate
 * (res->J0_final); of the per-iteration traces only trace_err is filled.  (sgp_plan_run takes SGP_ALG_OSEM as well.) */
int osem_multi(int p, const void *const *g, const void *const *psf, const void *const *b_arr,
               const double *b_const, const void *f0, void *f_out, int ny, int nx, int dtype,
               const sgp_options *opt, sgp_result *res, void *stream);
int osem_boundary(int p, const void *const *g, const void *const *psf, const void *const *b_arr,
                  const double *b_const, int oy, int ox, int sy, int sx, int ny, int nx,
                  const void *f0, void *f_out, unsigned char *maskR_out, int dtype,
                  const sgp_options *opt, sgp_result *res, void *stream);

/* ---- the same calls with HOST pointers (copies inside the call; what bench.py times as e2e) -- */
int sgp_single_host(const void *g, const void *psf, const void *b_arr, double b_const, const void *f0,
                    void *f_out, int ny, int nx, int dtype, const sgp_options *opt, sgp_result *res,
                    void *stream);
int sgp_multi_host(int p, const void *const *g, const void *const *psf, const void *const *b_arr,
                   const double *b_const, const void *f0, void *f_out, int ny, int nx, int dtype,
                   const sgp_options *opt, sgp_result *res, void *stream);
int sgp_boundary_host(int p, const void *const *g, const void *const *psf, const void *const *b_arr,
                      const double *b_const, int oy, int ox, int sy, int sx, int ny, int nx,
                      const void *f0, void *f_out, unsigned char *maskR_out, int dtype,
                      const sgp_options *opt, sgp_result *res, void *stream);
int rl_single_host(const void *g, const void *psf, const void *b_arr, double b_const, const void *f0,
                   void *f_out, int ny, int nx, int dtype, const sgp_options *opt, sgp_result *res,
                   void *stream);
int rl_multi_host(int p, const void *const *g, const void *const *psf, const void *const *b_arr,
                  const double *b_const, const void *f0, void *f_out, int ny, int nx, int dtype,
                  const sgp_options *opt, sgp_result *res, void *stream);
int rl_boundary_host(int p, const void *const *g, const void *const *psf, const void *const *b_arr,
                     const double *b_const, int oy, int ox, int sy, int sx, int ny, int nx,
                     const void *f0, void *f_out, unsigned char *maskR_out, int dtype,
                     const sgp_options *opt, sgp_result *res, void *stream);

int osem_multi_host(int p, const void *const *g, const void *const *psf, const void *const *b_arr, const double *b_const,
                    const void *f0, void *f_out, int ny, int nx, int dtype, const sgp_options *opt, sgp_result *res,
                    void *stream);
int osem_boundary_host(int p, const void *const *g, const void *const *psf, const void *const *b_arr, const double *b_const,
                       int oy, int ox, int sy, int sx, int ny, int nx, const void *f0, void *f_out,
                       unsigned char *maskR_out, int dtype, const sgp_options *opt, sgp_result *res, void *stream);

/* ---- plan form: set-up once (workspace, twiddles, transfer functions, boundary weights), run many -- */
/* kind SINGLE requires p = 1; for SINGLE / MULTI the (oy,ox,sy,sx) arguments are ignored (S = S-bar). */
int sgp_plan_create(sgp_plan **plan, int kind, int p, int ny, int nx, int oy, int ox, int sy, int sx,
                    int dtype, const sgp_options *opt);
/* K^_j = FFT2 of the normalised, origin-shifted PSFs; for BOUNDARY plans also alpha_j, alpha, R and
 * M_R/alpha (Eq.19-20).  psf: HOST array of p DEVICE pointers (ny x nx each). */
int sgp_plan_set_psf(sgp_plan *plan, const void *const *psf, void *stream);
/* One reconstruction.  g, b_arr: HOST arrays of p DEVICE pointers (sy x sx each; b_arr or its entries may
 * be NULL -> b_const[j]).  algorithm: sgp_algorithm.  opt (may be NULL = the plan's options) replaces the
 * run-time options; the plan-level fields (tile_cols, rows_per_block, sigma_R, psf_origin, use_graph bits > 0) must
 * equal the plan's, else SGP_ERR_ARG. */
int sgp_plan_run(sgp_plan *plan, int algorithm, const void *const *g, const void *const *b_arr,
                 const double *b_const, const void *f0, void *f_out, const sgp_options *opt,
                 sgp_result *res, void *stream);
/* Batched plan: nb problems of the SAME geometry, dtype and PSFs solved at once -- the sub-domains of a
 * mosaic, or a stack of frames from one instrument.  Every kernel of the iteration is launched once
 * for all problems; each problem keeps its own step lengths, line search and stopping test.  g, b_arr, b_const: nb * p
 * entries, problem-major (problem i, image j at i * p + j); f0 (may be NULL unless init = USER), f_out, res: nb entries.
 * Not available in batched runs (SGP_ERR_UNSUPPORTED): flux_constraint, refresh_every, SGP_STOP_MINERR, the smoothed start
 * with boundary correction, forced step lengths.  A plan created with nb = 1 is an ordinary plan. */
int sgp_plan_create_batched(sgp_plan **plan, int nb, int kind, int p, int ny, int nx, int oy, int ox, int sy, int sx,
                            int dtype, const sgp_options *opt);
int sgp_plan_run_batched(sgp_plan *plan, int algorithm, const void *const *g, const void *const *b_arr,
                         const double *b_const, const void *const *f0, void *const *f_out, const sgp_options *opt,
                         sgp_result *res, void *stream);
/* Mosaic of sub-domain reconstructions with boundary-effect correction ("the 256 x 256 ... images are
 * partitioned into four partially overlapping 160 x 160 subdomains. Each ... is merged, by zero-padding, in a 256 x 256 array
 * ... From the four reconstructions 128 x 128, nonoverlapping images are extracted and the complete reconstructed image is
 * formed as a mosaic of them").  g[j]: the p detected images, Ny x Nx; psf[j]: ny x nx, the S-bar grid of every sub-problem;
 * the image is cut into ty x tx sub-images of sy x sx pixels (sub-image t starts at clamp(t N/T - (s - N/T)/2, 0, N - s)), each
 * placed in the centre of S-bar (DESIGN reading A29) and reconstructed by `algorithm` with Eq.16-23 -- all ty * tx at once, as
 * one batched plan -- and the (Ny/ty) x (Nx/tx) parts are put together in f_out (Ny x Nx).  res: ty * tx entries, row-major
 * over the tiles.  DEVICE pointers; the _host variant takes HOST pointers and copies inside the call. */
int sgp_mosaic(int algorithm, int p, const void *const *g, const void *const *psf, const double *b_const, int Ny, int Nx,
               int ty, int tx, int sy, int sx, int ny, int nx, void *f_out, int dtype, const sgp_options *opt,
               sgp_result *res, void *stream);
int sgp_mosaic_host(int algorithm, int p, const void *const *g, const void *const *psf, const double *b_const, int Ny, int Nx,
                    int ty, int tx, int sy, int sx, int ny, int nx, void *f_out, int dtype, const sgp_options *opt,
                    sgp_result *res, void *stream);
/* Operators of the plan, for callers and tests: out = A_j x (Eq.16) / out = A_j^T y (Eq.17),
 * all ny x nx DEVICE arrays on the S-bar grid. */
int sgp_plan_apply_A(sgp_plan *plan, int j, const void *x, void *out, void *stream);
int sgp_plan_apply_AT(sgp_plan *plan, int j, const void *y, void *out, void *stream);
/* M_R (bytes), alpha = sum_j alpha_j and #R of a plan whose PSFs are set; pointers may be NULL (DEVICE). */
int sgp_plan_get_mask(sgp_plan *plan, unsigned char *maskR_out, void *alpha_out, long *nR, void *stream);
/* Unnormalised 2-D real-to-complex DFT of an ny x nx DEVICE array with the plan's own FFT kernels, written
 * as ny x (nx/2+1) interleaved complex numbers (the layout of numpy.fft.rfft2); for tests and for the
 * in-run comparison with cuFFT.  sgp_plan_irfft2 is the inverse including the 1/(ny nx) factor. */
int sgp_plan_rfft2(sgp_plan *plan, const void *x, void *spec_out, void *stream);
int sgp_plan_irfft2(sgp_plan *plan, const void *spec_in, void *x_out, void *stream);
/* Per-kernel device timing of the iteration loop.  on = 1: every launch of the following sgp_plan_run calls
 * is bracketed by a CUDA event pair on `stream` (this costs a little throughput, so loop_ms of such a run is
 * not a benchmark figure).  sgp_plan_get_kernel_ms returns, for the last run, the summed duration in ms and
 * the number of launches of every slot: ms_sum and launches are HOST arrays of SGP_PROF_SLOTS entries. */
int sgp_plan_set_profiling(sgp_plan *plan, int on);
int sgp_plan_get_kernel_ms(sgp_plan *plan, double *ms_sum, long *launches);
void sgp_plan_destroy(sgp_plan *plan);

/* ---- an entry point that allocates nothing ----------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid it): the relative reconstruction error of Eq.25,
 *     *rho_out = || f - truth ||_2 / || truth ||_2      over n elements, accumulated in double,
 * the quantity sgp_plan_run reports as trace_err[0] / err_final for a run given sgp_result.truth, computed by the same
 * kernel arithmetic (same grid, same reduction order) but with its scratch -- per-CTA partial sums and the arrival
 * counter -- in a file-scope device array of 19 200 bytes that every GPU which loads the library holds until exit.
 *   f, truth : DEVICE pointers, n elements of `dtype` (SGP_F32 or SGP_F64), not written;
 *   rho_out  : DEVICE pointer to one double, written by the kernel (read it after the stream reaches that point);
 *   n        : 1 .. SGP_STATIC_MAX_ELEMS (4096 x 4096, the largest grid a plan accepts).  A larger n is rejected with
 *              SGP_ERR_ARG and sgp_last_cuda_error() then says so ("n exceeds SGP_STATIC_MAX_ELEMS ..."); nothing is launched;
 *   stream   : the cudaStream_t the kernel is enqueued on.  The call does not synchronise, and calls no cudaMalloc,
 *              cudaFree or allocating library routine (the array's device address is looked up once per device with
 *              cudaGetSymbolAddress, with that device current).
 * Every call on a device shares the array, which keeps the previous call's contents (the kernel overwrites the partials
 * before reading them and re-arms the counter itself).  Calls that OVERLAP on the GPU -- two streams with no ordering
 * between them, or two host threads -- race on it: keep the calls of one device on one stream or order them with events.
 * Returns SGP_OK, SGP_ERR_ARG (null pointer, n = 0 or beyond the maximum, bad dtype) or SGP_ERR_CUDA. */
#define SGP_STATIC_MAX_ELEMS (4096L * 4096L)
int sgp_rel_error_static(const void *f, const void *truth, size_t n, int dtype, double *rho_out, void *stream);
size_t sgp_rel_error_static_max(void);       /* SGP_STATIC_MAX_ELEMS of the loaded library */

#ifdef __cplusplus
}
#endif
#endif /* SGP_B200_H */
