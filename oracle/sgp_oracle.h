/*
 * sgp_oracle.h -- CPU ORACLE for the SGP / RL deconvolution path of arXiv:1210.2258.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or helper with the CUDA library (include/sgp.h, paper_1210_2258_b200/csrc).
 *
 * Plain C99, one real type per build: `double` (default, liboracle_f64.so) or `float`
 * (-DORACLE_FLOAT, liboracle_f32.so; diagnostics only).  All reductions are accumulated in
 * double in both builds.  All arrays are HOST pointers, row-major, contiguous.
 *
 * Citations are PAPER.md:<line> (the text of the paper under /root/reference) plus the
 * equation / algorithm; "A<n>" are the readings of SURVEY.md section 8(c), restated in DESIGN.md.
 */
#ifndef SGP_ORACLE_H
#define SGP_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

#ifdef ORACLE_FLOAT
typedef float oreal;
#define ORACLE_DTYPE 0
#else
typedef double oreal;
#define ORACLE_DTYPE 1
#endif

/* stopping rules, PAPER.md:279-298 (Sect. 3.3).  max_iter is always an additional cap. */
enum { ORACLE_STOP_MAXIT = 0, ORACLE_STOP_RELJ = 1, ORACLE_STOP_DISCREPANCY = 2,
       ORACLE_STOP_MINERR = 3 /* Eq.25: needs oracle_result.truth (reading A27) */ };
/* initial guess, PAPER.md:260-267 (Sect. 3.1) */
enum { ORACLE_INIT_USER = 0, ORACLE_INIT_CONST = 1, ORACLE_INIT_ZERO = 2, ORACLE_INIT_G = 3,
       ORACLE_INIT_CONST_SMOOTH = 4 /* the constant image convolved with a Gaussian, PAPER.md:264 (reading A28) */ };
/* where the PSF centre sits in the input array (reading A18) */
enum { ORACLE_PSF_CENTER = 0, ORACLE_PSF_CORNER = 1 };
/* stop_reason values in oracle_result (>0) and error codes (<0) */
enum { ORACLE_REASON_MAXIT = 1, ORACLE_REASON_RELJ = 2, ORACLE_REASON_DISCREPANCY = 3, ORACLE_REASON_MINERR = 4 };
enum { ORACLE_OK = 0, ORACLE_ERR_ARG = -1, ORACLE_ERR_PSF = -2, ORACLE_ERR_DATA = -3,
       ORACLE_ERR_ALLOC = -4, ORACLE_ERR_LINESEARCH = -6, ORACLE_ERR_NONFINITE = -7 };

typedef struct {
    /* line search: beta = 1e-4, theta = 0.4 */
    double beta, theta;
    /* step length: alpha0 = 1.3, alpha_min = 1e-5, alpha_max = 1e5, tau1 = 0.5, M_alpha = 3 */
    double alpha0, alpha_min, alpha_max, tau1;
    int m_alpha;
    int alt_start;      /* 20: alternation only after the first 20 iterations, PAPER.md:155 (A9) */
    int armijo_memory;  /* M >= 1; 1 = monotone (the paper); A15 */
    /* scaling bounds, Eq.10 / PAPER.md:273-275 */
    double L1, L2;
    int adaptive_L;     /* 1: one RL step + min-positive/max rule */
    /* stopping */
    int max_iter;
    int stop_rule;
    double tol;             /* Eq.24 */
    double disc_threshold;  /* Eq.26, "b close to 1" (A7) */
    double sigma_R;         /* Eq.20 threshold (A13) */
    int max_backtracks;     /* A16 */
    int psf_origin;
    int init;
    int refresh_every;      /* A21: 0 = never recompute A f from f */
    int strict;             /* A17: 1 = negative g is an error instead of being clamped */
    double rl_relax;        /* Eq.3: exponent of the multiplicative relaxation of RL; 1 = plain RL */
    double rl_linear;       /* Eq.4: constant lambda_k of the linear relaxation of RL; result projected on f >= 0; 1 = plain RL (reading A25) */
    int flux_constraint;    /* 1: SGP projects on { f >= 0, sum_R f = c } (Bonettini et al. 2009; reading A26) */
    double flux_value;      /* c; <= 0: c = (1/p) sum_j sum_S (g_j - b_j), clipped at 0 ("background-subtracted flux") */
    double init_sigma;      /* ORACLE_INIT_CONST_SMOOTH: standard deviation of the Gaussian in pixels (reading A28) */
} oracle_options;

typedef struct {
    int iterations;
    int stop_reason;
    double J0_final;
    double discrepancy_final;
    int total_backtracks;
    double L1_used, L2_used;
    long n_fft2;            /* 2-D transforms executed inside the iteration loop (pin P11) */
    /* optional caller-allocated traces, each of length max_iter+1 (may be NULL):
       J[k] = J0(f(k)), k = 0..iterations; alpha[k], lambda[k], rule[k], backtracks[k] describe
       the step f(k) -> f(k+1).  rule: 0 = alpha0, 1 = BB1, 2 = min of last M_alpha BB2 values. */
    double *trace_J, *trace_alpha, *trace_lambda;
    int *trace_rule, *trace_backtracks;
    /* TEST-ONLY forcing (NULL = off): alpha_k and lambda_k are taken from these arrays
       (length max_iter) instead of the BB rules / the Armijo loop -- pin P4 and the replay
       mode of SURVEY.md section 7. */
    const double *force_alpha, *force_lambda;
    /* Eq.25: truth = the object f~ on the S-bar grid (ny*nx oreal values, input, may be NULL);
       trace_err[k] = ||f(k) - f~||_2 / ||f~||_2, k = 0..iterations (+1 entry for the discarded step of
       ORACLE_STOP_MINERR), optional, length max_iter + 2; err_final = the value at the returned iterate. */
    const void *truth;
    double *trace_err;
    double err_final;
} oracle_result;

void oracle_options_default(oracle_options *o);
int oracle_dtype(void);

/* ---- building blocks exposed for the pins (tests/test_oracle_*.py) ---- */

/* 2-D DFT of an ny x nx complex array given as separate re/im planes.
   sign = -1 forward, +1 inverse (inverse includes the 1/(ny nx) factor). */
int oracle_fft2(int ny, int nx, int sign, const oreal *re, const oreal *im, oreal *ore, oreal *oim);
/* direct O(n^2) circular convolution, out[m] = sum_n K[(m-n) mod N] x[n]; K has its origin at (0,0) */
int oracle_conv2_direct(int ny, int nx, const oreal *K, const oreal *x, oreal *out);

typedef struct oracle_problem oracle_problem;
/* psf[j]: ny x nx over the whole grid S-bar.  masked = 0: periodic problem, M_S = M_R = 1,
   (oy,ox,sy,sx) ignored.  masked = 1: S = [oy,oy+sy) x [ox,ox+sx), M_R from Eq.20 with sigma_R. */
oracle_problem *oracle_problem_create(int p, int ny, int nx, const oreal *const *psf, int masked,
                                      int oy, int ox, int sy, int sx, double sigma_R, int psf_origin,
                                      int *err);
void oracle_problem_destroy(oracle_problem *P);
/* copies of alpha (Eq.19 summed over j), W = M_R/alpha and M_R; any pointer may be NULL */
int oracle_problem_get(const oracle_problem *P, oreal *alpha, oreal *W, unsigned char *MR,
                       long *nS, long *nR);
int oracle_apply_A(const oracle_problem *P, int j, const oreal *x, oreal *out);   /* Eq.16 */
int oracle_apply_AT(const oracle_problem *P, int j, const oreal *y, oreal *out);  /* Eq.17 */
int oracle_all_A(const oracle_problem *P, const oreal *x, oreal *const *out);     /* A_j x, all j, one FFT of x */
int oracle_sum_AT(const oracle_problem *P, const oreal *const *r, oreal *out);    /* sum_j A_j^T r_j, one inverse */
/* g, b, q: p arrays on the S-bar grid (values outside S ignored) */
double oracle_J0(const oracle_problem *P, const oreal *const *q, const oreal *const *g,
                 const oreal *const *b);                                          /* Eq.2 / Eq.12 */
int oracle_gradient(const oracle_problem *P, const oreal *f, const oreal *const *g,
                    const oreal *const *b, oreal *grad);                          /* Eq.11/14/18 */
int oracle_rl_step(const oracle_problem *P, const oreal *f, const oreal *const *g,
                   const oreal *const *b, oreal *f_out);                          /* Eq.1/13/21 */
int oracle_scaling(const oracle_problem *P, const oreal *f, double L1, double L2, oreal *D); /* Eq.10/23 */
int oracle_project(long n, const oreal *f, const oreal *grad, const oreal *D, double alpha,
                   oreal *y);                                                     /* Eq.6 */
int oracle_adaptive_bounds(long n, const oreal *y, double *L1, double *L2);
/* Projection on { y >= 0, sum y = c } in the metric of D^-1 (Bonettini et al. 2009, cited PAPER.md:60, :68):
   y = argmin sum_i (y_i - x_i)^2 / D_i  =>  y_i = max(0, x_i - mu D_i) with mu the root of sum_i y_i = c, found exactly
   by sorting the break points x_i / D_i.  Entries with D_i = 0 (outside R) are fixed at y_i = 0.  *mu (may be NULL). */
int oracle_project_flux(long n, const oreal *x, const oreal *D, double c, oreal *y, double *mu);
/* relative reconstruction error of Eq.25 in the l2 norm over the whole grid */
double oracle_rel_error(long n, const oreal *f, const oreal *truth);

/* BB step-length state machine */
typedef struct {
    double alpha_prev;  /* the alpha actually used at the previous iteration (A10) */
    double tau;
    double ring[16];    /* last M_alpha values of alpha^(2) */
    int ring_len, ring_pos, m_alpha;
} oracle_bb_state;
void oracle_bb_init(oracle_bb_state *s, const oracle_options *o);
/* a = s'D^-2 s, c = s'D^-1 z, e = s'D z, h = z'D^2 z; k = iteration index (k >= 1).
   Returns alpha_k; *rule = 1 (BB1) or 2 (ring minimum of BB2); a1/a2 (may be NULL) receive
   the safeguarded alpha^(1), alpha^(2). */
double oracle_bb_next(oracle_bb_state *s, const oracle_options *o, int k, double a, double c,
                      double e, double h, int *rule, double *a1, double *a2);

/* full runs on the S-bar grid: g, b are p arrays of ny*nx (zero / ignored outside S);
   f0 may be NULL unless init = USER; f_out has ny*nx entries */
int oracle_sgp_run(const oracle_problem *P, const oreal *const *g, const oreal *const *b,
                   const oreal *f0, const oracle_options *o, oracle_result *res, oreal *f_out);
int oracle_rl_run(const oracle_problem *P, const oreal *const *g, const oreal *const *b,
                  const oreal *f0, const oracle_options *o, oracle_result *res, oreal *f_out);
/* OSEM, Algorithm 2 / Eq.15 / Eq.22: max_iter cycles over the p images; J0 evaluated at the end only */
int oracle_osem_run(const oracle_problem *P, const oreal *const *g, const oreal *const *b,
                    const oreal *f0, const oracle_options *o, oracle_result *res, oreal *f_out);

/* ---- the paper-level entry points (SURVEY.md 8(b) signatures, host pointers) ---- */
int oracle_sgp_single(const oreal *g, const oreal *psf, const oreal *b_arr, double b_const,
                      const oreal *f0, oreal *f_out, int ny, int nx, int dtype,
                      const oracle_options *o, oracle_result *res);
int oracle_sgp_multi(int p, const oreal *const *g, const oreal *const *psf,
                     const oreal *const *b_arr, const double *b_const, const oreal *f0,
                     oreal *f_out, int ny, int nx, int dtype, const oracle_options *o,
                     oracle_result *res);
/* g[j], b_arr[j]: sy x sx (the detected images); psf[j], f0, f_out, maskR_out: ny x nx over S-bar */
int oracle_sgp_boundary(int p, const oreal *const *g, const oreal *const *psf,
                        const oreal *const *b_arr, const double *b_const, int oy, int ox, int sy,
                        int sx, int ny, int nx, const oreal *f0, oreal *f_out,
                        unsigned char *maskR_out, int dtype, const oracle_options *o,
                        oracle_result *res);
int oracle_rl_single(const oreal *g, const oreal *psf, const oreal *b_arr, double b_const,
                     const oreal *f0, oreal *f_out, int ny, int nx, int dtype,
                     const oracle_options *o, oracle_result *res);
int oracle_rl_multi(int p, const oreal *const *g, const oreal *const *psf,
                    const oreal *const *b_arr, const double *b_const, const oreal *f0,
                    oreal *f_out, int ny, int nx, int dtype, const oracle_options *o,
                    oracle_result *res);
int oracle_rl_boundary(int p, const oreal *const *g, const oreal *const *psf,
                       const oreal *const *b_arr, const double *b_const, int oy, int ox, int sy,
                       int sx, int ny, int nx, const oreal *f0, oreal *f_out,
                       unsigned char *maskR_out, int dtype, const oracle_options *o,
                       oracle_result *res);

int oracle_osem_multi(int p, const oreal *const *g, const oreal *const *psf,
                      const oreal *const *b_arr, const double *b_const, const oreal *f0,
                      oreal *f_out, int ny, int nx, int dtype, const oracle_options *o,
                      oracle_result *res);
int oracle_osem_boundary(int p, const oreal *const *g, const oreal *const *psf,
                         const oreal *const *b_arr, const double *b_const, int oy, int ox, int sy,
                         int sx, int ny, int nx, const oreal *f0, oreal *f_out,
                         unsigned char *maskR_out, int dtype, const oracle_options *o,
                         oracle_result *res);

#ifdef __cplusplus
}
#endif
#endif
