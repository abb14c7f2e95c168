/*
 * sgp_oracle.c -- CPU ORACLE for the SGP / RL deconvolution path of arXiv:1210.2258
 * (Prato, Cavicchioli, Zanni, Boccacci, Bertero).
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT (see sgp_oracle.h).  Plain, slow, written to be
 * checked against the paper by eye: a mixed-radix recursive FFT, full complex 2-D
 * spectra (no half-spectrum tricks), every operator and every step of Algorithm 1 in
 * the paper's order.  No blocking, no fusion.  Shares nothing with the CUDA library.
 *
 * Pins (tests/test_oracle_*.py, run with -m "not gpu"): P1..P11 of SURVEY.md 8(c), P12-P14 (OSEM, Eq.3, Eq.4),
 * P15 (start points, data cleaning, refresh_every), P16 (flux-constrained projection), P17 (Eq.25 stop),
 * P18 (Gaussian-smoothed constant start), P19 (mosaic of sub-domain reconstructions, oracle/__init__.py).
 * Parity unpinned (oracle and GPU library merely share the option):
 *   A7 (disc_threshold = 1), A9 (off-by-one of "first 20 iterations"), A13 (sigma_R),
 *   A14 (which mean the constant start uses), A16 (backtrack cap).
 */
#include "sgp_oracle.h"

#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>

#ifdef ORACLE_FLOAT
typedef float _Complex ocplx;
#else
typedef double _Complex ocplx;
#endif

#define PI_D 3.14159265358979323846264338327950288

/* ------------------------------------------------------------------------------------
 * FFT: recursive decimation in time for any n; the smallest prime factor p is split off
 * at every level (X[k + q m] = sum_r w_n^{rk} w_p^{rq} F_r[k], n = p m), primes are done
 * by the O(p^2) definition.  Twiddles come from one table w[k] = exp(sign 2 pi i k / N)
 * evaluated with cos/sin in double.
 * ------------------------------------------------------------------------------------ */

static long g_fft2_count = 0;

static int smallest_factor(int n)
{
    for (int p = 2; (long)p * p <= n; ++p)
        if (n % p == 0) return p;
    return n;
}

static void fft_rec(int n, const ocplx *in, int is, ocplx *out, int N, const ocplx *w)
{
    if (n == 1) { out[0] = in[0]; return; }
    int p = smallest_factor(n), m = n / p;
    for (int r = 0; r < p; ++r) fft_rec(m, in + (long)r * is, is * p, out + (long)r * m, N, w);
    ocplx t[p], y[p];
    int wn = N / n;   /* w_n^k = w[k * N/n] */
    int wp = N / p;   /* w_p^k = w[k * N/p] */
    for (int k = 0; k < m; ++k) {
        for (int r = 0; r < p; ++r) t[r] = out[(long)r * m + k] * w[((long)r * k % n) * wn];
        for (int q = 0; q < p; ++q) {
            ocplx s = 0;
            for (int r = 0; r < p; ++r) s += t[r] * w[((long)r * q % p) * wp];
            y[q] = s;
        }
        for (int q = 0; q < p; ++q) out[(long)q * m + k] = y[q];
    }
}

static ocplx *make_twiddles(int N, int sign)
{
    ocplx *w = (ocplx *)malloc(sizeof(ocplx) * (size_t)N);
    if (!w) return NULL;
    for (int k = 0; k < N; ++k) {
        double a = sign * 2.0 * PI_D * (double)k / (double)N;
        w[k] = (oreal)cos(a) + (oreal)sin(a) * I;
    }
    return w;
}

/* in-place 2-D DFT of a[ny][nx]; sign -1 forward, +1 inverse (scaled by 1/(ny nx)) */
static int fft2_inplace(int ny, int nx, int sign, ocplx *a)
{
    ocplx *wx = make_twiddles(nx, sign), *wy = make_twiddles(ny, sign);
    if (!wx || !wy) { free(wx); free(wy); return ORACLE_ERR_ALLOC; }
    int bad = 0;
#pragma omp parallel
    {
        int nmax = nx > ny ? nx : ny;
        ocplx *bi = (ocplx *)malloc(sizeof(ocplx) * (size_t)nmax);
        ocplx *bo = (ocplx *)malloc(sizeof(ocplx) * (size_t)nmax);
        if (!bi || !bo) {
#pragma omp atomic write
            bad = 1;
        } else {
#pragma omp for schedule(static)
            for (int y = 0; y < ny; ++y) {           /* rows */
                memcpy(bi, a + (size_t)y * nx, sizeof(ocplx) * (size_t)nx);
                fft_rec(nx, bi, 1, bo, nx, wx);
                memcpy(a + (size_t)y * nx, bo, sizeof(ocplx) * (size_t)nx);
            }
#pragma omp for schedule(static)
            for (int x = 0; x < nx; ++x) {           /* columns */
                for (int y = 0; y < ny; ++y) bi[y] = a[(size_t)y * nx + x];
                fft_rec(ny, bi, 1, bo, ny, wy);
                for (int y = 0; y < ny; ++y) a[(size_t)y * nx + x] = bo[y];
            }
        }
        free(bi); free(bo);
    }
    free(wx); free(wy);
    if (bad) return ORACLE_ERR_ALLOC;
    if (sign > 0) {
        oreal sc = (oreal)(1.0 / ((double)ny * (double)nx));
        for (size_t i = 0; i < (size_t)ny * nx; ++i) a[i] *= sc;
    }
    g_fft2_count++;
    return ORACLE_OK;
}

int oracle_dtype(void) { return ORACLE_DTYPE; }

int oracle_fft2(int ny, int nx, int sign, const oreal *re, const oreal *im, oreal *ore, oreal *oim)
{
    if (ny < 1 || nx < 1 || !re || !ore || !oim || (sign != 1 && sign != -1)) return ORACLE_ERR_ARG;
    size_t n = (size_t)ny * nx;
    ocplx *a = (ocplx *)malloc(sizeof(ocplx) * n);
    if (!a) return ORACLE_ERR_ALLOC;
    for (size_t i = 0; i < n; ++i) a[i] = re[i] + (im ? im[i] : (oreal)0) * I;
    int rc = fft2_inplace(ny, nx, sign, a);
    for (size_t i = 0; i < n; ++i) { ore[i] = creal(a[i]); oim[i] = cimag(a[i]); }
    free(a);
    return rc;
}

int oracle_conv2_direct(int ny, int nx, const oreal *K, const oreal *x, oreal *out)
{
    if (ny < 1 || nx < 1 || !K || !x || !out) return ORACLE_ERR_ARG;
    for (int my = 0; my < ny; ++my)
        for (int mx = 0; mx < nx; ++mx) {
            double s = 0.0;
            for (int qy = 0; qy < ny; ++qy)
                for (int qx = 0; qx < nx; ++qx) {
                    int ky = ((my - qy) % ny + ny) % ny, kx = ((mx - qx) % nx + nx) % nx;
                    s += (double)K[(size_t)ky * nx + kx] * (double)x[(size_t)qy * nx + qx];
                }
            out[(size_t)my * nx + mx] = (oreal)s;
        }
    return ORACLE_OK;
}

/* ------------------------------------------------------------------------------------
 * The imaging problem: grid S-bar (ny x nx), image domain S (rectangle), object domain R,
 * transfer functions K^_j.  PAPER.md:216-238 (Sect. 2.4); unmasked problems have
 * M_S = M_R = 1 (Sect. 2.2, 2.3).
 * ------------------------------------------------------------------------------------ */
struct oracle_problem {
    int p, ny, nx;
    int masked, oy, ox, sy, sx;
    size_t n;
    long nS, nR;
    ocplx **Khat;        /* p transfer functions, full ny x nx */
    unsigned char *MS;   /* 1 on S */
    unsigned char *MR;   /* 1 on R */
    oreal *alpha;        /* sum_j alpha_j, Eq.19 (== p when unmasked) */
    oreal *W;            /* M_R / alpha, Eq.21/23 (== 1/p when unmasked) */
};

void oracle_problem_destroy(oracle_problem *P)
{
    if (!P) return;
    if (P->Khat) for (int j = 0; j < P->p; ++j) free(P->Khat[j]);
    free(P->Khat); free(P->MS); free(P->MR); free(P->alpha); free(P->W); free(P);
}

/* K^_j = FFT2 of the PSF normalised to unit volume over S-bar and
   circularly shifted so that its centre sits at index (0,0) (reading A18). */
static int make_otf(int ny, int nx, const oreal *psf, int origin, ocplx *Khat)
{
    size_t n = (size_t)ny * nx;
    double sum = 0.0;
    for (size_t i = 0; i < n; ++i) {
        if (!isfinite((double)psf[i])) return ORACLE_ERR_PSF;
        sum += (double)psf[i];
    }
    if (!(sum > 0.0) || !isfinite(sum)) return ORACLE_ERR_PSF;
    int cy = origin == ORACLE_PSF_CENTER ? ny / 2 : 0, cx = origin == ORACLE_PSF_CENTER ? nx / 2 : 0;
    for (int y = 0; y < ny; ++y)
        for (int x = 0; x < nx; ++x) {
            int ty = ((y - cy) % ny + ny) % ny, tx = ((x - cx) % nx + nx) % nx;
            Khat[(size_t)ty * nx + tx] = (oreal)((double)psf[(size_t)y * nx + x] / sum);
        }
    return fft2_inplace(ny, nx, -1, Khat);
}

oracle_problem *oracle_problem_create(int p, int ny, int nx, const oreal *const *psf, int masked,
                                      int oy, int ox, int sy, int sx, double sigma_R, int psf_origin,
                                      int *err)
{
    int rc = ORACLE_OK;
    oracle_problem *P = NULL;
    if (p < 1 || ny < 1 || nx < 1 || !psf) { rc = ORACLE_ERR_ARG; goto fail; }
    if (masked && (oy < 0 || ox < 0 || sy < 1 || sx < 1 || oy + sy > ny || ox + sx > nx)) {
        rc = ORACLE_ERR_ARG; goto fail;
    }
    P = (oracle_problem *)calloc(1, sizeof(*P));
    if (!P) { rc = ORACLE_ERR_ALLOC; goto fail; }
    P->p = p; P->ny = ny; P->nx = nx; P->n = (size_t)ny * nx; P->masked = masked;
    if (masked) { P->oy = oy; P->ox = ox; P->sy = sy; P->sx = sx; }
    else        { P->oy = 0; P->ox = 0; P->sy = ny; P->sx = nx; }
    size_t n = P->n;
    P->Khat = (ocplx **)calloc((size_t)p, sizeof(ocplx *));
    P->MS = (unsigned char *)calloc(n, 1);
    P->MR = (unsigned char *)calloc(n, 1);
    P->alpha = (oreal *)calloc(n, sizeof(oreal));
    P->W = (oreal *)calloc(n, sizeof(oreal));
    if (!P->Khat || !P->MS || !P->MR || !P->alpha || !P->W) { rc = ORACLE_ERR_ALLOC; goto fail; }
    for (int j = 0; j < p; ++j) {
        if (!psf[j]) { rc = ORACLE_ERR_ARG; goto fail; }
        P->Khat[j] = (ocplx *)malloc(sizeof(ocplx) * n);
        if (!P->Khat[j]) { rc = ORACLE_ERR_ALLOC; goto fail; }
        rc = make_otf(ny, nx, psf[j], psf_origin, P->Khat[j]);
        if (rc) goto fail;
    }
    for (int y = P->oy; y < P->oy + P->sy; ++y)
        for (int x = P->ox; x < P->ox + P->sx; ++x) P->MS[(size_t)y * nx + x] = 1;
    P->nS = (long)P->sy * P->sx;

    if (!masked) {
        /* alpha == p and W == 1/p analytically (unit-volume periodic PSFs) */
        for (size_t i = 0; i < n; ++i) { P->MR[i] = 1; P->alpha[i] = (oreal)p; P->W[i] = (oreal)(1.0 / p); }
        P->nR = (long)n;
    } else {
        /* alpha_j(n) = sum_m K_j(m - n) M_S(m)   (Eq.19 in reading A5: no data factor),
           i.e. the correlation of K_j with M_S = IFFT2(conj(K^_j) FFT2(M_S));
           alpha = sum_j alpha_j;  R = { n : alpha_j(n) >= sigma for all j }  (Eq.20) */
        ocplx *ms = (ocplx *)malloc(sizeof(ocplx) * n), *t = (ocplx *)malloc(sizeof(ocplx) * n);
        if (!ms || !t) { free(ms); free(t); rc = ORACLE_ERR_ALLOC; goto fail; }
        for (size_t i = 0; i < n; ++i) { ms[i] = (oreal)P->MS[i]; P->MR[i] = 1; }
        rc = fft2_inplace(ny, nx, -1, ms);
        for (int j = 0; j < p && !rc; ++j) {
            for (size_t i = 0; i < n; ++i) t[i] = conj(P->Khat[j][i]) * ms[i];
            rc = fft2_inplace(ny, nx, +1, t);
            for (size_t i = 0; i < n; ++i) {
                oreal aj = creal(t[i]);
                P->alpha[i] += aj;
                if (!((double)aj >= sigma_R)) P->MR[i] = 0;
            }
        }
        free(ms); free(t);
        if (rc) goto fail;
        P->nR = 0;
        for (size_t i = 0; i < n; ++i) {
            if (P->MR[i]) { P->W[i] = (oreal)1 / P->alpha[i]; P->nR++; }
            else          { P->W[i] = 0; }
        }
    }
    if (err) *err = ORACLE_OK;
    return P;
fail:
    oracle_problem_destroy(P);
    if (err) *err = rc;
    return NULL;
}

int oracle_problem_get(const oracle_problem *P, oreal *alpha, oreal *W, unsigned char *MR,
                       long *nS, long *nR)
{
    if (!P) return ORACLE_ERR_ARG;
    if (alpha) memcpy(alpha, P->alpha, sizeof(oreal) * P->n);
    if (W) memcpy(W, P->W, sizeof(oreal) * P->n);
    if (MR) memcpy(MR, P->MR, P->n);
    if (nS) *nS = P->nS;
    if (nR) *nR = P->nR;
    return ORACLE_OK;
}

/* (A_j x)(m) = M_S(m) sum_n K_j(m-n) M_R(n) x(n)            Eq.16 */
int oracle_apply_A(const oracle_problem *P, int j, const oreal *x, oreal *out)
{
    if (!P || j < 0 || j >= P->p || !x || !out) return ORACLE_ERR_ARG;
    size_t n = P->n;
    ocplx *t = (ocplx *)malloc(sizeof(ocplx) * n);
    if (!t) return ORACLE_ERR_ALLOC;
    for (size_t i = 0; i < n; ++i) t[i] = P->MR[i] ? x[i] : (oreal)0;
    int rc = fft2_inplace(P->ny, P->nx, -1, t);
    if (!rc) {
        for (size_t i = 0; i < n; ++i) t[i] *= P->Khat[j][i];
        rc = fft2_inplace(P->ny, P->nx, +1, t);
    }
    for (size_t i = 0; i < n; ++i) out[i] = P->MS[i] ? (oreal)creal(t[i]) : (oreal)0;
    free(t);
    return rc;
}

/* (A_j^T y)(n) = M_R(n) sum_m K_j(m-n) M_S(m) y(m)          Eq.17 */
int oracle_apply_AT(const oracle_problem *P, int j, const oreal *y, oreal *out)
{
    if (!P || j < 0 || j >= P->p || !y || !out) return ORACLE_ERR_ARG;
    size_t n = P->n;
    ocplx *t = (ocplx *)malloc(sizeof(ocplx) * n);
    if (!t) return ORACLE_ERR_ALLOC;
    for (size_t i = 0; i < n; ++i) t[i] = P->MS[i] ? y[i] : (oreal)0;
    int rc = fft2_inplace(P->ny, P->nx, -1, t);
    if (!rc) {
        for (size_t i = 0; i < n; ++i) t[i] *= conj(P->Khat[j][i]);
        rc = fft2_inplace(P->ny, P->nx, +1, t);
    }
    for (size_t i = 0; i < n; ++i) out[i] = P->MR[i] ? (oreal)creal(t[i]) : (oreal)0;
    free(t);
    return rc;
}

/* A_j x for all j with FFT2(M_R x) computed once: 1 forward + p inverse transforms.
   Same linear maps as oracle_apply_A (tests pin the equality). */
int oracle_all_A(const oracle_problem *P, const oreal *x, oreal *const *out)
{
    if (!P || !x || !out) return ORACLE_ERR_ARG;
    size_t n = P->n;
    ocplx *X = (ocplx *)malloc(sizeof(ocplx) * n), *t = (ocplx *)malloc(sizeof(ocplx) * n);
    if (!X || !t) { free(X); free(t); return ORACLE_ERR_ALLOC; }
    for (size_t i = 0; i < n; ++i) X[i] = P->MR[i] ? x[i] : (oreal)0;
    int rc = fft2_inplace(P->ny, P->nx, -1, X);
    for (int j = 0; j < P->p && !rc; ++j) {
        for (size_t i = 0; i < n; ++i) t[i] = X[i] * P->Khat[j][i];
        rc = fft2_inplace(P->ny, P->nx, +1, t);
        for (size_t i = 0; i < n; ++i) out[j][i] = P->MS[i] ? (oreal)creal(t[i]) : (oreal)0;
    }
    free(X); free(t);
    return rc;
}

/* sum_j A_j^T r_j with the sum over j taken in Fourier space: p forward + 1 inverse
   transform (linearity of the inverse DFT; tests pin the equality with the p separate
   applications of Eq.17). */
int oracle_sum_AT(const oracle_problem *P, const oreal *const *r, oreal *out)
{
    if (!P || !r || !out) return ORACLE_ERR_ARG;
    size_t n = P->n;
    ocplx *acc = (ocplx *)calloc(n, sizeof(ocplx)), *t = (ocplx *)malloc(sizeof(ocplx) * n);
    if (!acc || !t) { free(acc); free(t); return ORACLE_ERR_ALLOC; }
    int rc = ORACLE_OK;
    for (int j = 0; j < P->p && !rc; ++j) {
        for (size_t i = 0; i < n; ++i) t[i] = P->MS[i] ? r[j][i] : (oreal)0;
        rc = fft2_inplace(P->ny, P->nx, -1, t);
        for (size_t i = 0; i < n; ++i) acc[i] += conj(P->Khat[j][i]) * t[i];
    }
    if (!rc) rc = fft2_inplace(P->ny, P->nx, +1, acc);
    for (size_t i = 0; i < n; ++i) out[i] = P->MR[i] ? (oreal)creal(acc[i]) : (oreal)0;
    free(acc); free(t);
    return rc;
}

/* One summand of the KL divergence, Eq.2: g ln(g/y) + y - g, with y = Af + b.
   Reading A17: g = 0 gives y (the limit g -> 0+); for g > 0 the value is evaluated as
   g (t - log1p(t)), t = (y - g)/g, which is the same number without cancellation;
   y <= 0 (only possible through round-off when b = 0): log term taken as 0. */
static double kl_term(double g, double y)
{
    if (!(g > 0.0)) return y;
    if (!(y > 0.0)) return y - g;
    double t = (y - g) / g;
    return g * (t - log1p(t));
}

/* ratio g/(Af+b) (Eq.1/11); 0 where the denominator is <= 0 (A17) */
static oreal ratio_term(oreal g, oreal y)
{
    return (y > 0) ? g / y : (oreal)0;
}

/* J0 = sum_j sum_{m in S} kl(g_j(m), q_j(m) + b_j(m))       Eq.2 / Eq.12 (A4), summed over S (A12) */
double oracle_J0(const oracle_problem *P, const oreal *const *q, const oreal *const *g,
                 const oreal *const *b)
{
    double J = 0.0;
    for (int j = 0; j < P->p; ++j)
        for (size_t i = 0; i < P->n; ++i)
            if (P->MS[i]) J += kl_term((double)g[j][i], (double)q[j][i] + (double)b[j][i]);
    return J;
}

/* grad J0 = alpha - sum_j A_j^T (g_j / (A_j f + b_j)) on R, 0 elsewhere.
   Eq.11 (alpha = 1), Eq.14 (alpha = p), Eq.18 (alpha = sum_j A_j^T 1). */
static int gradient_from_q(const oracle_problem *P, oreal *const *q, const oreal *const *g,
                           const oreal *const *b, oreal *const *r /*scratch*/, oreal *grad)
{
    for (int j = 0; j < P->p; ++j)
        for (size_t i = 0; i < P->n; ++i)
            r[j][i] = P->MS[i] ? ratio_term(g[j][i], q[j][i] + b[j][i]) : (oreal)0;
    int rc = oracle_sum_AT(P, (const oreal *const *)r, grad);   /* grad <- w */
    if (rc) return rc;
    for (size_t i = 0; i < P->n; ++i) grad[i] = P->MR[i] ? P->alpha[i] - grad[i] : (oreal)0;
    return ORACLE_OK;
}

static oreal **alloc_planes(int p, size_t n)
{
    oreal **a = (oreal **)calloc((size_t)p, sizeof(oreal *));
    if (!a) return NULL;
    for (int j = 0; j < p; ++j) {
        a[j] = (oreal *)calloc(n, sizeof(oreal));
        if (!a[j]) { for (int i = 0; i < j; ++i) free(a[i]); free(a); return NULL; }
    }
    return a;
}
static void free_planes(oreal **a, int p)
{
    if (!a) return;
    for (int j = 0; j < p; ++j) free(a[j]);
    free(a);
}

int oracle_gradient(const oracle_problem *P, const oreal *f, const oreal *const *g,
                    const oreal *const *b, oreal *grad)
{
    if (!P || !f || !g || !b || !grad) return ORACLE_ERR_ARG;
    oreal **q = alloc_planes(P->p, P->n), **r = alloc_planes(P->p, P->n);
    int rc = (!q || !r) ? ORACLE_ERR_ALLOC : oracle_all_A(P, f, q);
    if (!rc) rc = gradient_from_q(P, q, g, b, r, grad);
    free_planes(q, P->p); free_planes(r, P->p);
    return rc;
}

/* f(k+1) = (M_R/alpha) o f(k) o sum_j A_j^T (g_j/(A_j f(k) + b_j))    Eq.1 / Eq.13 / Eq.21 */
static int rl_update_from_q(const oracle_problem *P, const oreal *f, oreal *const *q,
                            const oreal *const *g, const oreal *const *b, oreal *const *r,
                            oreal *w, oreal *f_out)
{
    for (int j = 0; j < P->p; ++j)
        for (size_t i = 0; i < P->n; ++i)
            r[j][i] = P->MS[i] ? ratio_term(g[j][i], q[j][i] + b[j][i]) : (oreal)0;
    int rc = oracle_sum_AT(P, (const oreal *const *)r, w);
    if (rc) return rc;
    for (size_t i = 0; i < P->n; ++i) f_out[i] = P->W[i] * f[i] * w[i];
    return ORACLE_OK;
}

int oracle_rl_step(const oracle_problem *P, const oreal *f, const oreal *const *g,
                   const oreal *const *b, oreal *f_out)
{
    if (!P || !f || !g || !b || !f_out) return ORACLE_ERR_ARG;
    oreal **q = alloc_planes(P->p, P->n), **r = alloc_planes(P->p, P->n);
    oreal *w = (oreal *)malloc(sizeof(oreal) * P->n);
    int rc = (!q || !r || !w) ? ORACLE_ERR_ALLOC : oracle_all_A(P, f, q);
    if (!rc) rc = rl_update_from_q(P, f, q, g, b, r, w, f_out);
    free_planes(q, P->p); free_planes(r, P->p); free(w);
    return rc;
}

/* D = (M_R/alpha) o min(L2, max(L1, f))        Eq.10 / Eq.23; unmasked W = 1/p (A8) */
int oracle_scaling(const oracle_problem *P, const oreal *f, double L1, double L2, oreal *D)
{
    if (!P || !f || !D) return ORACLE_ERR_ARG;
    for (size_t i = 0; i < P->n; ++i) {
        oreal c = f[i];
        if (c < (oreal)L1) c = (oreal)L1;
        if (c > (oreal)L2) c = (oreal)L2;
        D[i] = P->W[i] * c;
    }
    return ORACLE_OK;
}

/* y = P+(f - alpha D grad): projection onto the non-negative orthant      Eq.6 */
int oracle_project(long n, const oreal *f, const oreal *grad, const oreal *D, double alpha, oreal *y)
{
    if (n < 0 || !f || !grad || !D || !y) return ORACLE_ERR_ARG;
    for (long i = 0; i < n; ++i) {
        oreal v = f[i] - (oreal)alpha * D[i] * grad[i];
        y[i] = v > 0 ? v : (oreal)0;
    }
    return ORACLE_OK;
}

/* y_min = smallest strictly positive value, y_max = largest value (A19) */
int oracle_adaptive_bounds(long n, const oreal *y, double *L1, double *L2)
{
    if (n < 1 || !y || !L1 || !L2) return ORACLE_ERR_ARG;
    double ymin = INFINITY, ymax = -INFINITY;
    for (long i = 0; i < n; ++i) {
        double v = (double)y[i];
        if (v > 0.0 && v < ymin) ymin = v;
        if (v > ymax) ymax = v;
    }
    if (!(ymin < INFINITY) || !(ymax > 0.0)) return ORACLE_ERR_DATA;
    if (ymax / ymin < 50.0) { *L1 = ymin / 10.0; *L2 = ymax * 10.0; }
    else                    { *L1 = ymin;        *L2 = ymax; }
    return ORACLE_OK;
}

/* Projection on the set { y >= 0, sum_i y_i = c } in the norm induced by D^-1 -- the "additional flux
   constraint" of Bonettini et al. (2009) that the paper mentions and does not use (reading A26).
   KKT conditions of  min sum_i (y_i - x_i)^2 / (2 D_i)  s.t. y >= 0, sum y = c:
       y_i = max(0, x_i - mu D_i),   mu such that  h(mu) = sum_i max(0, x_i - mu D_i) = c.
   h is continuous, piecewise linear and non-increasing in mu with break points t_i = x_i / D_i.  The root is found
   exactly: sort the break points in decreasing order; with the m largest active, h(mu) = SX_m - mu SD_m, so the
   candidate mu_m = (SX_m - c) / SD_m is the root iff t_(m) > mu_m >= t_(m+1).  Entries with D_i = 0 (pixels outside
   R, Eq.23) cannot move: y_i = 0 there. */
typedef struct { double t; long i; } brk_t;
static int brk_cmp(const void *a, const void *b)
{
    double ta = ((const brk_t *)a)->t, tb = ((const brk_t *)b)->t;
    if (ta > tb) return -1;
    if (ta < tb) return 1;
    long ia = ((const brk_t *)a)->i, ib = ((const brk_t *)b)->i;
    return ia < ib ? -1 : (ia > ib ? 1 : 0);
}
int oracle_project_flux(long n, const oreal *x, const oreal *D, double c, oreal *y, double *mu_out)
{
    if (n < 1 || !x || !D || !y || !(c >= 0.0)) return ORACLE_ERR_ARG;
    brk_t *bk = (brk_t *)malloc(sizeof(brk_t) * (size_t)n);
    if (!bk) return ORACLE_ERR_ALLOC;
    long m = 0;
    for (long i = 0; i < n; ++i)
        if (D[i] > 0) { bk[m].t = (double)x[i] / (double)D[i]; bk[m].i = i; m++; }
    if (m == 0) { free(bk); return ORACLE_ERR_DATA; }
    qsort(bk, (size_t)m, sizeof(brk_t), brk_cmp);
    double SX = 0.0, SD = 0.0, mu = 0.0;
    int found = 0;
    for (long k = 0; k < m; ++k) {
        SX += (double)x[bk[k].i]; SD += (double)D[bk[k].i];
        double cand = (SX - c) / SD;
        double tnext = (k + 1 < m) ? bk[k + 1].t : -INFINITY;
        if (cand < bk[k].t && cand >= tnext) { mu = cand; found = 1; break; }
    }
    if (!found) {
        /* c = 0 with all x <= 0 etc.: the largest break point makes every entry inactive, h = 0 */
        if (c == 0.0) { mu = bk[0].t; found = 1; }
    }
    free(bk);
    if (!found) return ORACLE_ERR_DATA;
    for (long i = 0; i < n; ++i) {
        if (!(D[i] > 0)) { y[i] = 0; continue; }
        oreal v = x[i] - (oreal)mu * D[i];
        y[i] = v > 0 ? v : (oreal)0;
    }
    if (mu_out) *mu_out = mu;
    return ORACLE_OK;
}

/* rho = ||f - f~||_2 / ||f~||_2, Eq.25 with the l2 norm the paper's code uses */
double oracle_rel_error(long n, const oreal *f, const oreal *truth)
{
    double num = 0.0, den = 0.0;
    for (long i = 0; i < n; ++i) {
        double e = (double)f[i] - (double)truth[i];
        num += e * e; den += (double)truth[i] * (double)truth[i];
    }
    return sqrt(num) / sqrt(den);
}

/* ------------------------------------------------------------------------------------
 * Step-length selection.
 * ------------------------------------------------------------------------------------ */
void oracle_options_default(oracle_options *o)
{
    memset(o, 0, sizeof(*o));
    o->beta = 1e-4; o->theta = 0.4;
    o->alpha0 = 1.3; o->alpha_min = 1e-5; o->alpha_max = 1e5;
    o->tau1 = 0.5; o->m_alpha = 3;
    o->alt_start = 20;
    o->armijo_memory = 1;                                             /* PAPER.md:83 (monotone) */
    o->L1 = 1e-10; o->L2 = 1e10; o->adaptive_L = 1;
    o->max_iter = 100; o->stop_rule = ORACLE_STOP_MAXIT; o->tol = 1e-5;
    o->disc_threshold = 1.0; o->sigma_R = 1e-2; o->max_backtracks = 30;
    o->psf_origin = ORACLE_PSF_CENTER; o->init = ORACLE_INIT_CONST;
    o->refresh_every = 0; o->strict = 0; o->rl_relax = 1.0; o->rl_linear = 1.0;
    o->flux_constraint = 0; o->flux_value = 0.0; o->init_sigma = 2.0;
}

void oracle_bb_init(oracle_bb_state *s, const oracle_options *o)
{
    memset(s, 0, sizeof(*s));
    s->alpha_prev = o->alpha0;
    s->tau = o->tau1;
    s->m_alpha = o->m_alpha < 1 ? 1 : (o->m_alpha > 16 ? 16 : o->m_alpha);
}

double oracle_bb_next(oracle_bb_state *s, const oracle_options *o, int k, double a, double c,
                      double e, double h, int *rule, double *a1out, double *a2out)
{
    double a1, a2;
    /* IF s'D^-1 z <= 0 THEN alpha1 = min{10 alpha_{k-1}, alpha_max}
       ELSE alpha1 = min{alpha_max, max{alpha_min, BB1}},  BB1 = s'D^-2 s / s'D^-1 z   (Eq.7) */
    if (c <= 0.0) a1 = fmin(10.0 * s->alpha_prev, o->alpha_max);
    else          a1 = fmin(o->alpha_max, fmax(o->alpha_min, a / c));
    /* same with s'D z and BB2 = s'D z / z'D^2 z                                        (Eq.8) */
    if (e <= 0.0) a2 = fmin(10.0 * s->alpha_prev, o->alpha_max);
    else          a2 = fmin(o->alpha_max, fmax(o->alpha_min, e / h));
    /* ring of the last M_alpha values of alpha^(2) (Eq.9; A20: fewer at the start) */
    s->ring[s->ring_pos] = a2;
    s->ring_pos = (s->ring_pos + 1) % s->m_alpha;
    if (s->ring_len < s->m_alpha) s->ring_len++;
    double m = s->ring[0];
    for (int i = 1; i < s->ring_len; ++i) m = fmin(m, s->ring[i]);
    double alpha;
    if (k <= o->alt_start) {
        /* first 20 iterations: the Eq.9 value, no alternation, tau untouched (A9) */
        alpha = m; *rule = 2;
    } else if (a2 / a1 <= s->tau) {
        alpha = m; s->tau *= 0.9; *rule = 2;                          /* Eq.9 */
    } else {
        alpha = a1; s->tau *= 1.1; *rule = 1;
    }
    s->alpha_prev = alpha;
    if (a1out) *a1out = a1;
    if (a2out) *a2out = a2;
    return alpha;
}

/* ------------------------------------------------------------------------------------
 * Start point, PAPER.md:260-267 (readings A11, A14)
 * ------------------------------------------------------------------------------------ */
static int make_start(const oracle_problem *P, const oreal *const *g, const oreal *const *b,
                      const oreal *f0, int init, double init_sigma, oreal *f)
{
    size_t n = P->n;
    switch (init) {
    case ORACLE_INIT_USER:
        if (!f0) return ORACLE_ERR_ARG;
        for (size_t i = 0; i < n; ++i) {
            if (!(f0[i] >= 0)) return ORACLE_ERR_DATA;
            f[i] = P->MR[i] ? f0[i] : (oreal)0;
        }
        break;
    case ORACLE_INIT_CONST:
    case ORACLE_INIT_CONST_SMOOTH: {
        /* c = max(0, (1/p) sum_j mean_S(g_j - b_j)), placed on R */
        double s = 0.0;
        for (int j = 0; j < P->p; ++j)
            for (size_t i = 0; i < n; ++i)
                if (P->MS[i]) s += (double)g[j][i] - (double)b[j][i];
        double c = s / ((double)P->p * (double)P->nS);
        if (c < 0.0) c = 0.0;
        for (size_t i = 0; i < n; ++i) f[i] = P->MR[i] ? (oreal)c : (oreal)0;
        if (init == ORACLE_INIT_CONST_SMOOTH) {
            /* "the constant image will be convolved with a Gaussian to avoid the presence of sharp edges"
               (reading A28): f0 = M_R o max(0, G_sigma * (c M_R)), G_sigma the periodic Gaussian
               of standard deviation init_sigma pixels on the S-bar grid, unit sum, centred on pixel (0,0) */
            if (!(init_sigma > 0.0)) return ORACLE_ERR_ARG;
            ocplx *G = (ocplx *)malloc(sizeof(ocplx) * n), *t = (ocplx *)malloc(sizeof(ocplx) * n);
            if (!G || !t) { free(G); free(t); return ORACLE_ERR_ALLOC; }
            double sum = 0.0;
            for (int y = 0; y < P->ny; ++y)
                for (int x = 0; x < P->nx; ++x) {
                    double dy = y <= P->ny / 2 ? y : y - P->ny, dx = x <= P->nx / 2 ? x : x - P->nx;
                    sum += exp(-(dy * dy + dx * dx) / (2.0 * init_sigma * init_sigma));
                }
            for (int y = 0; y < P->ny; ++y)
                for (int x = 0; x < P->nx; ++x) {
                    double dy = y <= P->ny / 2 ? y : y - P->ny, dx = x <= P->nx / 2 ? x : x - P->nx;
                    G[(size_t)y * P->nx + x] = (oreal)(exp(-(dy * dy + dx * dx) / (2.0 * init_sigma * init_sigma)) / sum);
                }
            for (size_t i = 0; i < n; ++i) t[i] = f[i];
            int rc = fft2_inplace(P->ny, P->nx, -1, G);
            if (!rc) rc = fft2_inplace(P->ny, P->nx, -1, t);
            if (!rc) { for (size_t i = 0; i < n; ++i) t[i] *= G[i]; rc = fft2_inplace(P->ny, P->nx, +1, t); }
            if (!rc) for (size_t i = 0; i < n; ++i) { oreal v = (oreal)creal(t[i]); f[i] = (P->MR[i] && v > 0) ? v : (oreal)0; }
            free(G); free(t);
            if (rc) return rc;
        }
        break; }
    case ORACLE_INIT_ZERO:
        for (size_t i = 0; i < n; ++i) f[i] = 0;
        break;
    case ORACLE_INIT_G:
        for (size_t i = 0; i < n; ++i) f[i] = (P->MR[i] && P->MS[i] && g[0][i] > 0) ? g[0][i] : (oreal)0;
        break;
    default:
        return ORACLE_ERR_ARG;
    }
    return ORACLE_OK;
}

static int check_options(const oracle_options *o)
{
    if (o && !(o->rl_relax > 0.0)) return ORACLE_ERR_ARG;
    if (o && !(o->rl_linear > 0.0)) return ORACLE_ERR_ARG;
    if (o && o->rl_relax != 1.0 && o->rl_linear != 1.0) return ORACLE_ERR_ARG;      /* Eq.3 and Eq.4 are alternatives */
    if (!o) return ORACLE_ERR_ARG;
    if (!(o->beta > 0 && o->beta < 1 && o->theta > 0 && o->theta < 1)) return ORACLE_ERR_ARG;
    if (!(o->alpha_min > 0 && o->alpha_min < o->alpha_max)) return ORACLE_ERR_ARG;
    if (o->m_alpha < 1 || o->m_alpha > 16 || o->armijo_memory < 1 || o->max_iter < 0) return ORACLE_ERR_ARG;
    if (!o->adaptive_L && !(o->L1 > 0 && o->L1 < o->L2)) return ORACLE_ERR_ARG;
    if (o->max_backtracks < 0) return ORACLE_ERR_ARG;
    if (o->stop_rule < ORACLE_STOP_MAXIT || o->stop_rule > ORACLE_STOP_MINERR) return ORACLE_ERR_ARG;
    if (o->init == ORACLE_INIT_CONST_SMOOTH && !(o->init_sigma > 0.0)) return ORACLE_ERR_ARG;
    return ORACLE_OK;
}

/* copies g with negative values clamped to 0 (A17), or fails in strict mode */
static int clean_data(const oracle_problem *P, const oreal *const *g, int strict, oreal **gc)
{
    for (int j = 0; j < P->p; ++j)
        for (size_t i = 0; i < P->n; ++i) {
            oreal v = P->MS[i] ? g[j][i] : (oreal)0;
            if (!isfinite((double)v)) return ORACLE_ERR_DATA;
            if (v < 0) { if (strict) return ORACLE_ERR_DATA; v = 0; }
            gc[j][i] = v;
        }
    return ORACLE_OK;
}

static int stop_test(const oracle_options *o, const oracle_problem *P, int k_done, double Jnew,
                     double Jold, int have_old)
{
    /* Eq.24 */
    if (o->stop_rule == ORACLE_STOP_RELJ && have_old && fabs(Jnew - Jold) <= o->tol * Jold)
        return ORACLE_REASON_RELJ;
    /* Eq.26 in reading A6/A7: 2 J0 / (p #S) <= b */
    if (o->stop_rule == ORACLE_STOP_DISCREPANCY &&
        2.0 * Jnew / ((double)P->p * (double)P->nS) <= o->disc_threshold)
        return ORACLE_REASON_DISCREPANCY;
    if (k_done >= o->max_iter) return ORACLE_REASON_MAXIT;
    return 0;
}

/* ------------------------------------------------------------------------------------
 * SGP, Algorithm 1 with the step-length rules of PAPER.md:130-155 and the
 * scaling of Eq.10/23.  Follows SURVEY.md 8(c) "Iteration k" step by step.
 * ------------------------------------------------------------------------------------ */
int oracle_sgp_run(const oracle_problem *P, const oreal *const *g_in, const oreal *const *b,
                   const oreal *f0, const oracle_options *o, oracle_result *res, oreal *f_out)
{
    if (!P || !g_in || !b || !res || !f_out) return ORACLE_ERR_ARG;
    int rc = check_options(o);
    if (rc) return rc;
    const int p = P->p;
    const size_t n = P->n;
    oreal **g = alloc_planes(p, n), **q = alloc_planes(p, n), **u = alloc_planes(p, n), **r = alloc_planes(p, n);
    oreal *f = (oreal *)calloc(n, sizeof(oreal)), *fprev = (oreal *)calloc(n, sizeof(oreal));
    oreal *grad = (oreal *)calloc(n, sizeof(oreal)), *gprev = (oreal *)calloc(n, sizeof(oreal));
    oreal *D = (oreal *)calloc(n, sizeof(oreal)), *y = (oreal *)calloc(n, sizeof(oreal)), *d = (oreal *)calloc(n, sizeof(oreal));
    double *Jhist = (double *)calloc((size_t)o->armijo_memory, sizeof(double));
    if (!g || !q || !u || !r || !f || !fprev || !grad || !gprev || !D || !y || !d || !Jhist) { rc = ORACLE_ERR_ALLOC; goto done; }

    rc = clean_data(P, g_in, o->strict, g);                     if (rc) goto done;
    rc = make_start(P, (const oreal *const *)g, b, f0, o->init, o->init_sigma, f);   if (rc) goto done;
    /* flux constraint (reading A26): c = the background-subtracted flux of the data, averaged over the images */
    double flux_c = o->flux_value;
    if (o->flux_constraint && !(flux_c > 0.0)) {
        double sfl = 0.0;
        for (int j = 0; j < p; ++j)
            for (size_t i = 0; i < n; ++i)
                if (P->MS[i]) sfl += (double)g[j][i] - (double)b[j][i];
        flux_c = sfl / (double)p;
        if (flux_c < 0.0) flux_c = 0.0;
    }
    if (o->flux_constraint) {
        /* SGP needs a feasible f(0) (Bonettini et al. 2009: f(0) in Omega; d = P(f - alpha D grad) - f is a descent
           direction only from a feasible f): the start point is rescaled to the flux c, the null image becomes the
           constant c / #R on R (reading A26) */
        double s0 = 0.0;
        for (size_t i = 0; i < n; ++i) s0 += (double)f[i];
        if (!(flux_c > 0.0)) { rc = ORACLE_ERR_DATA; goto done; }
        for (size_t i = 0; i < n; ++i)
            f[i] = s0 > 0.0 ? (oreal)((double)f[i] * (flux_c / s0)) : (P->MR[i] ? (oreal)(flux_c / (double)P->nR) : (oreal)0);
    }
    rc = oracle_all_A(P, f, q);                                 if (rc) goto done;   /* q_j = A_j f(0) */
    double J = oracle_J0(P, (const oreal *const *)q, (const oreal *const *)g, b);
    if (!isfinite(J)) { rc = ORACLE_ERR_NONFINITE; goto done; }

    /* Eq.25 (reading A27): rho(k) = ||f(k) - f~|| / ||f~||; with ORACLE_STOP_MINERR the run stops at the first k whose
       step would increase rho ("reaches a minimum value"), that step is discarded and f(k) returned */
    const oreal *truth = (const oreal *)res->truth;
    if (o->stop_rule == ORACLE_STOP_MINERR && !truth) { rc = ORACLE_ERR_ARG; goto done; }
    double rho = truth ? oracle_rel_error((long)n, f, truth) : 0.0;
    if (truth && res->trace_err) res->trace_err[0] = rho;

    double L1 = o->L1, L2 = o->L2;
    if (o->adaptive_L) {
        rc = rl_update_from_q(P, f, q, (const oreal *const *)g, b, r, d, y);
        if (rc) goto done;
        rc = oracle_adaptive_bounds((long)n, y, &L1, &L2);
        if (rc) goto done;
    }
    res->L1_used = L1; res->L2_used = L2;

    oracle_bb_state bb;
    oracle_bb_init(&bb, o);
    int nJ = 0;                     /* number of accepted J values stored in the Armijo ring */
    Jhist[0] = J; nJ = 1;
    if (res->trace_J) res->trace_J[0] = J;
    res->total_backtracks = 0;
    res->iterations = 0;
    res->stop_reason = 0;
    long fft0 = g_fft2_count;

    int k = 0;
    if (o->max_iter == 0) res->stop_reason = ORACLE_REASON_MAXIT;
    while (!res->stop_reason) {
        /* step 1 of 8(c): r_j, w, grad */
        rc = gradient_from_q(P, q, (const oreal *const *)g, b, r, grad);
        if (rc) goto done;
        /* step 2: scaling D_k, Eq.10/23 */
        oracle_scaling(P, f, L1, L2, D);
        /* step 3: alpha_k */
        double alpha; int rule = 0;
        if (k == 0) {
            alpha = o->alpha0;
        } else {
            double a = 0, c = 0, e = 0, h = 0;
            for (size_t i = 0; i < n; ++i) {
                if (!P->MR[i]) continue;                         /* sums over R (A11) */
                double s = (double)f[i] - (double)fprev[i];      /* s(k-1) */
                double z = (double)grad[i] - (double)gprev[i];   /* z(k-1), PAPER.md:95 (A1) */
                double Di = (double)D[i];
                a += s * s / (Di * Di);                          /* s' D^-1 D^-1 s   (Eq.7) */
                c += s * z / Di;                                 /* s' D^-1 z        (Eq.7) */
                e += s * z * Di;                                 /* s' D z           (Eq.8) */
                h += z * z * Di * Di;                            /* z' D D z         (Eq.8) */
            }
            alpha = oracle_bb_next(&bb, o, k, a, c, e, h, &rule, NULL, NULL);
        }
        if (res->force_alpha && isfinite(res->force_alpha[k])) { alpha = res->force_alpha[k]; bb.alpha_prev = alpha; }
        /* step 4: y = P+(f - alpha D grad); d = y - f; gd = grad' d   (Alg.1 steps 2-3) */
        if (o->flux_constraint) {
            /* projection on { y >= 0, sum y = c } in the metric D^-1 (Bonettini et al. 2009) */
            for (size_t i = 0; i < n; ++i) y[i] = f[i] - (oreal)alpha * D[i] * grad[i];
            rc = oracle_project_flux((long)n, y, D, flux_c, y, NULL);
            if (rc) goto done;
        } else
        oracle_project((long)n, f, grad, D, alpha, y);
        double gd = 0.0;
        for (size_t i = 0; i < n; ++i) {
            d[i] = P->MR[i] ? y[i] - f[i] : (oreal)0;
            gd += (double)grad[i] * (double)d[i];
        }
        /* step 5: u_j = A_j d */
        rc = oracle_all_A(P, d, u);
        if (rc) goto done;
        /* step 6: Armijo backtracking on q_j + lambda u_j (Alg.1 steps 4-5), reference value =
           max of the last min(k+1, M) accepted J (M = 1: monotone, the paper; A15) */
        double Jref = Jhist[0];
        for (int i = 1; i < nJ; ++i) Jref = fmax(Jref, Jhist[i]);
        double lambda = 1.0, Jnew = 0.0;
        int nb = 0;
        if (res->force_lambda && isfinite(res->force_lambda[k])) {
            lambda = res->force_lambda[k];
            Jnew = 0.0;
            for (int j = 0; j < p; ++j)
                for (size_t i = 0; i < n; ++i)
                    if (P->MS[i])
                        Jnew += kl_term((double)g[j][i], (double)(oreal)(q[j][i] + (oreal)lambda * u[j][i]) + (double)b[j][i]);
        } else {
            for (;;) {
                Jnew = 0.0;
                for (int j = 0; j < p; ++j)
                    for (size_t i = 0; i < n; ++i)
                        if (P->MS[i])
                            Jnew += kl_term((double)g[j][i], (double)(oreal)(q[j][i] + (oreal)lambda * u[j][i]) + (double)b[j][i]);
                if (isfinite(Jnew) && Jnew <= Jref + o->beta * lambda * gd) break;
                if (nb >= o->max_backtracks) { rc = ORACLE_ERR_LINESEARCH; goto done; }
                lambda *= o->theta;
                nb++;
            }
        }
        /* Eq.25: error of the candidate f(k) + lambda d; an increase stops the run BEFORE the step is taken (A27) */
        double rho_new = 0.0;
        if (truth) {
            for (size_t i = 0; i < n; ++i) y[i] = f[i] + (oreal)lambda * d[i];
            rho_new = oracle_rel_error((long)n, y, truth);
            if (res->trace_err) res->trace_err[k + 1] = rho_new;
            if (o->stop_rule == ORACLE_STOP_MINERR && rho_new > rho) { res->stop_reason = ORACLE_REASON_MINERR; break; }
            rho = rho_new;
        }
        /* step 7: f(k+1) = f(k) + lambda d (Alg.1 step 6); q_j <- q_j + lambda u_j (A21) */
        for (size_t i = 0; i < n; ++i) {
            fprev[i] = f[i]; gprev[i] = grad[i];
            f[i] = f[i] + (oreal)lambda * d[i];
        }
        for (int j = 0; j < p; ++j)
            for (size_t i = 0; i < n; ++i) q[j][i] = q[j][i] + (oreal)lambda * u[j][i];
        if (o->refresh_every > 0 && (k + 1) % o->refresh_every == 0) {
            rc = oracle_all_A(P, f, q);
            if (rc) goto done;
            Jnew = oracle_J0(P, (const oreal *const *)q, (const oreal *const *)g, b);
        }
        if (res->trace_alpha) res->trace_alpha[k] = alpha;
        if (res->trace_lambda) res->trace_lambda[k] = lambda;
        if (res->trace_rule) res->trace_rule[k] = rule;
        if (res->trace_backtracks) res->trace_backtracks[k] = nb;
        if (res->trace_J) res->trace_J[k + 1] = Jnew;
        res->total_backtracks += nb;
        double Jold = J;
        J = Jnew;
        Jhist[(k + 1) % o->armijo_memory] = J;
        if (nJ < o->armijo_memory) nJ++;
        k++;
        res->iterations = k;
        /* step 8: stopping rules */
        res->stop_reason = stop_test(o, P, k, J, Jold, 1);
    }
    res->n_fft2 = g_fft2_count - fft0;
    res->J0_final = J;
    res->discrepancy_final = 2.0 * J / ((double)p * (double)P->nS);
    res->err_final = rho;
    rc = ORACLE_OK;
done:
    if (f) memcpy(f_out, f, sizeof(oreal) * n);     /* on error: the last accepted iterate */
    free_planes(g, p); free_planes(q, p); free_planes(u, p); free_planes(r, p);
    free(f); free(fprev); free(grad); free(gprev); free(D); free(y); free(d); free(Jhist);
    return rc;
}

/* ------------------------------------------------------------------------------------
 * Richardson-Lucy, Eq.1 / Eq.13 / Eq.21; A_j f recomputed from f every iteration.
 * J0(f(k)) is evaluated from the same A_j f(k), so the stopping rules see J at every k.
 * ------------------------------------------------------------------------------------ */
int oracle_rl_run(const oracle_problem *P, const oreal *const *g_in, const oreal *const *b,
                  const oreal *f0, const oracle_options *o, oracle_result *res, oreal *f_out)
{
    if (!P || !g_in || !b || !res || !f_out) return ORACLE_ERR_ARG;
    int rc = check_options(o);
    if (rc) return rc;
    const int p = P->p;
    const size_t n = P->n;
    oreal **g = alloc_planes(p, n), **q = alloc_planes(p, n), **r = alloc_planes(p, n);
    oreal *f = (oreal *)calloc(n, sizeof(oreal)), *w = (oreal *)calloc(n, sizeof(oreal)), *fn = NULL;
    if (!g || !q || !r || !f || !w) { rc = ORACLE_ERR_ALLOC; goto done; }
    rc = clean_data(P, g_in, o->strict, g);                           if (rc) goto done;
    rc = make_start(P, (const oreal *const *)g, b, f0, o->init, o->init_sigma, f);   if (rc) goto done;
    res->iterations = 0; res->stop_reason = 0; res->total_backtracks = 0;
    res->L1_used = 0; res->L2_used = 0;
    long fft0 = g_fft2_count;
    double J = 0.0, Jold = 0.0;
    /* Eq.25 (reading A27), as in oracle_sgp_run: an update that would increase rho is not taken */
    const oreal *truth = (const oreal *)res->truth;
    if (o->stop_rule == ORACLE_STOP_MINERR && !truth) { rc = ORACLE_ERR_ARG; goto done; }
    double rho = truth ? oracle_rel_error((long)n, f, truth) : 0.0;
    if (truth && res->trace_err) res->trace_err[0] = rho;
    fn = (oreal *)calloc(n, sizeof(oreal));
    if (!fn) { rc = ORACLE_ERR_ALLOC; goto done; }
    for (int k = 0;; ++k) {
        rc = oracle_all_A(P, f, q);                                   if (rc) goto done;
        Jold = J;
        J = oracle_J0(P, (const oreal *const *)q, (const oreal *const *)g, b);
        if (!isfinite(J)) { rc = ORACLE_ERR_NONFINITE; goto done; }
        if (res->trace_J) res->trace_J[k] = J;
        res->iterations = k;
        res->stop_reason = stop_test(o, P, k, J, Jold, k > 0);
        if (res->stop_reason) break;
        if (o->rl_linear != 1.0) {
            /* linear relaxation, Eq.4 (Adorf et al.): f(k+1) = f(k) - lambda_k f(k) o (1 - A^T g/(Af+b)), here with a
               constant lambda_k = rl_linear; for p images / boundary correction the subtracted array is f o (1 - W o sum_j
               A_j^T(...)), i.e. f minus the RL step of Eq.13 / Eq.21, and the result is projected on f >= 0 (reading A25). */
            for (int j = 0; j < p; ++j)
                for (size_t i2 = 0; i2 < n; ++i2)
                    r[j][i2] = P->MS[i2] ? ratio_term(g[j][i2], q[j][i2] + b[j][i2]) : (oreal)0;
            rc = oracle_sum_AT(P, (const oreal *const *)r, w);
            if (rc) goto done;
            for (size_t i2 = 0; i2 < n; ++i2)
            {
                oreal y = f[i2] - (oreal)o->rl_linear * (f[i2] * ((oreal)1 - P->W[i2] * w[i2]));
                fn[i2] = y > (oreal)0 ? y : (oreal)0;      /* the non-negativity constraint of the paper, reading A25 */
            }
        } else if (o->rl_relax == 1.0) {
            rc = rl_update_from_q(P, f, q, (const oreal *const *)g, b, r, w, fn);
            if (rc) goto done;
        } else {
            /* multiplicative relaxation, Eq.3 (Llacer & Nunez): f(k+1) = f(k) o (A^T g/(Af+b))^alpha;
               for p images / boundary correction the bracket is the RL factor W o sum_j A_j^T(...) of Eq.13 / Eq.21 (reading A24) */
            for (int j = 0; j < p; ++j)
                for (size_t i2 = 0; i2 < n; ++i2)
                    r[j][i2] = P->MS[i2] ? ratio_term(g[j][i2], q[j][i2] + b[j][i2]) : (oreal)0;
            rc = oracle_sum_AT(P, (const oreal *const *)r, w);
            if (rc) goto done;
            for (size_t i2 = 0; i2 < n; ++i2) fn[i2] = f[i2] * (oreal)pow(fmax(0.0, (double)(P->W[i2] * w[i2])), o->rl_relax);   /* base >= 0 up to FFT round-off */
        }
        if (truth) {
            double rho_new = oracle_rel_error((long)n, fn, truth);
            if (res->trace_err) res->trace_err[k + 1] = rho_new;
            if (o->stop_rule == ORACLE_STOP_MINERR && rho_new > rho) { res->stop_reason = ORACLE_REASON_MINERR; break; }
            rho = rho_new;
        }
        memcpy(f, fn, sizeof(oreal) * n);
    }
    res->n_fft2 = g_fft2_count - fft0;
    res->J0_final = J;
    res->discrepancy_final = 2.0 * J / ((double)p * (double)P->nS);
    res->err_final = rho;
    rc = ORACLE_OK;
done:
    if (f) memcpy(f_out, f, sizeof(oreal) * n);
    free_planes(g, p); free_planes(q, p); free_planes(r, p); free(f); free(w); free(fn);
    return rc;
}

/* ------------------------------------------------------------------------------------
 * OSEM, Algorithm 2: h(0) = f(k); for j = 1..p
 *   h(j) = h(j-1) o A_j^T( g_j / (A_j h(j-1) + b_j) )                         Eq.15
 * and with boundary-effect correction
 *   h(j) = (M_R / alpha_j) o h(j-1) o A_j^T( g_j / (A_j h(j-1) + b_j) )       Eq.22
 * f(k+1) = h(p).  alpha_j = A_j^T 1_S (Eq.19 in reading A5; == 1 analytically when unmasked,
 * the PSFs having unit volume).  4p transforms per iteration.  The paper stops
 * OSEM by the reconstruction error only (needs the true object: out of scope), so the run is
 * max_iter cycles; J0(f) of Eq.12 is evaluated once, at the final iterate.
 * ------------------------------------------------------------------------------------ */
int oracle_osem_run(const oracle_problem *P, const oreal *const *g_in, const oreal *const *b,
                    const oreal *f0, const oracle_options *o, oracle_result *res, oreal *f_out)
{
    if (!P || !g_in || !b || !res || !f_out) return ORACLE_ERR_ARG;
    int rc = check_options(o);
    if (rc) return rc;
    const int p = P->p;
    const size_t n = P->n;
    oreal **g = alloc_planes(p, n), **q = alloc_planes(p, n), **aj = alloc_planes(p, n);
    oreal *h = (oreal *)calloc(n, sizeof(oreal)), *w = (oreal *)calloc(n, sizeof(oreal));
    oreal *r = (oreal *)calloc(n, sizeof(oreal)), *hk = NULL;
    if (!g || !q || !aj || !h || !w || !r) { rc = ORACLE_ERR_ALLOC; goto done; }
    rc = clean_data(P, g_in, o->strict, g);                           if (rc) goto done;
    rc = make_start(P, (const oreal *const *)g, b, f0, o->init, o->init_sigma, h);   if (rc) goto done;
    for (int j = 0; j < p; ++j) {                                     /* alpha_j on R, 0 elsewhere */
        if (P->masked) {
            for (size_t i = 0; i < n; ++i) r[i] = P->MS[i] ? (oreal)1 : (oreal)0;
            rc = oracle_apply_AT(P, j, r, aj[j]);                     if (rc) goto done;
        } else {
            for (size_t i = 0; i < n; ++i) aj[j][i] = (oreal)1;
        }
    }
    res->iterations = 0; res->stop_reason = 0; res->total_backtracks = 0;
    res->L1_used = 0; res->L2_used = 0;
    long fft0 = g_fft2_count;
    /* Eq.25 (reading A27), per cycle: the paper stops OSEM (and RL, SGP) at the minimum r.m.s. error in its diffuse-object experiments */
    const oreal *truth = (const oreal *)res->truth;
    if (o->stop_rule == ORACLE_STOP_MINERR && !truth) { rc = ORACLE_ERR_ARG; goto done; }
    double rho = truth ? oracle_rel_error((long)n, h, truth) : 0.0;
    if (truth && res->trace_err) res->trace_err[0] = rho;
    hk = (oreal *)calloc(n, sizeof(oreal));
    if (!hk) { rc = ORACLE_ERR_ALLOC; goto done; }
    for (int k = 0; k < o->max_iter; ++k) {
        memcpy(hk, h, sizeof(oreal) * n);                             /* f(k), restored if the cycle is discarded */
        for (int j = 0; j < p; ++j) {
            rc = oracle_apply_A(P, j, h, q[j]);                       if (rc) goto done;
            for (size_t i = 0; i < n; ++i) r[i] = P->MS[i] ? ratio_term(g[j][i], q[j][i] + b[j][i]) : (oreal)0;
            rc = oracle_apply_AT(P, j, r, w);                         if (rc) goto done;
            for (size_t i = 0; i < n; ++i) h[i] = P->MR[i] ? h[i] * w[i] / aj[j][i] : (oreal)0;
        }
        if (truth) {
            double rho_new = oracle_rel_error((long)n, h, truth);
            if (res->trace_err) res->trace_err[k + 1] = rho_new;
            if (o->stop_rule == ORACLE_STOP_MINERR && rho_new > rho) {
                memcpy(h, hk, sizeof(oreal) * n);
                res->stop_reason = ORACLE_REASON_MINERR;
                break;
            }
            rho = rho_new;
        }
        res->iterations = k + 1;
    }
    res->n_fft2 = g_fft2_count - fft0;
    if (!res->stop_reason) res->stop_reason = ORACLE_REASON_MAXIT;
    res->err_final = rho;
    rc = oracle_all_A(P, h, q);                                       if (rc) goto done;
    {
        double J = oracle_J0(P, (const oreal *const *)q, (const oreal *const *)g, b);
        res->J0_final = J;
        res->discrepancy_final = 2.0 * J / ((double)p * (double)P->nS);
        rc = isfinite(J) ? ORACLE_OK : ORACLE_ERR_NONFINITE;
    }
done:
    if (h) memcpy(f_out, h, sizeof(oreal) * n);
    free_planes(g, p); free_planes(q, p); free_planes(aj, p); free(h); free(w); free(r); free(hk);
    return rc;
}

/* ------------------------------------------------------------------------------------
 * Paper-level entry points: marshal (g, K, b, f0) onto the S-bar grid and run.
 * ------------------------------------------------------------------------------------ */
typedef int (*run_fn)(const oracle_problem *, const oreal *const *, const oreal *const *,
                      const oreal *, const oracle_options *, oracle_result *, oreal *);

static int run_generic(run_fn run, int p, const oreal *const *g, const oreal *const *psf,
                       const oreal *const *b_arr, const double *b_const, int masked, int oy, int ox,
                       int sy, int sx, int ny, int nx, const oreal *f0, oreal *f_out,
                       unsigned char *maskR_out, int dtype, const oracle_options *o,
                       oracle_result *res)
{
    if (dtype != ORACLE_DTYPE || !g || !psf || !o || !res || !f_out || p < 1) return ORACLE_ERR_ARG;
    if (!b_arr && !b_const) return ORACLE_ERR_ARG;
    int rc;
    oracle_problem *P = oracle_problem_create(p, ny, nx, psf, masked, oy, ox, sy, sx, o->sigma_R,
                                              o->psf_origin, &rc);
    if (!P) return rc;
    size_t n = P->n;
    oreal **G = alloc_planes(p, n), **B = alloc_planes(p, n);
    if (!G || !B) { rc = ORACLE_ERR_ALLOC; goto done; }
    for (int j = 0; j < p; ++j) {
        if (!g[j]) { rc = ORACLE_ERR_ARG; goto done; }
        for (int y = 0; y < P->sy; ++y)
            for (int x = 0; x < P->sx; ++x) {
                size_t i = (size_t)(y + P->oy) * nx + (x + P->ox), s = (size_t)y * P->sx + x;
                G[j][i] = g[j][s];
                B[j][i] = (b_arr && b_arr[j]) ? b_arr[j][s] : (oreal)b_const[j];
            }
    }
    rc = run(P, (const oreal *const *)G, (const oreal *const *)B, f0, o, res, f_out);
    if (maskR_out) memcpy(maskR_out, P->MR, n);
done:
    free_planes(G, p); free_planes(B, p);
    oracle_problem_destroy(P);
    return rc;
}

int oracle_sgp_single(const oreal *g, const oreal *psf, const oreal *b_arr, double b_const,
                      const oreal *f0, oreal *f_out, int ny, int nx, int dtype,
                      const oracle_options *o, oracle_result *res)
{
    const oreal *gg[1] = { g }, *pp[1] = { psf }, *bb[1] = { b_arr };
    return run_generic(oracle_sgp_run, 1, gg, pp, b_arr ? bb : NULL, &b_const, 0, 0, 0, ny, nx, ny, nx,
                       f0, f_out, NULL, dtype, o, res);
}
int oracle_sgp_multi(int p, const oreal *const *g, const oreal *const *psf,
                     const oreal *const *b_arr, const double *b_const, const oreal *f0,
                     oreal *f_out, int ny, int nx, int dtype, const oracle_options *o,
                     oracle_result *res)
{
    return run_generic(oracle_sgp_run, p, g, psf, b_arr, b_const, 0, 0, 0, ny, nx, ny, nx, f0, f_out,
                       NULL, dtype, o, res);
}
int oracle_sgp_boundary(int p, const oreal *const *g, const oreal *const *psf,
                        const oreal *const *b_arr, const double *b_const, int oy, int ox, int sy,
                        int sx, int ny, int nx, const oreal *f0, oreal *f_out,
                        unsigned char *maskR_out, int dtype, const oracle_options *o,
                        oracle_result *res)
{
    return run_generic(oracle_sgp_run, p, g, psf, b_arr, b_const, 1, oy, ox, sy, sx, ny, nx, f0, f_out,
                       maskR_out, dtype, o, res);
}
int oracle_rl_single(const oreal *g, const oreal *psf, const oreal *b_arr, double b_const,
                     const oreal *f0, oreal *f_out, int ny, int nx, int dtype,
                     const oracle_options *o, oracle_result *res)
{
    const oreal *gg[1] = { g }, *pp[1] = { psf }, *bb[1] = { b_arr };
    return run_generic(oracle_rl_run, 1, gg, pp, b_arr ? bb : NULL, &b_const, 0, 0, 0, ny, nx, ny, nx,
                       f0, f_out, NULL, dtype, o, res);
}
int oracle_rl_multi(int p, const oreal *const *g, const oreal *const *psf,
                    const oreal *const *b_arr, const double *b_const, const oreal *f0,
                    oreal *f_out, int ny, int nx, int dtype, const oracle_options *o,
                    oracle_result *res)
{
    return run_generic(oracle_rl_run, p, g, psf, b_arr, b_const, 0, 0, 0, ny, nx, ny, nx, f0, f_out,
                       NULL, dtype, o, res);
}
int oracle_rl_boundary(int p, const oreal *const *g, const oreal *const *psf,
                       const oreal *const *b_arr, const double *b_const, int oy, int ox, int sy,
                       int sx, int ny, int nx, const oreal *f0, oreal *f_out,
                       unsigned char *maskR_out, int dtype, const oracle_options *o,
                       oracle_result *res)
{
    return run_generic(oracle_rl_run, p, g, psf, b_arr, b_const, 1, oy, ox, sy, sx, ny, nx, f0, f_out,
                       maskR_out, dtype, o, res);
}
int oracle_osem_multi(int p, const oreal *const *g, const oreal *const *psf,
                      const oreal *const *b_arr, const double *b_const, const oreal *f0,
                      oreal *f_out, int ny, int nx, int dtype, const oracle_options *o,
                      oracle_result *res)
{
    return run_generic(oracle_osem_run, p, g, psf, b_arr, b_const, 0, 0, 0, ny, nx, ny, nx, f0, f_out,
                       NULL, dtype, o, res);
}
int oracle_osem_boundary(int p, const oreal *const *g, const oreal *const *psf,
                         const oreal *const *b_arr, const double *b_const, int oy, int ox, int sy,
                         int sx, int ny, int nx, const oreal *f0, oreal *f_out,
                         unsigned char *maskR_out, int dtype, const oracle_options *o,
                         oracle_result *res)
{
    return run_generic(oracle_osem_run, p, g, psf, b_arr, b_const, 1, oy, ox, sy, sx, ny, nx, f0, f_out,
                       maskR_out, dtype, o, res);
}
