// sgp_dev.cuh -- device-resident control block, per-launch parameter structs and the scalar logic
// (step length, Armijo test, stopping rules) that runs on the device so that the iteration loop
// never synchronises with the host (keep everything on the GPU).
#pragma once
#include <cuda_runtime.h>
#include <math.h>
#include "../../include/sgp.h"

namespace sgpk {

constexpr int kMaxP = SGP_MAX_IMAGES;
constexpr int kNQ = 4;            // partial sums per block (max over the kernels)

// run-time options as the kernels see them
struct DevOpts {
    double beta, theta, alpha0, alpha_min, alpha_max, tol, disc_threshold;
    int m_alpha, alt_start, armijo_memory, max_iter, stop_rule, max_backtracks, adaptive_L, p;
    int flux_constraint;       // 1: projection on { f >= 0, sum f = c } (extra.cuh)
    int refresh_every;         // A21: recompute A f from f after every n-th iteration (0 = never)
    double nS_total;   // p * #S, the denominator of Eq.26
    double rl_relax;   // RL: exponent of the multiplicative relaxation, Eq.3; 1 = plain RL
    double rl_linear;  // RL: constant lambda_k of the linear relaxation, Eq.4; 1 = plain RL
};

// one per plan, in device memory; written only by single threads of "last block" epilogues
struct Ctrl {
    int k;                 // completed iterations
    int status;            // 0 = running, > 0 = sgp_reason, < 0 = sgp_status error
    int accepted;          // Armijo test outcome for lambda = 1 of the current iteration
    int rule;              // rule that produced alpha of the current iteration
    int total_backtracks;
    int ring_len, ring_pos, nJ;
    int flag_data;         // set by the input-cleaning kernels: 1 = non-finite g, 2 = negative g (strict), 4 = negative f0
    int pending;           // 1: the accepted step (lambda, d) has not been added to f yet (lazy update, a10)
    int qsel;              // which of the two q buffers holds A_j f(k): toggled by every finished iteration
    int need_k1;           // what the ratio kernel K1 has to do: 0 = nothing (the line-search kernel already formed q(k+1), the
                           // ratio and its row FFT at lambda = 1), 1 = ratio of the current q, 2 = q <- q + lambda u first
    double alpha;          // alpha_k of the current iteration
    double lambda;         // accepted lambda of the last completed iteration (s(k-1) = lambda d)
    double alpha_prev, tau;
    double J;              // J0(f(k))
    double Jtrial;         // J0 at f + lambda d of the current trial
    double Jref;           // Armijo reference value of the current iteration
    double gd;             // grad' d of the current iteration
    double L1, L2;
    double c0;             // constant start value (A14)
    double psf_sum;
    double ring[SGP_MAX_MALPHA];
    double Jhist[SGP_MAX_ARMIJO_MEMORY];
    unsigned int counter[8];   // "last block done" tickets, one per kernel family
    unsigned long long nfft;   // 2-D transforms executed by the column kernels since the run started (n_fft2)
    double Jprev;              // J0(f(k-1)): restored when the Eq.25 rule discards the last step
    int nbt_last;              // backtracks of the last accepted step (same purpose)
    double err, err_trial;     // Eq.25: rho(k) of the current iterate / of the candidate f(k) + lambda d
    double flux_c, mu;         // flux constraint: c and the multiplier of the current projection
    int refresh_due;           // 1: the step just accepted is followed by a recomputation of A f (refresh_every)
    int need_k1_next;          // refresh round: what the second instance of the ratio kernel has to do
    int err_pending;           // Eq.25: the error of the step just accepted has not been evaluated yet
    int commit;                // RL with the Eq.25 rule: adopt the candidate update
    int flux_rounds;           // Newton steps of the last flux-constrained projection
    double flux_cnt;           // active pixels of the previous Newton step
    double tmp_sum;            // scratch of the set-up kernels
    double bconst[SGP_MAX_IMAGES];   // batched plans: the background constants of this problem
};

// optional per-iteration traces (device arrays of max_iter+1 entries) and forced steps (test-only)
struct Trace {
    double *J, *alpha, *lambda;
    int *rule, *backtracks;
    const double *force_alpha, *force_lambda;
    double *err;               // Eq.25: rho(k), max_iter + 2 entries (nullptr without a true object)
};

// geometry shared by all kernels of a plan
struct Geom {
    int ny, nx;            // object grid S-bar
    int oy, ox, sy, sx;    // S inside S-bar
    int masked;            // boundary-effect problem: alphaR plane present
    int p;
    int C;                 // spectrum tile width (columns), a power of two
    int lc;                // log2(C)
    int RB;                // rows per block in the row kernels
};

__device__ __forceinline__ bool in_S(const Geom &G, int y, int x)
{
    return (unsigned)(y - G.oy) < (unsigned)G.sy && (unsigned)(x - G.ox) < (unsigned)G.sx;
}

// ---- step length: PAPER.md:130-155 (Eq.7-9, safeguards, alternation), run by one thread ----------
// a = s'D^-2 s, c = s'D^-1 z, e = s'D z, h = z'D^2 z with s = f(k)-f(k-1), z = grad(k)-grad(k-1)
__device__ inline void bb_step(Ctrl *ct, const DevOpts &o, const Trace &tr, double a, double c, double e, double h)
{
    const int k = ct->k;
    double alpha;
    int rule;
    if (k == 0) {
        alpha = o.alpha0; rule = 0;
    } else {
        double a1, a2;
        // IF s'D^-1 z <= 0 THEN alpha1 = min{10 alpha_{k-1}, alpha_max} ELSE clamp(BB1)
        if (c <= 0.0) a1 = fmin(10.0 * ct->alpha_prev, o.alpha_max);
        else          a1 = fmin(o.alpha_max, fmax(o.alpha_min, a / c));
        // IF s'D z <= 0 THEN alpha2 = min{10 alpha_{k-1}, alpha_max} ELSE clamp(BB2)
        if (e <= 0.0) a2 = fmin(10.0 * ct->alpha_prev, o.alpha_max);
        else          a2 = fmin(o.alpha_max, fmax(o.alpha_min, e / h));
        ct->ring[ct->ring_pos] = a2;
        ct->ring_pos = (ct->ring_pos + 1) % o.m_alpha;
        if (ct->ring_len < o.m_alpha) ct->ring_len++;
        double m = ct->ring[0];
        for (int i = 1; i < ct->ring_len; ++i) m = fmin(m, ct->ring[i]);       // Eq.9 (A20)
        if (k <= o.alt_start)             { alpha = m;  rule = 2; }             // PAPER.md:155 (A9)
        else if (a2 / a1 <= ct->tau)      { alpha = m;  rule = 2; ct->tau *= 0.9; }
        else                              { alpha = a1; rule = 1; ct->tau *= 1.1; }
        ct->alpha_prev = alpha;
    }
    if (tr.force_alpha) {
        double fa = tr.force_alpha[k];
        if (isfinite(fa)) { alpha = fa; ct->alpha_prev = fa; }
    }
    ct->alpha = alpha;
    ct->rule = rule;
}

// Armijo reference: max of the stored J values (M = 1: J(k), the paper; A15)
__device__ inline double armijo_ref(const Ctrl *ct)
{
    double r = ct->Jhist[0];
    for (int i = 1; i < ct->nJ; ++i) r = fmax(r, ct->Jhist[i]);
    return r;
}

// stopping rules; returns sgp_reason or 0
__device__ inline int stop_test(const DevOpts &o, int k_done, double Jnew, double Jold, bool have_old)
{
    if (o.stop_rule == SGP_STOP_RELJ && have_old && fabs(Jnew - Jold) <= o.tol * Jold) return SGP_REASON_RELJ;   // Eq.24
    if (o.stop_rule == SGP_STOP_DISCREPANCY && 2.0 * Jnew / o.nS_total <= o.disc_threshold)                      // Eq.26 (A6, A7)
        return SGP_REASON_DISCREPANCY;
    if (k_done >= o.max_iter) return SGP_REASON_MAXIT;
    return 0;
}

// book-keeping after an accepted step f(k+1) = f(k) + lambda d (Alg.1 step 6), one thread
__device__ inline void finish_iteration(Ctrl *ct, const DevOpts &o, const Trace &tr, double lambda, double Jnew, int nbt, int need_k1)
{
    const int k = ct->k;
    if (tr.alpha) tr.alpha[k] = ct->alpha;
    if (tr.lambda) tr.lambda[k] = lambda;
    if (tr.rule) tr.rule[k] = ct->rule;
    if (tr.backtracks) tr.backtracks[k] = nbt;
    if (tr.J) tr.J[k + 1] = Jnew;
    ct->total_backtracks += nbt;
    ct->nbt_last = nbt;
    const double Jold = ct->J;
    ct->Jprev = Jold;
    ct->J = Jnew;
    ct->lambda = lambda;
    ct->pending = 1;
    ct->qsel ^= 1;
    ct->need_k1 = need_k1;
    ct->Jhist[(k + 1) % o.armijo_memory] = Jnew;
    if (ct->nJ < o.armijo_memory) ct->nJ++;
    ct->k = k + 1;
    ct->err_pending = 1;
    // A21: after every refresh_every-th iteration A_j f and J0 are recomputed from f; the stopping rules then see the
    // recomputed J0 (extra.cuh / row_inv.cuh QJ_REFRESH), so the test is left to that kernel
    if (o.refresh_every > 0 && (k + 1) % o.refresh_every == 0) { ct->refresh_due = 1; return; }
    int r = stop_test(o, k + 1, Jnew, Jold, true);
    if (r) ct->status = r;
}

// ---- block-level reductions (deterministic: fixed tree) ------------------------------------------
template <int NQ>
__device__ __forceinline__ void block_reduce_sum(double (&v)[NQ], double *red /* >= NQ*32 doubles */)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) v[q] += __shfl_down_sync(0xffffffffu, v[q], off);
        if (lane == 0) red[q * 32 + wid] = v[q];
    }
    __syncthreads();
    if (wid == 0) {
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
            double x = lane < nw ? red[q * 32 + lane] : 0.0;
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) x += __shfl_down_sync(0xffffffffu, x, off);
            v[q] = x;   // valid in thread 0
        }
    }
    __syncthreads();
}

// Writes this block's partial sums, and returns true in EVERY thread of the last block to arrive
// (threadfence-reduction pattern); that block then owns all partials.
template <int NQ>
__device__ __forceinline__ bool publish_partials(const double (&v)[NQ], double *part, int block_id,
                                                 unsigned int total_blocks, unsigned int *ticket)
{
    __shared__ int s_last;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int q = 0; q < NQ; ++q) part[(size_t)block_id * NQ + q] = v[q];
        __threadfence();
        unsigned int t = atomicAdd(ticket, 1u);
        s_last = (t == total_blocks - 1);
        if (s_last) *ticket = 0;    // re-armed for the next launch
    }
    __syncthreads();
    bool last = s_last != 0;
    if (last) __threadfence();
    return last;
}

// the last block sums all partials in a fixed order; result valid in thread 0
template <int NQ>
__device__ __forceinline__ void final_sum(double (&v)[NQ], const double *part, unsigned int total_blocks, double *red)
{
#pragma unroll
    for (int q = 0; q < NQ; ++q) v[q] = 0.0;
    for (unsigned int b = threadIdx.x; b < total_blocks; b += blockDim.x) {
#pragma unroll
        for (int q = 0; q < NQ; ++q) v[q] += __ldcg(&part[(size_t)b * NQ + q]);
    }
    block_reduce_sum<NQ>(v, red);
}

}  // namespace sgpk
