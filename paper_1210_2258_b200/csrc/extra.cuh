// extra.cuh -- kernels of the optional parts of the driver (reading A21):
//   flux_mu_kernel      the multiplier mu of the flux-constrained projection (Bonettini et al. 2009)
//   err_kernel          the relative reconstruction error of Eq.25 and its stopping rule
//   apply_pending_kernel / the refresh round of reading A21 (recompute A_j f from f every n iterations)
//   gauss_plane_kernel  the periodic Gaussian of the smoothed constant start
// None of them contains an FFT; none runs unless its option is on.
#pragma once
#include "aux.cuh"

namespace sgpk {

// ---------------------------------------------------------------- flux-constrained projection: the multiplier
// y = argmin { sum_i (y_i - x_i)^2 / D_i : y >= 0, sum_R y = c },  x = f - alpha_k D grad   =>   y_i = max(0, x_i - mu D_i),
// mu the root of h(mu) = sum_R max(0, x_i - mu D_i) = c.  h is convex, piecewise linear and decreasing, so Newton's
// method started left of the root -- from the line through ALL pixels, mu_0 = (sum_R x - c) / sum_R D, which lies below h
// -- increases monotonically and ends after finitely many steps: when the set of active pixels { x_i - mu D_i > 0 } no
// longer shrinks, the step is the exact root.  A step is one pass over f and grad (2 planes, no FFT):
// (sum x, sum D, count) over the active set.  The passes are the "rounds" of the ticket scheme of aux.cuh (chunks drawn
// from a counter; the CTA that finishes the last chunk of a round takes the step), one launch per iteration.
template <typename T> struct FluxParams {
    Geom G; Ctrl *ct;
    const T *f, *grad, *alphaR;
    double *part;                                // 3 * nchunks doubles
    unsigned int *sync;                          // kBtSyncWords words of its own
    unsigned int nchunks, chunk_batches;
    int max_rounds;
};

template <typename T>
__global__ void __launch_bounds__(256) flux_mu_kernel(const FluxParams<T> P)
{
    using V = typename vec4_of<T>::type;
    constexpr int VN = vec4_of<T>::N;
    __shared__ double red[3 * 32];
    __shared__ unsigned int s_ticket;
    __shared__ int s_state, s_last;
    Ctrl *ct = P.ct;
    if (ct->status != 0) return;
    const Geom &G = P.G;
    const int tid = threadIdx.x, nthr = blockDim.x;
    const size_t n = (size_t)G.ny * G.nx;
    const T alpha = (T)ct->alpha, L1 = (T)ct->L1, L2 = (T)ct->L2;
    const T Wc = (T)(1.0 / (double)G.p);
    const double c = ct->flux_c;
    __threadfence();
    for (;;) {
        if (tid == 0) s_ticket = atomicAdd(&P.sync[kBtNext], 1u);
        __syncthreads();
        const unsigned int ticket = s_ticket;
        const unsigned int round = ticket / P.nchunks, chunk = ticket - round * P.nchunks;
        if (tid == 0) {
            int st = 0;
            for (;;) {
                if (ld_volatile_u32(&P.sync[kBtFinal]) != 0u) { st = 1; break; }
                if (ld_volatile_u32(&P.sync[kBtDecided]) >= round) break;
                __nanosleep(300);
            }
            __threadfence();
            s_state = st;
        }
        __syncthreads();
        if (s_state != 0) return;
        const bool all = round == 0;                                  // round 0: every pixel of R is taken as active
        const T mu = all ? (T)0 : (T)__ldcg(&ct->mu);
        double acc[3] = {0.0, 0.0, 0.0};
        const int CHV = 256 * kBtVecPerThread * (int)P.chunk_batches;
        const size_t e_begin = (size_t)chunk * (size_t)CHV * VN;
        for (int v0 = tid; v0 < CHV; v0 += nthr * kBtVecPerThread) {
            V f4[kBtVecPerThread], g4[kBtVecPerThread], a4[kBtVecPerThread];
            bool ok[kBtVecPerThread];
#pragma unroll
            for (int v = 0; v < kBtVecPerThread; ++v) {
                const size_t e0 = e_begin + (size_t)(v0 + v * nthr) * VN;
                ok[v] = (v0 + v * nthr) < CHV && e0 < n;
                if (ok[v]) {
                    f4[v] = *reinterpret_cast<const V *>(P.f + e0); g4[v] = *reinterpret_cast<const V *>(P.grad + e0);
                    if (G.masked) a4[v] = *reinterpret_cast<const V *>(P.alphaR + e0);
                }
            }
#pragma unroll
            for (int v = 0; v < kBtVecPerThread; ++v) {
                if (!ok[v]) continue;
                const T *fa = reinterpret_cast<const T *>(&f4[v]), *ga = reinterpret_cast<const T *>(&g4[v]), *aa = reinterpret_cast<const T *>(&a4[v]);
#pragma unroll
                for (int k = 0; k < VN; ++k) {
                    T w = Wc; bool inR = true;
                    if (G.masked) { inR = aa[k] > (T)0; w = inR ? (T)1 / aa[k] : (T)0; }
                    if (!inR) continue;
                    const T D = w * clipT<T>(fa[k], L1, L2);
                    const T x = fa[k] - alpha * D * ga[k];            // the argument of P+ in Eq.6, as the projection kernel forms it
                    if (all || x - mu * D > (T)0) { acc[0] += (double)x; acc[1] += (double)D; acc[2] += 1.0; }
                }
            }
        }
        block_reduce_sum<3>(acc, red);
        if (tid == 0) {
            P.part[3 * chunk] = acc[0]; P.part[3 * chunk + 1] = acc[1]; P.part[3 * chunk + 2] = acc[2];
            __threadfence();
            s_last = (atomicAdd(&P.sync[kBtDone], 1u) == P.nchunks - 1) ? 1 : 0;
        }
        __syncthreads();
        if (s_last) {
            __threadfence();
            double tot[3] = {0.0, 0.0, 0.0};
            for (unsigned int ch = tid; ch < P.nchunks; ch += nthr) {
                tot[0] += __ldcg(&P.part[3 * ch]); tot[1] += __ldcg(&P.part[3 * ch + 1]); tot[2] += __ldcg(&P.part[3 * ch + 2]);
            }
            block_reduce_sum<3>(tot, red);
            if (tid == 0) {
                P.sync[kBtDone] = 0;
                const double cnt_prev = ct->flux_cnt;
                bool fin = false;
                if (tot[1] > 0.0) ct->mu = (tot[0] - c) / tot[1]; else fin = true;       // no active pixel: mu stays
                if (!all && tot[2] == cnt_prev) fin = true;                              // the active set did not shrink: exact root
                if ((int)round + 1 >= P.max_rounds) fin = true;
                ct->flux_cnt = tot[2];
                ct->flux_rounds = (int)round + 1;
                __threadfence();
                if (fin) *reinterpret_cast<volatile unsigned int *>(&P.sync[kBtFinal]) = 1u;
                else     *reinterpret_cast<volatile unsigned int *>(&P.sync[kBtDecided]) = round + 1u;
            }
            __syncthreads();
        }
    }
}

// re-arms the counters of flux_mu_kernel; one thread, enqueued before it
template <int DUMMY = 0> __global__ void flux_arm_kernel(unsigned int *sync, Ctrl *ct)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        sync[kBtNext] = 0; sync[kBtDone] = 0; sync[kBtDecided] = 0; sync[kBtFinal] = 0;
        ct->flux_cnt = -1.0;
    }
}

// f(0) rescaled to the flux c (reading A26): f <- f c / sum f; the null image becomes c / #R on R.  s0 = ct->tmp_sum.
template <typename T>
__global__ void flux_rescale_kernel(T *f, const T *alphaR, size_t n, Geom Gm, double nR, Ctrl *ct)
{
    const double s0 = ct->tmp_sum, c = ct->flux_c;
    if (!(c > 0.0)) { if (threadIdx.x == 0 && blockIdx.x == 0) ct->status = SGP_ERR_DATA; return; }
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const bool inR = Gm.masked ? (alphaR[i] > (T)0) : true;
        f[i] = s0 > 0.0 ? (T)((double)f[i] * (c / s0)) : (inR ? (T)(c / nR) : (T)0);
    }
}

// sum of a plane -> ct->tmp_sum (single CTA; set-up only)
template <typename T>
__global__ void plane_sum_tmp_kernel(const T *x, size_t n, Ctrl *ct)
{
    __shared__ double red[32];
    double acc[1] = {0.0};
    for (size_t i = threadIdx.x; i < n; i += blockDim.x) acc[0] += (double)x[i];
    block_reduce_sum<1>(acc, red);
    if (threadIdx.x == 0) ct->tmp_sum = acc[0];
}

// ---------------------------------------------------------------- Eq.25: relative reconstruction error and its stopping rule
// rho = || f + [pending] lambda d - f~ ||_2 / || f~ ||_2 over the whole grid.  mode 0: rho(0) of the start point.  mode 1
// (SGP loop, after the book-keeping of an accepted step, whose f + lambda d is still pending, a10): rho(k+1) of the
// candidate; with SGP_STOP_MINERR an increase discards the step (pending <- 0, k, J0 and the backtrack count are taken
// back) and stops the run, so that the iterate of minimum error is returned (reading A27).  mode 2 (RL): the candidate is
// the plane `cand` (the update was written there instead of f); ct->commit tells rl_commit_kernel whether to adopt it.
// mode 3 (OSEM, per cycle): the candidate h(k+1) is already in f, h(k) was saved by osem_backup_kernel; the cycle counter
// Ctrl::k advances here (nothing else on the device counts OSEM cycles), and a refused cycle is undone by osem_restore_kernel.
template <typename T>
__global__ void __launch_bounds__(256) err_kernel(const T *f, const T *d, const T *cand, const T *truth, size_t n, Ctrl *ct, DevOpts o,
                                                  Trace tr, double *part, int mode)
{
    __shared__ double red[2 * 32];
    if (mode == 1 && ct->err_pending == 0) return;
    if (mode >= 2 && ct->status != 0) return;
    const bool pend = mode == 1 && ct->pending != 0;
    const T lam = (T)ct->lambda;
    double acc[2] = {0.0, 0.0};
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        T v = mode == 2 ? cand[i] : f[i];
        if (pend) v = v + lam * d[i];
        const double t = (double)truth[i], e = (double)v - t;
        acc[0] += e * e; acc[1] += t * t;
    }
    block_reduce_sum<2>(acc, red);
    if (publish_partials<2>(acc, part, blockIdx.x, gridDim.x, &ct->counter[TK_ERR])) {
        final_sum<2>(acc, part, gridDim.x, red);
        if (threadIdx.x == 0) {
            const double rho = sqrt(acc[0]) / sqrt(acc[1]);
            if (mode == 0) {
                ct->err = rho;
                if (tr.err) tr.err[0] = rho;
            } else {
                const int k = ct->k + (mode == 3 ? 1 : 0);             // index of the candidate iterate
                if (tr.err) tr.err[k] = rho;
                ct->err_pending = 0;
                if (mode == 3) ct->k = k;
                if (o.stop_rule == SGP_STOP_MINERR && rho > ct->err) {
                    ct->status = SGP_REASON_MINERR;
                    ct->k = k - 1;
                    if (mode == 1) { ct->pending = 0; ct->J = ct->Jprev; ct->total_backtracks -= ct->nbt_last; }
                    ct->commit = 0;
                } else {
                    ct->err = rho;
                    ct->commit = 1;
                }
            }
        }
    }
}

// RL with the Eq.25 rule: adopt the candidate update unless err_kernel refused it
template <typename T>
__global__ void rl_commit_kernel(T *f, const T *cand, size_t n, const Ctrl *ct)
{
    if (ct->commit == 0) return;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) f[i] = cand[i];
}

// OSEM with the Eq.25 rule: h(k) is kept in the plane `d` (unused by OSEM) while the cycle works on f in place ...
template <typename T>
__global__ void osem_backup_kernel(const T *f, T *keep, size_t n, const Ctrl *ct)
{
    if (ct->status != 0) return;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) keep[i] = f[i];
}
// ... and comes back when err_kernel (mode 3) refused the cycle: the run returns h(k), the iterate of minimum error.
// (The cycles that remain in a captured graph find the status set and `keep` unchanged, so repeating the copy is harmless.)
template <typename T>
__global__ void osem_restore_kernel(T *f, const T *keep, size_t n, const Ctrl *ct)
{
    if (!(ct->status == SGP_REASON_MINERR && ct->commit == 0)) return;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) f[i] = keep[i];
}

// ---------------------------------------------------------------- refresh_every (reading A21)
// First kernel of the refresh round that follows every iteration when the option is on: if the iteration just finished is
// one after which A_j f is recomputed (Ctrl::refresh_due, set by finish_iteration), the pending step is applied to f
// (a10) so that the transforms that follow see f(k+1); Ctrl::need_k1 tells the second instance of the ratio kernel, at
// the end of the round, whether the ratio has to be formed again from the recomputed q.
template <typename T>
__global__ void apply_pending_kernel(T *f, const T *d, size_t n, Ctrl *ct)
{
    const bool due = ct->refresh_due != 0 && ct->status == 0;
    if (blockIdx.x == 0 && threadIdx.x == 0) ct->need_k1_next = due ? 1 : 0;
    if (!due || ct->pending == 0) return;
    const T lam = (T)ct->lambda;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) f[i] = f[i] + lam * d[i];
}
// closes the bracket: pending <- 0 after every CTA of apply_pending_kernel has read it; hands need_k1 to the ratio kernel;
// and sets the status of the SHADOW control block that the column pass of the refresh round tests (0 = run, 1 = not this
// iteration), so that the column kernel needs no test of its own for the refresh round
template <int DUMMY = 0> __global__ void refresh_flags_kernel(Ctrl *ct, Ctrl *shadow)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        const bool due = ct->refresh_due != 0 && ct->status == 0;
        if (due) ct->pending = 0;
        ct->need_k1 = ct->need_k1_next;
        shadow->status = due ? 0 : 1;
    }
}

// ---------------------------------------------------------------- Gaussian of the smoothed constant start (A28)
// periodic Gaussian of standard deviation sigma pixels centred on pixel (0,0), divided by `sum` (computed by the host)
template <typename T>
__global__ void gauss_plane_kernel(T *out, int ny, int nx, double sigma, double sum)
{
    const size_t n = (size_t)ny * nx;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const int y = (int)(i / nx), x = (int)(i - (size_t)y * nx);
        const double dy = y <= ny / 2 ? y : y - ny, dx = x <= nx / 2 ? x : x - nx;
        out[i] = (T)(exp(-(dy * dy + dx * dx) / (2.0 * sigma * sigma)) / sum);
    }
}

}  // namespace sgpk
