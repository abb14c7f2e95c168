// aux.cuh -- the elementwise kernels around the FFT passes: Armijo backtracking (a9), the final lazy update (a10),
// and the set-up / marshalling kernels (not on the hot path).
#pragma once
#include "ew.cuh"

namespace sgpk {

// ---------------------------------------------------------------- a9 (backtracks) + a11
// The Armijo loop lambda <- theta lambda for the iterations whose lambda = 1 was rejected by the
// line-search kernel.  Every trial is one elementwise pass over q_j + lambda u_j (no FFT).  It runs as a PROLOGUE of the
// ratio kernel K1 (row_fwd.cuh), which follows the line-search kernel anyway: there is no kernel of its own and, when
// lambda = 1 was accepted (the usual case), no work at all.
//
// Grid-wide coordination WITHOUT assuming that the CTAs of the grid are resident together (round 1 used a spinning
// grid barrier, which hangs when another plan or an SM-limited context keeps part of the grid from being scheduled):
// a trial is cut into `nchunks` fixed chunks of pixels; CTAs draw tickets T = 0, 1, 2, ... from one counter, ticket T
// being chunk T % nchunks of trial T / nchunks.  A CTA holding a ticket of trial t waits until trials < t are decided
// -- it waits only for chunks that are held by RUNNING CTAs (tickets are handed out in order), so it always makes
// progress; CTAs scheduled late find the decision taken and leave.  The CTA that finishes the last chunk of a trial
// sums the per-chunk partials in a fixed order (runs are deterministic whatever CTA did which chunk) and takes the
// decision: accept (book-keeping by finish_iteration), give up (A16) or open the next trial.
template <typename T> struct vec4_of;
template <> struct vec4_of<float>  { using type = float4;  static constexpr int N = 4; };
template <> struct vec4_of<double> { using type = double2; static constexpr int N = 2; };

constexpr int kBtVecPerThread = 4;                                   // vectors per thread and chunk
template <typename T> __host__ __device__ constexpr size_t bt_chunk_elems() { return (size_t)256 * kBtVecPerThread * vec4_of<T>::N; }

__device__ __forceinline__ unsigned int ld_volatile_u32(const unsigned int *p) { return *reinterpret_cast<const volatile unsigned int *>(p); }

// The arguments live in a block in DEVICE memory (BtInfo, written by run() before the loop) and the function is NOT
// inlined: compiled into the ratio kernel -- or called with arguments that take the address of the kernel's parameter
// block -- it costs that kernel 7 us per launch at 2048^2 whether it runs or not (measured: 26.4 vs 19.0 us).
template <typename T> struct BtInfo {
    Geom G; DevOpts o; Trace tr; Ctrl *ct;
    const T *q, *u, *g, *b;                      // p contiguous planes each; q: buffer Ctrl::qsel at + qsel*qbuf
    size_t qbuf;
    int b_is_array;
    unsigned int nchunks;                        // chunks per trial, ~ one per CTA of the ratio kernel
    unsigned int chunk_batches;                  // batches (of 256 x kBtVecPerThread vectors) per chunk
    double bconst[kMaxP];
    double *part;                                // nchunks doubles
    unsigned int *sync;                          // the counters, one 128-byte line each (kBtNext ...): tickets and polls do not share a line with each other or with Ctrl
};
enum BtSyncSlot { kBtNext = 0, kBtDone = 32, kBtDecided = 64, kBtFinal = 65, kBtSyncWords = 96 };
// Called by ALL threads of a CTA (blockDim.x <= 256).
template <typename T>
__device__ __noinline__ void backtrack_rounds(const BtInfo<T> *__restrict__ I)
{
    __shared__ double red[32];
    const BtInfo<T> &P = *I;
    using V = typename vec4_of<T>::type;
    constexpr int VN = vec4_of<T>::N;
    __shared__ unsigned int s_ticket;
    __shared__ int s_state;
    Ctrl *ct = P.ct;
    const Geom &G = P.G;
    const int tid = threadIdx.x, nthr = blockDim.x;
    const size_t n = (size_t)G.ny * G.nx, ntot = n * (size_t)G.p;
    // everything the trials need is read BEFORE the first ticket is drawn (see the header)
    const int k = ct->k;
    const T *qcur = P.q + (size_t)ct->qsel * P.qbuf;
    const double Jref = ct->Jref, gd = ct->gd;
    double forced_lambda = 0.0;
    bool forced = false;
    if (P.tr.force_lambda) {
        const double fl = P.tr.force_lambda[k];
        if (isfinite(fl)) { forced = true; forced_lambda = fl; }
    }
    __threadfence();
    for (;;) {
        if (tid == 0) s_ticket = atomicAdd(&P.sync[kBtNext], 1u);
        __syncthreads();
        const unsigned int ticket = s_ticket;
        const unsigned int nchunks = P.nchunks;
        const unsigned int trial = ticket / nchunks, chunk = ticket - trial * nchunks;
        if (tid == 0) {
            int st = 0;                                               // 0 = go, 1 = decision already taken
            for (;;) {
                if (ld_volatile_u32(&P.sync[kBtFinal]) != 0u) { st = 1; break; }
                if (ld_volatile_u32(&P.sync[kBtDecided]) >= trial) break;
                __nanosleep(100);
            }
            __threadfence();
            s_state = st;
        }
        __syncthreads();
        if (s_state != 0) return;
        double lambda = 1.0;
        for (unsigned int i = 0; i <= trial; ++i) lambda *= P.o.theta;       // PAPER.md:124, the oracle's own sequence of products
        if (forced) lambda = forced_lambda;
        const T lam = (T)lambda;
        // ---- this chunk of J(lambda) = sum_j sum_S kl(g_j, q_j + lambda u_j + b_j)
        double acc[1] = {0.0};
        const int CHV = 256 * kBtVecPerThread * (int)P.chunk_batches; // vectors per chunk
        const size_t e_begin = (size_t)chunk * (size_t)CHV * VN;
        // kBtVecPerThread vectors per thread and step, all loads issued before the first use
        for (int v0 = tid; v0 < CHV; v0 += nthr * kBtVecPerThread) {
            V q4[kBtVecPerThread], u4[kBtVecPerThread], g4[kBtVecPerThread];
            bool ok[kBtVecPerThread];
#pragma unroll
            for (int v = 0; v < kBtVecPerThread; ++v) {
                const int vi = v0 + v * nthr;
                const size_t e0 = e_begin + (size_t)vi * VN;
                ok[v] = vi < CHV && e0 < ntot;
                if (ok[v]) {
                    q4[v] = *reinterpret_cast<const V *>(qcur + e0); u4[v] = *reinterpret_cast<const V *>(P.u + e0);
                    g4[v] = *reinterpret_cast<const V *>(P.g + e0);
                }
            }
#pragma unroll
            for (int v = 0; v < kBtVecPerThread; ++v) {
                if (!ok[v]) continue;
                const size_t e0 = e_begin + (size_t)(v0 + v * nthr) * VN;
                const int j = (int)(e0 / n);
                const size_t ip = e0 - (size_t)j * n;
                const int y = (int)(ip / G.nx), x = (int)(ip - (size_t)y * G.nx);
                if ((unsigned)(y - G.oy) >= (unsigned)G.sy) continue;
                const T bc = (T)P.bconst[j];
                const T *qa = reinterpret_cast<const T *>(&q4[v]), *ua = reinterpret_cast<const T *>(&u4[v]), *ga = reinterpret_cast<const T *>(&g4[v]);
                if constexpr (VN == 4) {
                    T yv[4], gv[4]; bool s[4];
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        s[c] = (unsigned)(x + c - G.ox) < (unsigned)G.sx;
                        const T bb = P.b_is_array ? P.b[e0 + c] : bc;
                        yv[c] = (T)((T)(qa[c] + lam * ua[c]) + bb); gv[c] = ga[c];
                    }
                    acc[0] += (double)kl_quad(gv, yv, s);
                } else {
#pragma unroll
                    for (int c = 0; c < VN; ++c) {
                        if ((unsigned)(x + c - G.ox) < (unsigned)G.sx) {
                            const T bb = P.b_is_array ? P.b[e0 + c] : bc;
                            acc[0] += (double)kl_term(ga[c], (T)((T)(qa[c] + lam * ua[c]) + bb));
                        }
                    }
                }
            }
        }
        block_reduce_sum<1>(acc, red);
        __shared__ int s_last;
        if (tid == 0) {
            P.part[chunk] = acc[0];
            __threadfence();
            s_last = (atomicAdd(&P.sync[kBtDone], 1u) == nchunks - 1) ? 1 : 0;
        }
        __syncthreads();
        if (s_last) {                                                 // this CTA closes the trial
            __threadfence();
            double tot[1] = {0.0};
            for (unsigned int c = tid; c < nchunks; c += nthr) tot[0] += __ldcg(&P.part[c]);
            block_reduce_sum<1>(tot, red);
            if (tid == 0) {
                const double Jnew = tot[0];
                const int nbt = (int)trial + 1;
                const bool accepted = forced || (isfinite(Jnew) && Jnew <= Jref + P.o.beta * lambda * gd);
                P.sync[kBtDone] = 0;
                if (accepted) {
                    finish_iteration(ct, P.o, P.tr, lambda, Jnew, forced ? 0 : nbt, 2);
                    __threadfence();
                    *reinterpret_cast<volatile unsigned int *>(&P.sync[kBtFinal]) = 1u;
                } else if (nbt >= P.o.max_backtracks) {                // A16
                    ct->status = SGP_ERR_LINESEARCH;
                    __threadfence();
                    *reinterpret_cast<volatile unsigned int *>(&P.sync[kBtFinal]) = 1u;
                } else {
                    __threadfence();
                    *reinterpret_cast<volatile unsigned int *>(&P.sync[kBtDecided]) = trial + 1u;
                }
            }
            __syncthreads();
        }
    }
}

// f_out = f + lambda d if a step is still pending (a10, lazy), else f
template <typename T>
__global__ void final_update_kernel(const T *f, const T *d, T *f_out, size_t n, const Ctrl *ct)
{
    const bool pend = ct->pending != 0;
    const T lam = (T)ct->lambda;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        T v = f[i];
        if (pend) v = v + lam * d[i];
        f_out[i] = v;
    }
}

// addresses of the caller's arrays of a batched run (see embed_inputs_batched_kernel below)
struct BatchTab {
    const void *const *g, *const *b, *const *f0;
    void *const *f_out;
};
template <typename T>
__global__ void final_update_batched_kernel(BatchTab tab, const T *f, const T *d, size_t n, const Ctrl *ct, size_t slab)
{
    const size_t off = (size_t)blockIdx.z * slab;
    const Ctrl *ctz = bshift(ct, off);
    const T *fz = bshift(f, off), *dz = bshift(d, off);
    T *f_out = (T *)tab.f_out[blockIdx.z];
    const bool pend = ctz->pending != 0;
    const T lam = (T)ctz->lambda;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        T v = fz[i];
        if (pend) v = v + lam * dz[i];
        f_out[i] = v;
    }
}

// ---------------------------------------------------------------- set-up and marshalling kernels (not on the hot path)
// sum of a plane (PSF volume) with a non-finite check -> ct->psf_sum.  Per-CTA partials, the last CTA adds them in a
// fixed order (a single CTA of 1024 threads took 1.9 ms for a 2048^2 plane: 4096 dependent loads per thread, in every *_host call)
template <typename T>
__global__ void __launch_bounds__(256) plane_sum_kernel(const T *x, size_t n, Ctrl *ct, double *part /* gridDim.x doubles */)
{
    __shared__ double red[32];
    double acc[1] = {0.0};
    bool bad = false;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        double v = (double)x[i];
        if (!isfinite(v)) bad = true;
        acc[0] += v;
    }
    if (bad) acc[0] = NAN;
    block_reduce_sum<1>(acc, red);
    if (publish_partials<1>(acc, part, blockIdx.x, gridDim.x, &ct->counter[TK_ERR])) {
        final_sum<1>(acc, part, gridDim.x, red);
        if (threadIdx.x == 0) ct->psf_sum = acc[0];
    }
}

// transfer function from the raw column-FFT output: scale by 1/(ny nx) and split the packed column of tile 0
// into A = (K0+KM)/2 (column 0 of khat) and B = (K0-KM)/2 (khatB), K0[ky] = (C[ky] + conj C[-ky])/2, KM[ky] = -i (C[ky] - conj C[-ky])/2
template <typename T>
__global__ void khat_fixup_kernel(const cx<T> *raw, cx<T> *khat, cx<T> *khatB, int ny, int nx, int Cc)
{
    using C = cx<T>;
    const size_t n = (size_t)ny * (nx / 2);
    const T sc = (T)(1.0 / ((double)ny * (double)nx));
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        C v = raw[i];
        const size_t tile = i / ((size_t)ny * Cc), rem = i - tile * ((size_t)ny * Cc);
        const int ky = (int)(rem / Cc), c = (int)(rem - (size_t)ky * Cc);
        if (tile == 0 && c == 0) {
            const int kyn = ky == 0 ? 0 : ny - ky;
            const C ct = cconj(raw[(size_t)kyn * Cc]);
            const C K0 = mk<T>((T)0.5 * (v.x + ct.x), (T)0.5 * (v.y + ct.y));
            const C Dm = mk<T>((T)0.5 * (v.x - ct.x), (T)0.5 * (v.y - ct.y));
            const C KM = mk<T>(Dm.y, -Dm.x);
            khat[i] = mk<T>((T)0.5 * (K0.x + KM.x) * sc, (T)0.5 * (K0.y + KM.y) * sc);
            khatB[ky] = mk<T>((T)0.5 * (K0.x - KM.x) * sc, (T)0.5 * (K0.y - KM.y) * sc);
        } else {
            khat[i] = mk<T>(v.x * sc, v.y * sc);
        }
    }
}

// g_j, b_j (sy x sx, caller's arrays) -> S-bar planes; negative g clamped to 0 (A17) or flagged (strict);
// also sum_S (g - b) for the constant start (A14), accumulated per block into part[] (deterministic final sum later)
template <typename T>
__device__ __forceinline__ void embed_inputs_body(const T *g, const T *b, T *G_out, T *B_out, const Geom &Gm, double bconst, int strict,
                                                  Ctrl *ct, double *part)
{
    __shared__ double red[32];
    const size_t n = (size_t)Gm.ny * Gm.nx;
    double acc[1] = {0.0};
    int flag = 0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const int y = (int)(i / Gm.nx), x = (int)(i - (size_t)y * Gm.nx);
        T gv = (T)0, bv = (T)0;
        if (in_S(Gm, y, x)) {
            const size_t s = (size_t)(y - Gm.oy) * Gm.sx + (x - Gm.ox);
            gv = g[s];
            bv = b ? b[s] : (T)bconst;
            if (!isfinite((double)gv)) flag |= 1;
            if (gv < (T)0) { if (strict) flag |= 2; gv = (T)0; }
            acc[0] += (double)gv - (double)bv;
        }
        G_out[i] = gv;
        if (B_out) B_out[i] = bv;
    }
    if (flag) atomicOr(&ct->flag_data, flag);
    block_reduce_sum<1>(acc, red);
    if (threadIdx.x == 0) part[blockIdx.x] = acc[0];
}
template <typename T>
__global__ void embed_inputs_kernel(const T *g, const T *b, T *G_out, T *B_out, Geom Gm, double bconst, int strict,
                                    Ctrl *ct, double *part)
{
    embed_inputs_body<T>(g, b, G_out, B_out, Gm, bconst, strict, ct, part);
}

// Batched plans (sgp_plan_run_batched): the set-up kernels of ALL problems in one launch each, blockIdx.z = problem (and
// blockIdx.y = image where there is one).  The caller's arrays are separate allocations, so their addresses come from a table in
// device memory: [g: nb*p][b: nb*p][f0: nb][f_out: nb]; the plan's own per-problem arrays are `slab` bytes apart (ew.cuh).
template <typename T>
__global__ void embed_inputs_batched_kernel(BatchTab tab, T *Gp, T *Bp, Geom Gm, int p, int b_is_array, int strict,
                                            Ctrl *ct, double *part_misc, size_t slab)
{
    const int j = blockIdx.y, z = blockIdx.z;
    const size_t n = (size_t)Gm.ny * Gm.nx, off = (size_t)z * slab;
    Ctrl *ctz = bshift(ct, off);
    embed_inputs_body<T>((const T *)tab.g[z * p + j], b_is_array ? (const T *)tab.b[z * p + j] : nullptr, bshift(Gp, off) + (size_t)j * n,
                         b_is_array ? bshift(Bp, off) + (size_t)j * n : nullptr, Gm, ctz->bconst[j], strict, ctz,
                         bshift(part_misc, off) + (size_t)j * 1024);
}

// c = max(0, (1/p) sum_j mean_S (g_j - b_j)) (A14); single thread, partials in fixed order.  Also the flux of the
// flux-constrained projection (A26): flux_value if > 0, else max(0, (1/p) sum_j sum_S (g_j - b_j)).
template <typename T> __global__ void const_start_kernel(const double *part, int nparts, double denom, int p, double flux_value, Ctrl *ct)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        double s = 0.0;
        for (int i = 0; i < nparts; ++i) s += part[i];
        double c = s / denom;
        ct->c0 = c < 0.0 ? 0.0 : c;
        double fc = flux_value > 0.0 ? flux_value : s / (double)p;
        ct->flux_c = fc < 0.0 ? 0.0 : fc;
    }
}

template <typename T> __global__ void const_start_batched_kernel(const double *part_misc, int nparts, double denom, int p, double flux_value, Ctrl *ct, size_t slab)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        const size_t off = (size_t)blockIdx.z * slab;
        const double *part = bshift(part_misc, off);
        Ctrl *ctz = bshift(ct, off);
        double s = 0.0;
        for (int i = 0; i < nparts; ++i) s += part[i];
        double c = s / denom;
        ctz->c0 = c < 0.0 ? 0.0 : c;
        double fc = flux_value > 0.0 ? flux_value : s / (double)p;
        ctz->flux_c = fc < 0.0 ? 0.0 : fc;
    }
}

// start point f(0): user image / constant / zero / g_1, restricted to R (A11)
template <typename T>
__device__ __forceinline__ void start_point_body(T *f, const T *f0, const T *g0, const T *alphaR, const Geom &Gm, int init, Ctrl *ct)
{
    const size_t n = (size_t)Gm.ny * Gm.nx;
    int flag = 0;
    const T c0 = (T)ct->c0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const bool inR = Gm.masked ? (alphaR[i] > (T)0) : true;
        T v = (T)0;
        if (init == SGP_INIT_USER) { T u = f0[i]; if (!(u >= (T)0)) flag = 4; v = inR ? u : (T)0; }
        else if (init == SGP_INIT_CONST) v = inR ? c0 : (T)0;
        else if (init == SGP_INIT_G) {
            const int y = (int)(i / Gm.nx), x = (int)(i - (size_t)y * Gm.nx);
            T gv = g0[i];
            v = (inR && in_S(Gm, y, x) && gv > (T)0) ? gv : (T)0;
        }
        f[i] = v;
    }
    if (flag) atomicOr(&ct->flag_data, flag);
}
template <typename T>
__global__ void start_point_kernel(T *f, const T *f0, const T *g0, const T *alphaR, Geom Gm, int init, Ctrl *ct)
{
    start_point_body<T>(f, f0, g0, alphaR, Gm, init, ct);
}
template <typename T>
__global__ void start_point_batched_kernel(BatchTab tab, T *f, const T *Gp, const T *alphaR, Geom Gm, int init, Ctrl *ct, size_t slab)
{
    const size_t off = (size_t)blockIdx.z * slab;
    start_point_body<T>(bshift(f, off), init == SGP_INIT_USER ? (const T *)tab.f0[blockIdx.z] : nullptr, bshift(Gp, off), alphaR, Gm, init, bshift(ct, off));
}

// boundary weights (Eq.19-20): alpha += alpha_j; M_R &= (alpha_j >= sigma)
template <typename T>
__global__ void alpha_accum_kernel(const T *aj, T *alpha, unsigned char *MR, size_t n, double sigma, int first)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const T a = aj[i];
        alpha[i] = first ? a : alpha[i] + a;
        const unsigned char ok = ((double)a >= sigma) ? 1 : 0;
        MR[i] = first ? ok : (unsigned char)(MR[i] & ok);
    }
}
// alphaR = alpha on R, 0 outside (so that "alphaR > 0" is M_R and 1/alphaR is M_R/alpha of Eq.21/23)
template <typename T>
__global__ void alpha_finish_kernel(const T *alpha, const unsigned char *MR, T *alphaR, size_t n)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        alphaR[i] = MR[i] ? alpha[i] : (T)0;
}

template <typename T>
__global__ void copy_plane_kernel(const T *src, T *dst, size_t n)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) dst[i] = src[i];
}

// tile-major half spectrum <-> ny x (nx/2+1) interleaved complex (numpy.fft.rfft2 layout); column kernel CM_FWD
// output in, or input for the inverse.  Only for sgp_plan_rfft2 / irfft2 (tests, cuFFT comparison).
template <typename T>
__global__ void spec_to_rfft2_kernel(const cx<T> *spec, cx<T> *out, int ny, int nx, int Cc)
{
    using C = cx<T>;
    const int M = nx / 2;
    const size_t n = (size_t)ny * (M + 1);
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const int ky = (int)(i / (M + 1)), kx = (int)(i - (size_t)ky * (M + 1));
        C r;
        if (kx == 0 || kx == M) {
            const int kyn = ky == 0 ? 0 : ny - ky;
            const C a = spec[(size_t)ky * Cc], ct = cconj(spec[(size_t)kyn * Cc]);
            if (kx == 0) r = mk<T>((T)0.5 * (a.x + ct.x), (T)0.5 * (a.y + ct.y));
            else { const C Dm = mk<T>((T)0.5 * (a.x - ct.x), (T)0.5 * (a.y - ct.y)); r = mk<T>(Dm.y, -Dm.x); }
        } else {
            r = spec[(size_t)(kx / Cc) * ((size_t)ny * Cc) + (size_t)ky * Cc + kx % Cc];
        }
        out[i] = r;
    }
}
template <typename T>
__global__ void rfft2_to_spec_kernel(const cx<T> *in, cx<T> *spec, int ny, int nx, int Cc, T scale)
{
    using C = cx<T>;
    const int M = nx / 2;
    const size_t n = (size_t)ny * M;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const size_t tile = i / ((size_t)ny * Cc), rem = i - tile * ((size_t)ny * Cc);
        const int ky = (int)(rem / Cc), c = (int)(rem - (size_t)ky * Cc);
        const int kx = (int)tile * Cc + c;
        C r;
        if (kx == 0) {   // packed: F[ky][0] + i F[ky][M]
            const C a = in[(size_t)ky * (M + 1)], b = in[(size_t)ky * (M + 1) + M];
            r = mk<T>(a.x - b.y, a.y + b.x);
        } else r = in[(size_t)ky * (M + 1) + kx];
        spec[i] = mk<T>(r.x * scale, r.y * scale);
    }
}

}  // namespace sgpk
