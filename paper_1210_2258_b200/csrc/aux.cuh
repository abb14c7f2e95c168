// aux.cuh -- the elementwise kernels around the FFT passes: Armijo backtracking (a9), the final lazy update (a10),
// and the set-up / marshalling kernels (not on the hot path).
#pragma once
#include "ew.cuh"

namespace sgpk {

// ---------------------------------------------------------------- a9 (backtracks) + a11
// Launched every iteration; returns at once when lambda = 1 was accepted by the RI_LS epilogue (the usual case).
// Otherwise the Armijo loop lambda <- theta lambda runs here: every trial is one elementwise
// pass over q_j + lambda u_j (no FFT), one grid-wide barrier, and the same decision taken redundantly by every
// CTA.  The grid is sized by the occupancy API so that all CTAs are resident together, and the barrier is a
// sense-reversing counter in the control block: an ordinary launch, because the empty cooperative launches of the
// usual case cost 7 us per iteration.  The accepted step is NOT applied here: f + lambda d and q_j + lambda u_j
// are formed by the next iteration's kernels (K1 in repair mode, Ctrl::need_k1 = 2; K3) or by final_update_kernel.
template <typename T> struct BtParams {
    Geom G;
    DevOpts o;
    Trace tr;
    Ctrl *ct;
    const T *q, *u, *g, *b;                      // image j at + j*plane; q: buffer Ctrl::qsel at + qsel*qbuf
    size_t plane, qbuf;
    int b_is_array;
    double bconst[kMaxP];
    double *part;                                // gridDim.x doubles
};

template <typename T> struct vec4_of;
template <> struct vec4_of<float>  { using type = float4;  static constexpr int N = 4; };
template <> struct vec4_of<double> { using type = double2; static constexpr int N = 2; };

// all CTAs of the grid (resident together) meet here; bar[0] = arrival count, bar[1] = generation
__device__ __forceinline__ void grid_barrier(unsigned int *bar)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned int gen = atomicAdd(&bar[1], 0u);
        __threadfence();
        if (atomicAdd(&bar[0], 1u) == gridDim.x - 1) {
            atomicExch(&bar[0], 0u);
            __threadfence();
            atomicAdd(&bar[1], 1u);
        } else {
            while (atomicAdd(&bar[1], 0u) == gen) __nanosleep(64);
        }
        __threadfence();
    }
    __syncthreads();
}

template <typename T>
__global__ void __launch_bounds__(256) backtrack_kernel(const BtParams<T> P)
{
    using V = typename vec4_of<T>::type;
    constexpr int VN = vec4_of<T>::N;
    __shared__ double red[32];
    __shared__ double s_J;
    Ctrl *ct = P.ct;
    if (ct->status != 0 || ct->accepted != 0) return;
    const Geom &G = P.G;
    const size_t n = (size_t)G.ny * G.nx, nv = n / VN;
    const size_t gtid = (size_t)blockIdx.x * blockDim.x + threadIdx.x, gstride = (size_t)gridDim.x * blockDim.x;
    const int k = ct->k;
    const T *qcur = P.q + (size_t)ct->qsel * P.qbuf;           // A_j f(k): the buffer the line-search kernel read
    const double Jref = ct->Jref, gd = ct->gd;
    double lambda = 1.0, Jnew = ct->Jtrial;
    bool accepted = false, forced = false;
    if (P.tr.force_lambda) {
        const double fl = P.tr.force_lambda[k];
        if (isfinite(fl)) { forced = true; lambda = fl / P.o.theta; }
    }
    grid_barrier(&ct->counter[6]);                             // every CTA has read the control block
    int nbt = 0;
    while (!accepted) {
        if (!forced && nbt >= P.o.max_backtracks) {            // A16
            if (blockIdx.x == 0 && threadIdx.x == 0) ct->status = SGP_ERR_LINESEARCH;
            return;
        }
        lambda *= P.o.theta;
        nbt++;
        const T lam = (T)lambda;
        double acc[1] = {0.0};
        for (int j = 0; j < G.p; ++j) {
            const T *q = qcur + (size_t)j * P.plane, *u = P.u + (size_t)j * P.plane, *g = P.g + (size_t)j * P.plane;
            const T *b = P.b_is_array ? P.b + (size_t)j * P.plane : nullptr;
            const T bc = (T)P.bconst[j];
            // four vectors per thread and step, all loads issued before the first use (the trial is one pass over three
            // planes: what counts is how many bytes each thread has in flight)
            constexpr int UN = 4;
            for (size_t i0 = gtid; i0 < nv; i0 += UN * gstride) {
                V q4[UN], u4[UN], g4[UN];
                bool ok[UN];
#pragma unroll
                for (int k4 = 0; k4 < UN; ++k4) {
                    const size_t i = i0 + (size_t)k4 * gstride;
                    ok[k4] = i < nv;
                    if (ok[k4]) {
                        q4[k4] = reinterpret_cast<const V *>(q)[i]; u4[k4] = reinterpret_cast<const V *>(u)[i];
                        g4[k4] = reinterpret_cast<const V *>(g)[i];
                    }
                }
#pragma unroll
                for (int k4 = 0; k4 < UN; ++k4) {
                    if (!ok[k4]) continue;
                    const size_t e0 = (i0 + (size_t)k4 * gstride) * VN;
                    const int y = (int)(e0 / G.nx), x = (int)(e0 - (size_t)y * G.nx);
                    if ((unsigned)(y - G.oy) >= (unsigned)G.sy) continue;
                    const T *qa = reinterpret_cast<const T *>(&q4[k4]), *ua = reinterpret_cast<const T *>(&u4[k4]), *ga = reinterpret_cast<const T *>(&g4[k4]);
                    if constexpr (VN == 4) {
                        T yv[4], gv[4]; bool s[4];
#pragma unroll
                        for (int c = 0; c < 4; ++c) {
                            s[c] = (unsigned)(x + c - G.ox) < (unsigned)G.sx;
                            const T bb = b ? b[e0 + c] : bc;
                            yv[c] = (T)((T)(qa[c] + lam * ua[c]) + bb); gv[c] = ga[c];
                        }
                        acc[0] += (double)kl_quad(gv, yv, s);
                    } else {
#pragma unroll
                        for (int c = 0; c < VN; ++c) {
                            if ((unsigned)(x + c - G.ox) < (unsigned)G.sx) {
                                const T bb = b ? b[e0 + c] : bc;
                                acc[0] += (double)kl_term(ga[c], (T)((T)(qa[c] + lam * ua[c]) + bb));
                            }
                        }
                    }
                }
            }
        }
        block_reduce_sum<1>(acc, red);
        if (threadIdx.x == 0) P.part[blockIdx.x] = acc[0];
        grid_barrier(&ct->counter[6]);
        double tot[1] = {0.0};
        for (unsigned int bI = threadIdx.x; bI < gridDim.x; bI += blockDim.x) tot[0] += __ldcg(&P.part[bI]);
        block_reduce_sum<1>(tot, red);
        if (threadIdx.x == 0) s_J = tot[0];
        __syncthreads();
        Jnew = s_J;
        accepted = forced || (isfinite(Jnew) && Jnew <= Jref + P.o.beta * lambda * gd);
        grid_barrier(&ct->counter[6]);     // partials may be overwritten by the next trial
    }
    if (forced) nbt = 0;
    // ---- book-keeping by the last CTA to finish (every CTA has read the control block by now)
    if (threadIdx.x == 0) {
        __threadfence();
        unsigned int tk = atomicAdd(&ct->counter[TK_BACKTRACK], 1u);
        if (tk == gridDim.x - 1) { ct->counter[TK_BACKTRACK] = 0; finish_iteration(ct, P.o, P.tr, lambda, Jnew, nbt, 2); }
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

// ---------------------------------------------------------------- set-up and marshalling kernels (not on the hot path)
// sum of a plane (PSF volume) with a non-finite check -> ct->psf_sum; single CTA
template <typename T>
__global__ void plane_sum_kernel(const T *x, size_t n, Ctrl *ct)
{
    __shared__ double red[32];
    double acc[1] = {0.0};
    bool bad = false;
    for (size_t i = threadIdx.x; i < n; i += blockDim.x) { double v = (double)x[i]; if (!isfinite(v)) bad = true; acc[0] += v; }
    if (bad) acc[0] = NAN;
    block_reduce_sum<1>(acc, red);
    if (threadIdx.x == 0) ct->psf_sum = acc[0];
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
__global__ void embed_inputs_kernel(const T *g, const T *b, T *G_out, T *B_out, Geom Gm, double bconst, int strict,
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

// c = max(0, (1/p) sum_j mean_S (g_j - b_j)) (A14); single thread, partials in fixed order
template <typename T> __global__ void const_start_kernel(const double *part, int nparts, double denom, Ctrl *ct)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        double s = 0.0;
        for (int i = 0; i < nparts; ++i) s += part[i];
        double c = s / denom;
        ct->c0 = c < 0.0 ? 0.0 : c;
    }
}

// start point f(0): user image / constant / zero / g_1, restricted to R (A11)
template <typename T>
__global__ void start_point_kernel(T *f, const T *f0, const T *g0, const T *alphaR, Geom Gm, int init, Ctrl *ct)
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
