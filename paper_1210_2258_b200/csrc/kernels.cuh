// kernels.cuh -- the hot-path kernels of the SGP / RL iteration.
//
// Data layout.  Real planes are row-major ny x nx.  A half spectrum of a real plane holds nx/2 complex
// numbers per row: entry kx = 1..nx/2-1 is the DFT coefficient, entry 0 packs the two real coefficients
// (kx = 0, kx = nx/2) as (re, im).  Spectra are stored COLUMN-TILE-MAJOR: tile = kx / C, and inside a tile
// element (ky, kx % C) sits at ky*C + kx%C, so a block of the column kernel reads one contiguous chunk of
// ny*C complex numbers and a block of the row kernels writes RB*C contiguous numbers per tile.
//
// Row kernels: one CTA transforms RB rows; the elementwise work of the iteration (ratio, gradient,
// scaling, projection, line-search sums) is fused into their load / store stages.
// Column kernel: one CTA owns a tile: forward column FFTs, pointwise product with the transfer
// function(s) (conjugated and summed over the images for A^T), inverse column FFTs -- the spectrum
// never leaves the registers between the three steps.
#pragma once
#include <cooperative_groups.h>
#include "fft_core.cuh"
#include "sgp_dev.cuh"

namespace sgpk {
namespace cg = cooperative_groups;

enum RowFwdMode { RF_PLAIN = 0, RF_PSF = 1, RF_MASK_S = 2, RF_RATIO = 3, RF_PROJECT = 4 };
enum RowInvMode { RI_PLAIN = 0, RI_GRAD = 1, RI_LS = 2, RI_QJ = 3, RI_RLMINMAX = 4, RI_RLUPDATE = 5 };
enum MaskMode { MM_NONE = 0, MM_S = 1, MM_R = 2 };
enum QJSub { QJ_INIT = 0, QJ_RL = 1, QJ_PLAIN = 2 };
enum Ticket { TK_GRAD = 0, TK_LS = 1, TK_QJ = 2, TK_MINMAX = 3, TK_UPDATE = 4 };

template <typename T> struct RowParams {
    Geom G;
    DevOpts o;
    Trace tr;
    Ctrl *ct;
    int mode, submode, maskmode, b_is_array;
    const T *in0, *in1, *in2, *in3;   // real planes; image j at + j*plane
    T *out0;
    cx<T> *spec;                      // spectrum of image j at + j*specplane
    size_t plane, specplane;
    const cx<T> *tw;                  // exp(-2 pi i k / (nx/2)), k < nx/2
    const cx<T> *twh;                 // exp(-2 pi i k / nx),     k <= nx/2
    const T *alphaR;                  // boundary problems: alpha on R, 0 outside R (Eq.19-20)
    double *part, *part2;
    double bconst[kMaxP];
    int cy, cxs;                      // PSF centre (RF_PSF)
    int check_status;                 // 1: return immediately when ct->status != 0
};

template <typename T> struct ColParams {
    Geom G;
    Ctrl *ct;
    const cx<T> *in;                  // spectrum of image j at + j*specplane
    cx<T> *out;
    const cx<T> *khat;                // tiled transfer function of image j at + j*specplane (scaled by 1/(ny nx))
    const cx<T> *khatB;               // column-0 companion of image j at + j*ny
    size_t specplane;
    const cx<T> *tw;                  // exp(-2 pi i k / ny)
    cx<T> *pack;                      // ny entries of scratch for the packed column of tile 0
    int p;
    int check_status;
};

// ---------------------------------------------------------------- elementwise pieces
// One summand of Eq.2: g ln(g/y) + y - g with y = A f + b, evaluated without
// cancellation (A17): g = 0 gives y; y <= 0 drops the log term.
__device__ __forceinline__ double kl_term(double g, double y)
{
    if (!(g > 0.0)) return y;
    if (!(y > 0.0)) return y - g;
    double t = (y - g) / g;
    return g * (t - log1p(t));
}
// float version: with u = (y-g)/(y+g), ln(y/g) = 2 atanh(u), hence
//   g ln(g/y) + y - g = u [ (y-g) - 2 g u^2 (1/3 + u^2/5 + u^4/7 + ...) ]      (|u| < 0.2)
// and the plain form (y-g) - g log1p((y-g)/g) otherwise (no cancellation there).
__device__ __forceinline__ float kl_term(float g, float y)
{
    if (!(g > 0.f)) return y;
    if (!(y > 0.f)) return y - g;
    const float dy = y - g;
    const float u = dy / (y + g);
    const float w = u * u;
    if (w < 0.04f) {
        float S = fmaf(w, 1.f / 13.f, 1.f / 11.f);
        S = fmaf(w, S, 1.f / 9.f);
        S = fmaf(w, S, 1.f / 7.f);
        S = fmaf(w, S, 1.f / 5.f);
        S = fmaf(w, S, 1.f / 3.f);
        return u * (dy - 2.f * g * w * S);
    }
    return dy - g * log1pf(dy / g);
}
// ratio g/(Af+b) of Eq.1/11; 0 where the denominator is <= 0 (A17)
template <typename T> __device__ __forceinline__ T ratio_term(T g, T y) { return (y > (T)0) ? g / y : (T)0; }
template <typename T> __device__ __forceinline__ T clipT(T f, T L1, T L2) { return fmin(L2, fmax(L1, f)); }

template <typename T> __device__ __forceinline__ cx<T> ld2(const T *p) { return *reinterpret_cast<const cx<T> *>(p); }
template <typename T> __device__ __forceinline__ void st2(T *p, cx<T> v) { *reinterpret_cast<cx<T> *>(p) = v; }

// ---------------------------------------------------------------- row forward (real rows -> half spectrum)
// grid = (ny/RB, images), block = RB * (L/E) threads, dynamic smem = RB * row_stride(L) complex.
__host__ __device__ constexpr int row_stride(int L) { return fft_padded_len(L) + 2; }

template <typename T, int L>
__global__ void __launch_bounds__(512) row_fwd_kernel(const RowParams<T> P)
{
    using C = cx<T>;
    constexpr int E = fft_E<T>(L);
    constexpr int TF = L / E;
    constexpr int RS = row_stride(L);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double red[kNQ * 32];
    C *sm = reinterpret_cast<C *>(smem_raw);
    if (P.check_status && P.ct->status != 0) return;

    const Geom &G = P.G;
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int row = tid / TF, t = tid - row * TF;
    const int y0 = blockIdx.x * G.RB, y = y0 + row;
    const int j = blockIdx.y;
    const int nx = G.nx;
    C v[E];
    double acc[1] = {0.0};

    // ---- load stage with the fused elementwise work
    if (P.mode == RF_PLAIN) {
        // plain rows, optionally multiplied by M_S (input of A^T, Eq.17) or M_R (input of A, Eq.16)
        const T *src = P.in0 + (size_t)j * P.plane + (size_t)y * nx;
        const bool rowin = (unsigned)(y - G.oy) < (unsigned)G.sy;
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int x0 = 2 * (t + TF * e);
            C w2 = ld2<T>(src + x0);
            if (P.maskmode == MM_S) {
                if (!(rowin && (unsigned)(x0 - G.ox) < (unsigned)G.sx)) w2.x = (T)0;
                if (!(rowin && (unsigned)(x0 + 1 - G.ox) < (unsigned)G.sx)) w2.y = (T)0;
            } else if (P.maskmode == MM_R && G.masked) {
                C a2 = ld2<T>(P.alphaR + (size_t)y * nx + x0);
                if (!(a2.x > (T)0)) w2.x = (T)0;
                if (!(a2.y > (T)0)) w2.y = (T)0;
            }
            v[e] = w2;
        }
    } else if (P.mode == RF_PSF) {
        // K_j normalised to unit volume and circularly shifted so that its centre sits at (0,0) (A18)
        const T *src = P.in0 + (size_t)j * P.plane;
        const T inv = (T)(1.0 / P.ct->psf_sum);
        int ys = y + P.cy; if (ys >= G.ny) ys -= G.ny;
#pragma unroll
        for (int e = 0; e < E; ++e) {
            int x0 = 2 * (t + TF * e) + P.cxs; if (x0 >= nx) x0 -= nx;
            int x1 = x0 + 1; if (x1 >= nx) x1 -= nx;
            v[e] = mk<T>(src[(size_t)ys * nx + x0] * inv, src[(size_t)ys * nx + x1] * inv);
        }
    } else if (P.mode == RF_MASK_S) {
#pragma unroll
        for (int e = 0; e < E; ++e) {
            int x0 = 2 * (t + TF * e);
            v[e] = mk<T>(in_S(G, y, x0) ? (T)1 : (T)0, in_S(G, y, x0 + 1) ? (T)1 : (T)0);
        }
    } else if (P.mode == RF_RATIO) {
        // a1: r_j = g_j / (A_j f + b_j) on S, 0 elsewhere (Eq.11/14/18)
        const size_t base = (size_t)j * P.plane + (size_t)y * nx;
        const T bc = (T)P.bconst[j];
        const bool rowin = (unsigned)(y - G.oy) < (unsigned)G.sy;
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int x0 = 2 * (t + TF * e);
            C r = mk<T>((T)0, (T)0);
            if (rowin) {
                C g2 = ld2<T>(P.in0 + base + x0), q2 = ld2<T>(P.in1 + base + x0);
                C b2 = P.b_is_array ? ld2<T>(P.in2 + base + x0) : mk<T>(bc, bc);
                if ((unsigned)(x0 - G.ox) < (unsigned)G.sx)     r.x = ratio_term<T>(g2.x, q2.x + b2.x);
                if ((unsigned)(x0 + 1 - G.ox) < (unsigned)G.sx) r.y = ratio_term<T>(g2.y, q2.y + b2.y);
            }
            v[e] = r;
        }
    } else {   // RF_PROJECT
        // a4 + a7: D = (M_R/alpha) clip(f,L1,L2) (Eq.10/23); y = P+(f - alpha_k D grad) (Eq.6); d = y - f; gd = grad'd
        const size_t base = (size_t)y * nx;
        const T alpha = (T)P.ct->alpha, L1 = (T)P.ct->L1, L2 = (T)P.ct->L2;
        const T Wc = (T)(1.0 / (double)G.p);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int x0 = 2 * (t + TF * e);
            C f2 = ld2<T>(P.in0 + base + x0), g2 = ld2<T>(P.in1 + base + x0);
            C w2 = mk<T>(Wc, Wc);
            bool r0 = true, r1 = true;
            if (G.masked) {
                C a2 = ld2<T>(P.alphaR + base + x0);
                r0 = a2.x > (T)0; r1 = a2.y > (T)0;
                w2.x = r0 ? (T)1 / a2.x : (T)0; w2.y = r1 ? (T)1 / a2.y : (T)0;
            }
            C d2;
            {
                T D = w2.x * clipT<T>(f2.x, L1, L2);
                T yv = f2.x - alpha * D * g2.x;
                d2.x = r0 ? ((yv > (T)0 ? yv : (T)0) - f2.x) : (T)0;
                D = w2.y * clipT<T>(f2.y, L1, L2);
                yv = f2.y - alpha * D * g2.y;
                d2.y = r1 ? ((yv > (T)0 ? yv : (T)0) - f2.y) : (T)0;
            }
            acc[0] += (double)g2.x * (double)d2.x + (double)g2.y * (double)d2.y;
            st2<T>(P.out0 + base + x0, d2);
            v[e] = d2;
        }
    }

    // ---- complex FFT of length L = nx/2 over z[m] = x[2m] + i x[2m+1]
    C *smrow = sm + row * RS;
    fft_block<T, L, -1>(v, smrow, 1, t, P.tw);
    __syncthreads();
#pragma unroll
    for (int e = 0; e < E; ++e) smrow[fft_pad(t + TF * e)] = v[e];
    __syncthreads();

    // ---- untangle the two interleaved real transforms and store tile-major
    //      X[k] = (Z[k] + conj Z[L-k])/2 - (i/2) exp(-2 pi i k/nx) (Z[k] - conj Z[L-k]);  entry 0 = (X[0], X[L])
    C *dst = P.spec + (size_t)j * P.specplane;
    const int Cc = G.C, RBC = G.RB * Cc;
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int o = tid + nthr * e;
        const int tile = o / RBC, rem = o - tile * RBC;
        const int rr = rem / Cc, c = rem - rr * Cc;
        const int kx = tile * Cc + c;
        const C *zr = sm + rr * RS;
        const C a = zr[fft_pad(kx)];
        C S;
        if (kx == 0) {
            S = mk<T>(a.x + a.y, a.x - a.y);
        } else {
            const C b = cconj(zr[fft_pad(L - kx)]);
            const C w = __ldg(&P.twh[kx]);
            const C Ek = mk<T>((T)0.5 * (a.x + b.x), (T)0.5 * (a.y + b.y));
            const C Dk = mk<T>((T)0.5 * (a.x - b.x), (T)0.5 * (a.y - b.y));
            const C Ok = mk<T>(Dk.y, -Dk.x);          // -i * Dk
            S = cadd(Ek, cmul(w, Ok));
        }
        dst[(size_t)tile * ((size_t)G.ny * Cc) + (size_t)(y0 + rr) * Cc + c] = S;
    }

    if (P.mode == RF_PROJECT) {
        block_reduce_sum<1>(acc, red);
        if (tid == 0) P.part[blockIdx.x] = acc[0];
    }
}

// ---------------------------------------------------------------- row inverse (half spectrum -> real rows)
// grid = (ny/RB, images).  The epilogue modes carry steps a3+a5 (gradient + BB sums), a9 (line-search
// sum at lambda = 1), the start-point / RL objective, the adaptive bounds and the RL update.
template <typename T, int L>
__global__ void __launch_bounds__(512) row_inv_kernel(const RowParams<T> P)
{
    using C = cx<T>;
    constexpr int E = fft_E<T>(L);
    constexpr int TF = L / E;
    constexpr int RS = row_stride(L);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double red[kNQ * 32];
    C *sm = reinterpret_cast<C *>(smem_raw);
    if (P.check_status && P.ct->status != 0) return;

    const Geom &G = P.G;
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int row = tid / TF, t = tid - row * TF;
    const int y0 = blockIdx.x * G.RB, y = y0 + row;
    const int j = blockIdx.y;
    const int nx = G.nx;

    // ---- tile-major spectrum -> shared memory
    {
        const C *src = P.spec + (size_t)j * P.specplane;
        const int Cc = G.C, RBC = G.RB * Cc;
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int o = tid + nthr * e;
            const int tile = o / RBC, rem = o - tile * RBC;
            const int rr = rem / Cc, c = rem - rr * Cc;
            const int kx = tile * Cc + c;
            sm[rr * RS + fft_pad(kx)] = src[(size_t)tile * ((size_t)G.ny * Cc) + (size_t)(y0 + rr) * Cc + c];
        }
    }
    __syncthreads();
    // ---- re-tangle: Z[k] = (X[k] + conj X[L-k]) + i exp(+2 pi i k/nx) (X[k] - conj X[L-k]);  Z[0] = (X0+XL) + i (X0-XL)
    C v[E];
    C *smrow = sm + row * RS;
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int k = t + TF * e;
        const C a = smrow[fft_pad(k)];
        if (k == 0) {
            v[e] = mk<T>(a.x + a.y, a.x - a.y);
        } else {
            const C b = cconj(smrow[fft_pad(L - k)]);
            const C w = __ldg(&P.twh[k]);
            const C Sk = cadd(a, b), Dk = csub(a, b);
            const C iD = mk<T>(-Dk.y, Dk.x);          // i * Dk
            v[e] = cadd(Sk, cmulc(iD, w));            // times conj(w) = exp(+2 pi i k/nx)
        }
    }
    fft_block<T, L, +1>(v, smrow, 1, t, P.tw);

    // ---- epilogue: v[e] = (w(y, 2m), w(y, 2m+1)), m = t + TF e
    const size_t rowbase = (size_t)y * nx;
    const size_t base = (size_t)j * P.plane + rowbase;
    const bool rowin = (unsigned)(y - G.oy) < (unsigned)G.sy;
    const unsigned int nblk = gridDim.x * gridDim.y;
    const int bid = blockIdx.y * gridDim.x + blockIdx.x;

    if (P.mode == RI_PLAIN) {
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int x0 = 2 * (t + TF * e);
            C w2 = v[e];
            if (P.maskmode == MM_S) {
                if (!(rowin && (unsigned)(x0 - G.ox) < (unsigned)G.sx)) w2.x = (T)0;
                if (!(rowin && (unsigned)(x0 + 1 - G.ox) < (unsigned)G.sx)) w2.y = (T)0;
            } else if (P.maskmode == MM_R && G.masked) {
                C a2 = ld2<T>(P.alphaR + rowbase + x0);
                if (!(a2.x > (T)0)) w2.x = (T)0;
                if (!(a2.y > (T)0)) w2.y = (T)0;
            }
            st2<T>(P.out0 + base + x0, w2);
        }
    } else if (P.mode == RI_GRAD) {
        // a3: grad = alpha - w on R (Eq.11/14/18).  a5: the four BB dot products with s = lambda d (= f(k)-f(k-1)),
        // z = grad - grad_prev and D = (M_R/alpha) clip(f,L1,L2) (Eq.7-8), accumulated in double.
        const int k = P.ct->k;
        const double lam = P.ct->lambda;
        const T L1 = (T)P.ct->L1, L2 = (T)P.ct->L2;
        const T pT = (T)G.p, Wc = (T)(1.0 / (double)G.p);
        double acc[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int x0 = 2 * (t + TF * e);
            C a2 = mk<T>(pT, pT), w2 = mk<T>(Wc, Wc);
            bool r0 = true, r1 = true;
            if (G.masked) {
                a2 = ld2<T>(P.alphaR + rowbase + x0);
                r0 = a2.x > (T)0; r1 = a2.y > (T)0;
                w2.x = r0 ? (T)1 / a2.x : (T)0; w2.y = r1 ? (T)1 / a2.y : (T)0;
            }
            C gn = mk<T>(r0 ? a2.x - v[e].x : (T)0, r1 ? a2.y - v[e].y : (T)0);
            if (k > 0) {
                C f2 = ld2<T>(P.in0 + rowbase + x0), d2 = ld2<T>(P.in1 + rowbase + x0), go = ld2<T>(P.out0 + rowbase + x0);
                if (r0) {
                    const double s = lam * (double)d2.x, z = (double)gn.x - (double)go.x;
                    const double Di = (double)(w2.x * clipT<T>(f2.x, L1, L2)), inv = 1.0 / Di;
                    const double si = s * inv, zd = z * Di;
                    acc[0] += si * si; acc[1] += si * z; acc[2] += s * zd; acc[3] += zd * zd;
                }
                if (r1) {
                    const double s = lam * (double)d2.y, z = (double)gn.y - (double)go.y;
                    const double Di = (double)(w2.y * clipT<T>(f2.y, L1, L2)), inv = 1.0 / Di;
                    const double si = s * inv, zd = z * Di;
                    acc[0] += si * si; acc[1] += si * z; acc[2] += s * zd; acc[3] += zd * zd;
                }
            }
            st2<T>(P.out0 + rowbase + x0, gn);
        }
        block_reduce_sum<4>(acc, red);
        if (publish_partials<4>(acc, P.part, bid, nblk, &P.ct->counter[TK_GRAD])) {
            final_sum<4>(acc, P.part, nblk, red);
            if (tid == 0) bb_step(P.ct, P.o, P.tr, acc[0], acc[1], acc[2], acc[3]);   // a6
        }
    } else if (P.mode == RI_LS || P.mode == RI_QJ) {
        // RI_LS (a8 tail + a9): u_j = A_j d on S; J(1) = sum kl(g_j, q_j + u_j + b_j).
        // RI_QJ: q_j = A_j f on S; J0(f) = sum kl(g_j, q_j + b_j) (Eq.2/12 over S, A12).
        const T bc = (T)P.bconst[j];
        double acc[1] = {0.0};
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int x0 = 2 * (t + TF * e);
            const bool s0 = rowin && (unsigned)(x0 - G.ox) < (unsigned)G.sx;
            const bool s1 = rowin && (unsigned)(x0 + 1 - G.ox) < (unsigned)G.sx;
            C u2 = mk<T>(s0 ? v[e].x : (T)0, s1 ? v[e].y : (T)0);
            st2<T>(P.out0 + base + x0, u2);
            if (rowin && P.submode != QJ_PLAIN) {
                C g2 = ld2<T>(P.in0 + base + x0);
                C b2 = P.b_is_array ? ld2<T>(P.in2 + base + x0) : mk<T>(bc, bc);
                C y2 = u2;
                if (P.mode == RI_LS) { C q2 = ld2<T>(P.in1 + base + x0); y2.x += q2.x; y2.y += q2.y; }
                if (s0) acc[0] += (double)kl_term(g2.x, (T)(y2.x + b2.x));
                if (s1) acc[0] += (double)kl_term(g2.y, (T)(y2.y + b2.y));
            }
        }
        if (P.submode == QJ_PLAIN && P.mode == RI_QJ) return;
        block_reduce_sum<1>(acc, red);
        const int tk = (P.mode == RI_LS) ? TK_LS : TK_QJ;
        if (publish_partials<1>(acc, P.part, bid, nblk, &P.ct->counter[tk])) {
            final_sum<1>(acc, P.part, nblk, red);
            const double J = acc[0];
            Ctrl *ct = P.ct;
            if (P.mode == RI_LS) {
                double gd[1];
                final_sum<1>(gd, P.part2, gridDim.x, red);     // grad'd partials of the projection kernel
                if (tid == 0) {
                    // Alg.1 step 5 at lambda = 1: J(f + d) <= J_ref + beta * 1 * grad'd
                    const double Jref = armijo_ref(ct);
                    ct->gd = gd[0]; ct->Jref = Jref; ct->Jtrial = J;
                    int acc1 = (isfinite(J) && J <= Jref + P.o.beta * gd[0]) ? 1 : 0;
                    if (P.tr.force_lambda) {
                        const double fl = P.tr.force_lambda[ct->k];
                        if (isfinite(fl)) acc1 = (fl == 1.0) ? 1 : 0;
                    }
                    ct->accepted = acc1;
                }
            } else if (tid == 0) {
                if (P.submode == QJ_INIT) {
                    ct->J = J; ct->Jhist[0] = J; ct->nJ = 1;
                    if (P.tr.J) P.tr.J[0] = J;
                    if (!isfinite(J)) ct->status = SGP_ERR_NONFINITE;
                } else {   // QJ_RL: J0(f(k)) and the stopping rules before the k-th RL update
                    const int k = ct->k;
                    const double Jold = ct->J;
                    ct->J = J;
                    if (P.tr.J) P.tr.J[k] = J;
                    if (!isfinite(J)) ct->status = SGP_ERR_NONFINITE;
                    else {
                        int r = stop_test(P.o, k, J, Jold, k > 0);
                        if (r) ct->status = r; else ct->k = k + 1;
                    }
                }
            }
        }
    } else if (P.mode == RI_RLMINMAX) {
        // adaptive bounds (A19): y = one RL step from f(0); smallest strictly positive value and maximum
        const T Wc = (T)(1.0 / (double)G.p);
        double acc[2] = {-INFINITY, -INFINITY};   // (-min positive, max)
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int x0 = 2 * (t + TF * e);
            C f2 = ld2<T>(P.in0 + rowbase + x0);
            C w2 = mk<T>(Wc, Wc);
            if (G.masked) {
                C a2 = ld2<T>(P.alphaR + rowbase + x0);
                w2.x = a2.x > (T)0 ? (T)1 / a2.x : (T)0; w2.y = a2.y > (T)0 ? (T)1 / a2.y : (T)0;
            }
            const double ya = (double)(w2.x * f2.x * v[e].x), yb = (double)(w2.y * f2.y * v[e].y);
            if (ya > 0.0) acc[0] = fmax(acc[0], -ya);
            if (yb > 0.0) acc[0] = fmax(acc[0], -yb);
            acc[1] = fmax(acc[1], fmax(ya, yb));
        }
        // max-reduction over the block (fixed tree)
        const int lane = tid & 31, wid = tid >> 5, nw = (nthr + 31) >> 5;
#pragma unroll
        for (int q = 0; q < 2; ++q) {
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) acc[q] = fmax(acc[q], __shfl_down_sync(0xffffffffu, acc[q], off));
            if (lane == 0) red[q * 32 + wid] = acc[q];
        }
        __syncthreads();
        if (tid == 0) {
            for (int q = 0; q < 2; ++q) { double m = red[q * 32]; for (int w = 1; w < nw; ++w) m = fmax(m, red[q * 32 + w]); acc[q] = m; }
        }
        __syncthreads();
        if (publish_partials<2>(acc, P.part, bid, nblk, &P.ct->counter[TK_MINMAX])) {
            if (tid == 0) {
                double mn = -INFINITY, mx = -INFINITY;
                for (unsigned int b = 0; b < nblk; ++b) { mn = fmax(mn, __ldcg(&P.part[2 * b])); mx = fmax(mx, __ldcg(&P.part[2 * b + 1])); }
                const double ymin = -mn, ymax = mx;
                if (!(ymin < INFINITY) || !(ymax > 0.0)) P.ct->status = SGP_ERR_DATA;
                else if (ymax / ymin < 50.0) { P.ct->L1 = ymin / 10.0; P.ct->L2 = ymax * 10.0; }
                else                         { P.ct->L1 = ymin;        P.ct->L2 = ymax; }
            }
        }
    } else {   // RI_RLUPDATE, a12: f <- (M_R/alpha) o f o sum_j A_j^T(g_j/(A_j f + b_j))   (Eq.1/13/21)
        const T Wc = (T)(1.0 / (double)G.p);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int x0 = 2 * (t + TF * e);
            C f2 = ld2<T>(P.in0 + rowbase + x0);
            C w2 = mk<T>(Wc, Wc);
            if (G.masked) {
                C a2 = ld2<T>(P.alphaR + rowbase + x0);
                w2.x = a2.x > (T)0 ? (T)1 / a2.x : (T)0; w2.y = a2.y > (T)0 ? (T)1 / a2.y : (T)0;
            }
            st2<T>(P.out0 + rowbase + x0, mk<T>(w2.x * f2.x * v[e].x, w2.y * f2.y * v[e].y));
        }
    }
}

// ---------------------------------------------------------------- column kernel
// grid = (nx/2)/C tiles, block = C * (L/E) threads (thread = (t, c), c fastest), dynamic smem = C * padded(L) complex.
//   CM_FWD / CM_INV: out = forward / unnormalised inverse column FFT of in (set-up of the transfer functions, rfft2 helpers)
//   CM_CONJSUM: out = IFFTcol( sum_j conj(K^_j) o FFTcol(in_j) )         (a2: sum_j A_j^T r_j in Fourier space, Eq.17)
//   CM_MULT   : out_j = IFFTcol( K^_j o FFTcol(in) ), j < p              (a8: A_j d, Eq.16)
// Column 0 of tile 0 carries the packed pair (kx = 0, kx = nx/2): with C~[ky] = conj(C[-ky]) the product is
//   C'[ky] = A[ky] C[ky] + B[ky] C~[ky],  A = (K0 + KM)/2 (stored in column 0 of khat), B = (K0 - KM)/2 (khatB).
// The partner values C[-ky] of that one column go through a small global scratch line (P.pack, L entries).
enum ColMode { CM_FWD = 0, CM_CONJSUM = 1, CM_MULT = 2, CM_INV = 3 };

template <typename T, int L, int MODE, bool MULTI>
__global__ void __launch_bounds__(512) col_kernel(const ColParams<T> P)
{
    using C = cx<T>;
    constexpr int E = fft_E<T>(L);
    constexpr int TF = L / E;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *sm = reinterpret_cast<C *>(smem_raw);
    if (P.check_status && P.ct->status != 0) return;

    const int Cc = P.G.C;
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int t = tid / Cc, c = tid - t * Cc;
    const size_t tbase = (size_t)blockIdx.x * ((size_t)L * Cc) + tid;
    C *smc = sm + c;
    const bool packed = (blockIdx.x == 0);      // tile 0 holds the packed column
    const bool pk = packed && c == 0;
    volatile C *pack = P.pack;
    C v[E];

    if constexpr (MODE == CM_FWD || MODE == CM_INV) {
#pragma unroll
        for (int e = 0; e < E; ++e) v[e] = P.in[tbase + (size_t)e * nthr];
        fft_block<T, L, (MODE == CM_FWD ? -1 : +1)>(v, smc, Cc, t, P.tw);
#pragma unroll
        for (int e = 0; e < E; ++e) P.out[tbase + (size_t)e * nthr] = v[e];
    } else if constexpr (MODE == CM_CONJSUM) {
        C acc[MULTI ? E : 1];
        const int p = MULTI ? P.p : 1;
        for (int j = 0; j < p; ++j) {
            const C *src = P.in + (size_t)j * P.specplane;
            const C *kh = P.khat + (size_t)j * P.specplane;
#pragma unroll
            for (int e = 0; e < E; ++e) v[e] = src[tbase + (size_t)e * nthr];
            fft_block<T, L, -1>(v, smc, Cc, t, P.tw);
            if (packed) {
                if (pk) {
#pragma unroll
                    for (int e = 0; e < E; ++e) { pack[t + TF * e].x = v[e].x; pack[t + TF * e].y = v[e].y; }
                }
                __syncthreads();
            }
#pragma unroll
            for (int e = 0; e < E; ++e) {
                const C k = kh[tbase + (size_t)e * nthr];
                C r = cmulc(v[e], k);
                if (pk) {
                    const int ky = t + TF * e, kyn = ky == 0 ? 0 : L - ky;
                    C ct; ct.x = pack[kyn].x; ct.y = -pack[kyn].y;
                    r = cadd(r, cmulc(ct, P.khatB[(size_t)j * L + ky]));
                }
                if constexpr (MULTI) { if (j == 0) acc[e] = r; else acc[e] = cadd(acc[e], r); }
                else v[e] = r;
            }
        }
        if constexpr (MULTI) {
#pragma unroll
            for (int e = 0; e < E; ++e) v[e] = acc[e];
        }
        fft_block<T, L, +1>(v, smc, Cc, t, P.tw);
#pragma unroll
        for (int e = 0; e < E; ++e) P.out[tbase + (size_t)e * nthr] = v[e];
    } else {   // CM_MULT
#pragma unroll
        for (int e = 0; e < E; ++e) v[e] = P.in[tbase + (size_t)e * nthr];
        fft_block<T, L, -1>(v, smc, Cc, t, P.tw);
        if (packed) {
            if (pk) {
#pragma unroll
                for (int e = 0; e < E; ++e) { pack[t + TF * e].x = v[e].x; pack[t + TF * e].y = v[e].y; }
            }
            __syncthreads();
        }
        const int p = MULTI ? P.p : 1;
        for (int j = 0; j < p; ++j) {
            const C *kh = P.khat + (size_t)j * P.specplane;
            C w[E];
#pragma unroll
            for (int e = 0; e < E; ++e) {
                const C k = kh[tbase + (size_t)e * nthr];
                w[e] = cmul(v[e], k);
                if (pk) {
                    const int ky = t + TF * e, kyn = ky == 0 ? 0 : L - ky;
                    C ct; ct.x = pack[kyn].x; ct.y = -pack[kyn].y;
                    w[e] = cadd(w[e], cmul(ct, P.khatB[(size_t)j * L + ky]));
                }
            }
            fft_block<T, L, +1>(w, smc, Cc, t, P.tw);
            C *dst = P.out + (size_t)j * P.specplane;
#pragma unroll
            for (int e = 0; e < E; ++e) dst[tbase + (size_t)e * nthr] = w[e];
        }
    }
}

// ---------------------------------------------------------------- a9 (backtracks) + a10 + a11: line search and update
// Cooperative kernel (all CTAs resident).  lambda = 1 was tested by the RI_LS epilogue; if it failed, the
// Armijo loop lambda <- theta lambda runs here: every trial is one elementwise pass over
// q_j + lambda u_j (no FFT), one grid-wide barrier, and the same decision taken redundantly by every CTA.
// Then f <- f + lambda d, q_j <- q_j + lambda u_j (Alg.1 step 6, A21), and the last CTA does the
// book-keeping (history, trace, stopping rules).
template <typename T> struct UpdParams {
    Geom G;
    DevOpts o;
    Trace tr;
    Ctrl *ct;
    T *f; const T *d;
    T *q; const T *u; const T *g; const T *b;    // image j at + j*plane
    size_t plane;
    int b_is_array;
    double bconst[kMaxP];
    double *part;                                // gridDim.x doubles
};

template <typename T> struct vec4_of;
template <> struct vec4_of<float>  { using type = float4;  static constexpr int N = 4; };
template <> struct vec4_of<double> { using type = double2; static constexpr int N = 2; };

template <typename T>
__global__ void __launch_bounds__(256) update_kernel(const UpdParams<T> P)
{
    using V = typename vec4_of<T>::type;
    constexpr int VN = vec4_of<T>::N;
    __shared__ double red[32];
    __shared__ double s_J;
    Ctrl *ct = P.ct;
    if (ct->status != 0) return;
    const Geom &G = P.G;
    const size_t n = (size_t)G.ny * G.nx, nv = n / VN;
    const size_t gtid = (size_t)blockIdx.x * blockDim.x + threadIdx.x, gstride = (size_t)gridDim.x * blockDim.x;
    const int k = ct->k;
    const double Jref = ct->Jref, gd = ct->gd;
    double lambda = 1.0, Jnew = ct->Jtrial;
    bool accepted = ct->accepted != 0;
    bool forced = false;
    if (P.tr.force_lambda) {
        const double fl = P.tr.force_lambda[k];
        if (isfinite(fl)) { forced = true; if (fl != 1.0) { lambda = fl / P.o.theta; accepted = false; } }
    }
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
            const T *q = P.q + (size_t)j * P.plane, *u = P.u + (size_t)j * P.plane, *g = P.g + (size_t)j * P.plane;
            const T *b = P.b_is_array ? P.b + (size_t)j * P.plane : nullptr;
            const T bc = (T)P.bconst[j];
            for (size_t i = gtid; i < nv; i += gstride) {
                const size_t i0 = i * VN;
                const int y = (int)(i0 / G.nx), x = (int)(i0 - (size_t)y * G.nx);
                if ((unsigned)(y - G.oy) >= (unsigned)G.sy) continue;
                V q4 = reinterpret_cast<const V *>(q)[i], u4 = reinterpret_cast<const V *>(u)[i], g4 = reinterpret_cast<const V *>(g)[i];
                const T *qa = reinterpret_cast<const T *>(&q4), *ua = reinterpret_cast<const T *>(&u4), *ga = reinterpret_cast<const T *>(&g4);
#pragma unroll
                for (int c = 0; c < VN; ++c) {
                    if ((unsigned)(x + c - G.ox) < (unsigned)G.sx) {
                        const T bb = b ? b[i0 + c] : bc;
                        acc[0] += (double)kl_term(ga[c], (T)((T)(qa[c] + lam * ua[c]) + bb));
                    }
                }
            }
        }
        block_reduce_sum<1>(acc, red);
        if (threadIdx.x == 0) P.part[blockIdx.x] = acc[0];
        __threadfence();
        cg::this_grid().sync();
        double tot[1] = {0.0};
        for (unsigned int bI = threadIdx.x; bI < gridDim.x; bI += blockDim.x) tot[0] += __ldcg(&P.part[bI]);
        block_reduce_sum<1>(tot, red);
        if (threadIdx.x == 0) s_J = tot[0];
        __syncthreads();
        Jnew = s_J;
        accepted = forced || (isfinite(Jnew) && Jnew <= Jref + P.o.beta * lambda * gd);
        cg::this_grid().sync();     // partials may be overwritten by the next trial
    }
    if (forced && nbt > 0) nbt = 0;
    // ---- update
    const T lam = (T)lambda;
    {
        V *f = reinterpret_cast<V *>(P.f); const V *d = reinterpret_cast<const V *>(P.d);
        for (size_t i = gtid; i < nv; i += gstride) {
            V a = f[i], dd = d[i];
            T *aa = reinterpret_cast<T *>(&a); const T *da = reinterpret_cast<const T *>(&dd);
#pragma unroll
            for (int c = 0; c < VN; ++c) aa[c] = aa[c] + lam * da[c];
            f[i] = a;
        }
        for (int j = 0; j < G.p; ++j) {
            V *q = reinterpret_cast<V *>(P.q + (size_t)j * P.plane); const V *u = reinterpret_cast<const V *>(P.u + (size_t)j * P.plane);
            for (size_t i = gtid; i < nv; i += gstride) {
                V a = q[i], dd = u[i];
                T *aa = reinterpret_cast<T *>(&a); const T *da = reinterpret_cast<const T *>(&dd);
#pragma unroll
                for (int c = 0; c < VN; ++c) aa[c] = aa[c] + lam * da[c];
                q[i] = a;
            }
        }
    }
    // ---- book-keeping by the last CTA to finish
    __shared__ int s_last;
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        unsigned int tk = atomicAdd(&ct->counter[TK_UPDATE], 1u);
        s_last = (tk == gridDim.x - 1);
        if (s_last) { ct->counter[TK_UPDATE] = 0; finish_iteration(ct, P.o, P.tr, lambda, Jnew, nbt); }
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
