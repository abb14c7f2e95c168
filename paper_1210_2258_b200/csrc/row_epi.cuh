// row_epi.cuh -- elementwise epilogues of the inverse row kernel.  The transformed row w (2L reals) has been
// parked in shared memory, so the registers of the FFT are free and the planes of the iteration are streamed
// with 128-bit loads, four pixels per step and thread: x = 4 (t + TF it) .. + 3.
#pragma once
#include "ew.cuh"

namespace sgpk {

// quads loaded ahead of the first store of a batch
template <typename T> __host__ __device__ constexpr int batch_len(int nit)
{
    return sizeof(T) == 8 ? (nit % 2 == 0 ? 2 : 1) : (nit % 4 == 0 ? 4 : (nit % 2 == 0 ? 2 : 1));
}

// quads of g and q loaded ahead in epi_kl.  Measured at 2048^2 (K6, us): 2 quads 30.6, 4 quads 29.8, 8 quads 36.3 (3 x 2048^2:
// 101 / 99 / 130) -- longer batches do not hide more latency, they delay the first KL evaluation of every warp
#ifndef SGP_KL_BATCH
#define SGP_KL_BATCH 4
#endif
template <typename T> __host__ __device__ constexpr int batch_len_kl(int nit)
{
    return (sizeof(T) == 4 && nit % SGP_KL_BATCH == 0) ? SGP_KL_BATCH : batch_len<T>(nit);
}

// M_S for the four pixels of a quad
template <typename T>
__device__ __forceinline__ void quad_in_S(const Geom &G, bool rowin, int x, bool (&s)[4])
{
#pragma unroll
    for (int c = 0; c < 4; ++c) s[c] = rowin && (unsigned)(x + c - G.ox) < (unsigned)G.sx;
}

// a10 (lazy) + a3 + a5: f <- f + lambda d; grad = alpha - w on R (Eq.11/14/18); the four BB dot products with
// s = lambda d, z = grad - grad_prev, D = (M_R/alpha) clip(f(k),L1,L2) (Eq.7-8).  s/D and z D are formed in T; float:
// the four products of a pixel are summed over its quad in float (fma) and each quad sum is added to a double
// accumulator (6 instructions per pixel less than converting every factor); double: everything in double.
template <typename T, int L, int TF, bool MASKED>
__device__ __forceinline__ void epi_grad(const RowParams<T> &P, const RowPtrs<T> &X, const T *wrow, int t, size_t rowbase, double (&acc)[4])
{
    const Geom &G = P.G;
    const int k = X.ct->k;
    const bool pend = X.ct->pending != 0;          // 0 after a refresh round (A21), which has already applied the step
    const T lam = (T)X.ct->lambda;
    const T L1 = (T)X.ct->L1, L2 = (T)X.ct->L2;
    const T pT = (T)G.p, Wc = (T)(1.0 / (double)G.p);
    constexpr int NIT = (L / 2) / TF;
    if (k == 0) {
#pragma unroll 4
        for (int it = 0; it < NIT; ++it) {
            const int x = 4 * (t + TF * it);
            const Quad<T> w4 = ldq<T>(wrow + x);
            Quad<T> g4;
            if constexpr (MASKED) {
                const Quad<T> a4 = ldq<T>(P.alphaR + rowbase + x);
#pragma unroll
                for (int c = 0; c < 4; ++c) g4.a[c] = a4.a[c] > (T)0 ? a4.a[c] - w4.a[c] : (T)0;
            } else {
#pragma unroll
                for (int c = 0; c < 4; ++c) g4.a[c] = pT - w4.a[c];
            }
            stq_if<T>(X.act, X.out0 + rowbase + x, g4);
        }
        return;
    }
    // loads of a batch are issued before its stores: the planes are updated in place, so the compiler must not be
    // left to order them (it would serialise every load behind the previous store)
    constexpr int U = batch_len<T>(NIT);
    for (int it0 = 0; it0 < NIT; it0 += U) {
        Quad<T> f4[U], d4[U], go4[U], a4[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int x = 4 * (t + TF * (it0 + u));
            f4[u] = ldq<T>(X.in0 + rowbase + x);
            d4[u] = ldq<T>(X.in1 + rowbase + x);
            go4[u] = ldq<T>(X.out0 + rowbase + x);
            if constexpr (MASKED) a4[u] = ldq<T>(P.alphaR + rowbase + x);
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int x = 4 * (t + TF * (it0 + u));
            const Quad<T> w4 = ldq<T>(wrow + x);          // shared memory: fetched when used
            Quad<T> g4;
            T pq[4] = {(T)0, (T)0, (T)0, (T)0};     // the four sums over this quad, in T; added to the double accumulators once per quad
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const T s = lam * d4[u].a[c];
                const T fn = pend ? f4[u].a[c] + s : f4[u].a[c];
                f4[u].a[c] = fn;
                bool inR = true;
                T av = pT, wv = Wc;
                if constexpr (MASKED) { av = a4[u].a[c]; inR = av > (T)0; wv = inR ? (T)1 / av : (T)0; }
                const T gn = inR ? av - w4.a[c] : (T)0;
                g4.a[c] = gn;
                const T Di = wv * clipT<T>(fn, L1, L2);
                const T zf = gn - go4[u].a[c];
                if constexpr (sizeof(T) == 8) {
                    const double si = inR ? fast_div(s, Di) : 0.0, z = inR ? zf : 0.0, zd = inR ? zf * Di : 0.0;
                    acc[0] += si * si; acc[1] += si * z; acc[2] += s * zd; acc[3] += zd * zd;
                } else {
                    const T si = inR ? fast_div(s, Di) : (T)0, z = inR ? zf : (T)0, zd = inR ? zf * Di : (T)0;
                    pq[0] = fmaf(si, si, pq[0]); pq[1] = fmaf(si, z, pq[1]); pq[2] = fmaf(s, zd, pq[2]); pq[3] = fmaf(zd, zd, pq[3]);
                }
            }
            if constexpr (sizeof(T) == 4) {
#pragma unroll
                for (int k4 = 0; k4 < 4; ++k4) acc[k4] += (double)pq[k4];
            }
            stq_if<T>(X.act, X.out1 + rowbase + x, f4[u]);
            stq_if<T>(X.act, X.out0 + rowbase + x, g4);
        }
    }
}

// RI_LS (a8 tail + a9): u_j = A_j d on S; J(1) = sum kl(g_j, q_j + u_j + b_j).
// RI_QJ: q_j = A_j f on S; J0(f) = sum kl(g_j, q_j + b_j) (Eq.2/12 over S, A12); QJ_PLAIN only stores.
// RATIO: besides that, the ratio r_j = g_j / (y_j + b_j) of the step that follows (a1) replaces the row in shared memory
// (wmut), from where the caller transforms it:
//   RI_LSF (WITH_Q, STORE_ROW, STORE_Q): the step lambda = 1 is applied speculatively -- q_j + u_j goes to the other q
//     buffer (qout); if the Armijo test then accepts lambda = 1 (the usual case) the next iteration needs no ratio kernel;
//   RI_QJF (RL / OSEM, SURVEY.md 8(d) "RL schedule": row C2R -> ratio -> row R2C in one kernel): A_j f is used for J0 and
//     the ratio and never stored.
template <typename T, int L, int TF, bool WITH_Q, bool MASKED, bool RATIO, bool STORE_ROW, bool STORE_Q>
__device__ __forceinline__ void epi_kl(const RowParams<T> &P, const RowPtrs<T> &X, const T *wrow, T *wmut, const T *qin, T *qout, T *rowout, int t, int y, int j,
                                       size_t base, bool plain, double (&acc)[1])
{
    const Geom &G = P.G;
    const T bc = (T)(P.slab ? X.ct->bconst[j] : P.bconst[j]);
    const bool rowin = (unsigned)(y - G.oy) < (unsigned)G.sy;
    constexpr int NIT = (L / 2) / TF;
    constexpr int U = batch_len_kl<T>(NIT);
    const bool need = rowin && (!plain || RATIO);
    for (int it0 = 0; it0 < NIT; it0 += U) {
        Quad<T> g4[U], q4[U], b4[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int x = 4 * (t + TF * (it0 + u));
            if (need) {
                g4[u] = ldq<T>(X.in0 + base + x);
                if constexpr (WITH_Q) q4[u] = ldq<T>(qin + base + x);
                if (P.b_is_array) b4[u] = ldq<T>(X.in2 + base + x);
            }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int x = 4 * (t + TF * (it0 + u));
            bool s[4] = {true, true, true, true};      // without a boundary mask S is the whole grid
            if constexpr (MASKED) quad_in_S<T>(G, rowin, x, s);
            const Quad<T> w4 = ldq<T>(wrow + x);          // the row itself sits in shared memory: fetched when used
            Quad<T> u4;
#pragma unroll
            for (int c = 0; c < 4; ++c) u4.a[c] = s[c] ? w4.a[c] : (T)0;
            if constexpr (STORE_ROW) stq_if<T>(X.act, rowout + base + x, u4);
            Quad<T> r4;
#pragma unroll
            for (int c = 0; c < 4; ++c) r4.a[c] = (T)0;
            if (need) {
                T yv[4];
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    yv[c] = u4.a[c];
                    if constexpr (WITH_Q) yv[c] += q4[u].a[c];
                }
                if constexpr (STORE_Q) {
                    Quad<T> q1;
#pragma unroll
                    for (int c = 0; c < 4; ++c) q1.a[c] = yv[c];
                    stq_if<T>(X.act, qout + base + x, q1);
                }
#pragma unroll
                for (int c = 0; c < 4; ++c) yv[c] += P.b_is_array ? b4[u].a[c] : bc;
                if (!plain) acc[0] += (double)kl_quad(g4[u].a, yv, s);
                if constexpr (RATIO) {
#pragma unroll
                    for (int c = 0; c < 4; ++c) r4.a[c] = s[c] ? ratio_term(g4[u].a[c], yv[c]) : (T)0;
                }
            }
            if constexpr (RATIO) stq<T>(wmut + x, r4);
        }
    }
}

// plain store with the output mask of Eq.16 (M_S) or Eq.17 (M_R)
template <typename T, int L, int TF, bool MK>
__device__ __forceinline__ void epi_store(const RowParams<T> &P, const RowPtrs<T> &X, const T *wrow, int t, int y, size_t rowbase, size_t base)
{
    const Geom &G = P.G;
    const bool rowin = (unsigned)(y - G.oy) < (unsigned)G.sy;
    constexpr int NIT = (L / 2) / TF;
#pragma unroll 4
    for (int it = 0; it < NIT; ++it) {
        const int x = 4 * (t + TF * it);
        Quad<T> w4 = ldq<T>(wrow + x);
        if (P.maskmode == MM_S) {
            bool s[4];
            quad_in_S<T>(G, rowin, x, s);
#pragma unroll
            for (int c = 0; c < 4; ++c) if (!s[c]) w4.a[c] = (T)0;
        } else if (P.maskmode == MM_R && MK) {
            const Quad<T> a4 = ldq<T>(P.alphaR + rowbase + x);
#pragma unroll
            for (int c = 0; c < 4; ++c) if (!(a4.a[c] > (T)0)) w4.a[c] = (T)0;
        }
        if (P.submode == RIP_STORE_POS) {
#pragma unroll
            for (int c = 0; c < 4; ++c) w4.a[c] = w4.a[c] > (T)0 ? w4.a[c] : (T)0;
        }
        stq_if<T>(X.act, X.out0 + base + x, w4);
    }
}

// y = (M_R/alpha) f w: one RL step (Eq.1/13/21).  STORE: write it (a12); else accumulate (-min positive, max) for
// the adaptive bounds (A19).
// FUSE (RI_RLUPF, SURVEY.md 8(d) "RL schedule": row C2R -> f update -> row R2C of the new f in one kernel): the new f also
// replaces the row in shared memory (wmut), from where the caller transforms it for the next round.
template <typename T, int L, int TF, bool STORE, bool MK, bool FUSE = false>
__device__ __forceinline__ void epi_rl(const RowParams<T> &P, const RowPtrs<T> &X, const T *wrow, int t, size_t rowbase, double (&acc)[2], T *wmut = nullptr)
{
    const Geom &G = P.G;
    const T Wc = (T)(1.0 / (double)G.p);
    const bool relax = P.o.rl_relax != 1.0;          // multiplicative relaxation of RL, Eq.3
    const T rx = (T)P.o.rl_relax;
    const bool lin = P.o.rl_linear != 1.0;           // linear relaxation of RL, Eq.4
    const T lam = (T)P.o.rl_linear;
    constexpr int NIT = (L / 2) / TF;
    constexpr int U = batch_len<T>(NIT);
    for (int it0 = 0; it0 < NIT; it0 += U) {
        Quad<T> w4[U], f4[U], a4[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int x = 4 * (t + TF * (it0 + u));
            w4[u] = ldq<T>(wrow + x);
            f4[u] = ldq<T>(X.in0 + rowbase + x);
            if (MK) a4[u] = ldq<T>(P.alphaR + rowbase + x);
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int x = 4 * (t + TF * (it0 + u));
            Quad<T> y4;
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                T wv = Wc;
                if (MK) wv = a4[u].a[c] > (T)0 ? (T)1 / a4[u].a[c] : (T)0;
                y4.a[c] = wv * f4[u].a[c] * w4[u].a[c];
                if (STORE && relax) y4.a[c] = f4[u].a[c] * pow(fmax(wv * w4[u].a[c], (T)0), rx);      // Eq.3
                if (STORE && lin) y4.a[c] = fmax(f4[u].a[c] - lam * (f4[u].a[c] * ((T)1 - wv * w4[u].a[c])), (T)0);   // Eq.4, projected on f >= 0 (A25)
                if constexpr (!STORE) {
                    const double yd = (double)y4.a[c];
                    if (yd > 0.0) acc[0] = fmax(acc[0], -yd);
                    acc[1] = fmax(acc[1], yd);
                }
            }
            if constexpr (STORE) stq_if<T>(X.act, X.out0 + rowbase + x, y4);
            if constexpr (FUSE) stq<T>(wmut + x, y4);
        }
    }
}

}  // namespace sgpk
